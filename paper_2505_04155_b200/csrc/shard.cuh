// shard.cuh — device side of the row-sharded solve (include/amp_pcg.h, "row-sharded solve").
//
// Algorithm 4.1 split by block rows: per iteration the ranks exchange (1) the halo of p that the
// mat-vec of line 11 gathers, in the precision it gathers, and (2) the three inner products of lines 6, 13, 17.
// Both exchanges are plain stores into peer-mapped device memory issued by the loop kernels themselves:
//   * halo: the p update (phase_p) stores every chunk that lies in a send range a second time, straight into the
//     neighbour's halo band; the block that finishes last raises the neighbours' flags (st.release.sys); the mat-vec
//     waits for its own two flags (ld.acquire.sys) before its first gather.
//   * sums: the block that finishes a grid reduction posts (v0, v1, tag) into EVERY rank's mailbox (its own included);
//     k_epi, one warp, waits until the entries of all ranks carry the tag, adds them in rank order and runs the scalar
//     step (epi_rho / epi_gamma / epi_delta ...) — the same numbers in the same order on every rank, so all ranks take
//     identical decisions and no result is ever broadcast.
// Tags are (solve counter << 32) | sequence number, so nothing is ever reset and a stale entry can not be mistaken.
// A wait that lasts longer than kShardTimeoutNs gives up: status AMP_ERR_CUDA (-3), done = 1.
#pragma once
#include "phases.cuh"

namespace amp {

constexpr unsigned long long kShardTimeoutNs = 10ull * 1000ull * 1000ull * 1000ull;
// sequence numbers of the halo exchanges that are not the loop's (the loop uses k + 1)
constexpr unsigned int kHaloTagSetup = 0xfffffff0u, kHaloTagFinal = 0xfffffff1u, kHaloTagSpmv = 0xfffffff2u;

__device__ __forceinline__ void st_release_sys_u64(unsigned long long* p, unsigned long long v) {
  asm volatile("st.release.sys.global.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}
__device__ __forceinline__ unsigned long long ld_acquire_sys_u64(const unsigned long long* p) {
  unsigned long long v;
  asm volatile("ld.acquire.sys.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ unsigned long long global_timer_ns() {
  unsigned long long t;
  asm volatile("mov.u64 %0, %globaltimer;" : "=l"(t));
  return t;
}
// wait until *p == want with relaxed loads (the caller fences once after all its waits); false on timeout
__device__ __forceinline__ bool shard_spin_relaxed(const unsigned long long* p, unsigned long long want) {
  const volatile unsigned long long* vp = p;
  if (*vp == want) return true;
  const unsigned long long t0 = global_timer_ns();
  while (*vp != want) {
    if (global_timer_ns() - t0 > kShardTimeoutNs) return false;
    __nanosleep(50);
  }
  return true;
}
// wait until *p == want; false on timeout
__device__ __forceinline__ bool shard_spin(const unsigned long long* p, unsigned long long want) {
  if (ld_acquire_sys_u64(p) == want) return true;
  const unsigned long long t0 = global_timer_ns();
  while (ld_acquire_sys_u64(p) != want) {
    if (global_timer_ns() - t0 > kShardTimeoutNs) return false;
    __nanosleep(100);
  }
  return true;
}
__device__ __forceinline__ unsigned long long shard_tag(const DevState* s, unsigned int seq) {
  return ((unsigned long long)s->epoch << 32) | (unsigned long long)seq;
}
__device__ __forceinline__ int shard_slot(const DevState* s, unsigned int xseq) {
  return (int)(((s->epoch & 1u) * kMailSlots + (xseq & (kMailSlots - 1))) * kMaxWorld);
}

// ---- sums: post this rank's partial sums of the reduction point that follows s->xseq completed ones (one thread) ----
// Values to every rank first, ONE system-scope fence, then the tags (fence + relaxed store = release): the cost of a
// reduction point does not grow with a fence per peer.
// (small arguments by value: a reference to the kernel's Ctx would force a stack copy of the whole parameter block)
__device__ __noinline__ void shard_post(const DevState* s, const ShardCtx* sh, double v0, double v1) {
  const unsigned int xseq = s->xseq;
  const unsigned long long tag = shard_tag(s, xseq + 1u);
  const int slot = shard_slot(s, xseq) + sh->rank;
  for (int r = 0; r < sh->world; ++r) {
    Mail* m = sh->peer_mbox[r] + slot;
    *reinterpret_cast<volatile double*>(&m->v0) = v0;
    *reinterpret_cast<volatile double*>(&m->v1) = v1;
  }
  __threadfence_system();
  for (int r = 0; r < sh->world; ++r) *reinterpret_cast<volatile unsigned long long*>(&(sh->peer_mbox[r] + slot)->tag) = tag;
}

// ---- halo: wait until both neighbours have completed their push with sequence number seq (whole block) ----
__device__ __forceinline__ void shard_wait_halo(const Ctx& c, unsigned int seq) {
  const ShardCtx* sh = c.sh;
  if (threadIdx.x == 0) {
    DevState* s = c.st;
    const unsigned long long tag = shard_tag(s, seq);
    bool ok = true;
    if (sh->rank > 0) ok = shard_spin(sh->flags + 0, tag);
    if (ok && sh->rank + 1 < sh->world) ok = shard_spin(sh->flags + 1, tag);
    if (!ok) { s->status = -3; s->done = 1; }
  }
  __syncthreads();
}
__device__ __forceinline__ void shard_wait_halo_warp(const Ctx& c, unsigned int seq) {  // one warp (pipelined mat-vec)
  const ShardCtx* sh = c.sh;
  if ((threadIdx.x & 31) == 0) {
    DevState* s = c.st;
    const unsigned long long tag = shard_tag(s, seq);
    bool ok = true;
    if (sh->rank > 0) ok = shard_spin(sh->flags + 0, tag);
    if (ok && sh->rank + 1 < sh->world) ok = shard_spin(sh->flags + 1, tag);
    if (!ok) { s->status = -3; s->done = 1; }
  }
  __syncwarp();
}

// ---- halo: after this block's pushes, count it; the block that arrives last raises the neighbours' flags ----
__device__ __forceinline__ void shard_signal_halo(const Ctx& c, unsigned int seq, unsigned int* counter, int nb) {
  __syncthreads();  // every thread's peer stores are issued
  if (threadIdx.x == 0) {
    __threadfence_system();
    if (atomicAdd(counter, 1u) == (unsigned int)nb - 1u) {
      *counter = 0u;
      __threadfence_system();
      const ShardCtx* sh = c.sh;
      const unsigned long long tag = shard_tag(c.st, seq);
      if (sh->peer_flag_lo) st_release_sys_u64(sh->peer_flag_lo, tag);
      if (sh->peer_flag_hi) st_release_sys_u64(sh->peer_flag_hi, tag);
    }
  }
}

// ---- copy a caller's block of a vector into the internal p vector of the same precision and push its halo ----
// (set-up: x0 for r0 = b - A x0; after the loop: x for the true residual; amp_spmv_sharded)
template <int P>
__device__ __forceinline__ void shard_load_p_body(const Ctx& c, const typename Store<P>::T* src) {
  using T = typename Store<P>::T;
  T* dst = pvec<P>(c);
  const HaloPush<T> h = halo_push_of<P>(c);
  const int64_t stride = (int64_t)gridDim.x * blockDim.x;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < c.npad; i += stride) {
    const T v = (i < c.n) ? src[i] : T(0);
    dst[i] = v;
    if (i < h.send_lo) h.lo[i] = v;
    if (i >= h.hi0 && i < h.n) h.hi[i - h.hi0] = v;
  }
}
__global__ void __launch_bounds__(kVecThreads) k_shard_load_p(const Ctx c, const void* src, int prec, unsigned int seq) {
  if (prec == P64) shard_load_p_body<P64>(c, static_cast<const double*>(src));
  else if (prec == P32) shard_load_p_body<P32>(c, static_cast<const float*>(src));
  else shard_load_p_body<P16>(c, static_cast<const __half*>(src));
  if (c.sh != nullptr) shard_signal_halo(c, seq, &c.st->counter[3], (int)gridDim.x);
}

// ---- the scalar step of a reduction point, from the partial sums of all ranks ----
enum { kEpiSetup = 0, kEpiRho = 1, kEpiGamma = 2, kEpiDelta = 3, kEpiDeltaLagged = 4, kEpiFinal = 5 };

// one thread: wait until the entries of all ranks carry the tag of the reduction point that follows s->xseq completed
// ones, add them in rank order (the same sum on every rank), count the point, run the scalar step
__device__ __noinline__ void shard_collect_and_step(const EpiCtx ec, const ShardCtx* sh, int which) {
  DevState* s = ec.st;
  const unsigned int xseq = s->xseq;
  const unsigned long long tag = shard_tag(s, xseq + 1u);
  const Mail* m = sh->mbox + shard_slot(s, xseq);
  double t0 = 0.0, t1 = 0.0;
  bool ok = true;
  for (int r = 0; r < sh->world && ok; ++r) ok = shard_spin_relaxed(&m[r].tag, tag);
  __threadfence_system();  // relaxed loads + fence = acquire: the values below are the ones posted before the tags
  for (int r = 0; r < sh->world; ++r) {  // rank order: the same sum on every rank
    t0 += *reinterpret_cast<const volatile double*>(&m[r].v0);
    t1 += *reinterpret_cast<const volatile double*>(&m[r].v1);
  }
  s->xseq = xseq + 1u;
  if (!ok) {
    s->status = -3; s->done = 1;
    set_loop_cond(ec, 0);
    return;
  }
  switch (which) {
    case kEpiSetup: epi_setup(ec, t0, t1); break;
    case kEpiRho: epi_rho(ec, t0); break;
    case kEpiGamma: epi_gamma(ec, t0); break;
    case kEpiDelta: epi_delta(ec, t0); break;
    case kEpiDeltaLagged: epi_delta_lagged(ec, t0, t1); break;
    default: s->relres_true = (s->bnorm > 0.0) ? sqrt(t0) / s->bnorm : 0.0; break;
  }
}

// what the thread that completes a grid reduction does in a sharded solve: publish, and — when the ranks run
// concurrently — collect and step at once (no extra kernel on the critical path)
__device__ __forceinline__ void shard_reduce_point(const Ctx& c, int which, double v0, double v1) {
  shard_post(c.st, c.sh, v0, v1);
  if (c.sh->inline_epi) shard_collect_and_step(epi_ctx(c), c.sh, which);
}

// the same step as a kernel of its own (one thread), for ranks that share a device: launched for every rank AFTER the
// reducing kernels of all ranks, so that the wait finds every entry in place
__global__ void __launch_bounds__(32) k_epi(const Ctx c, int which) {
  pdl_launch_dependents();
  pdl_wait();
  if (threadIdx.x != 0) return;
  DevState* s = c.st;
  const bool in_loop = which >= kEpiRho && which <= kEpiDeltaLagged;
  if (in_loop && s->done) {  // the reducing kernel returned without posting (converged, breakdown, time-out)
    if (which == kEpiDelta || which == kEpiDeltaLagged) set_loop_cond(epi_ctx(c), 0);
    return;
  }
  if (which == kEpiFinal && s->zero_x) return;  // b = 0 (identical on all ranks): nothing was posted
  shard_collect_and_step(epi_ctx(c), c.sh, which);
}

}  // namespace amp
