// spmv_pipe.cuh — step a4 (q = A p in u_r, gamma = q^T p; Alg 4.1 lines 11-13) as a persistent,
// bulk-copy pipelined kernel for matrices whose SELL-32 slices are all diagonal-aligned (stencil / structured-grid
// matrices: c1-c4 of BASELINE.json).
//
// Why a second SpMV kernel.  With the per-entry index stream gone (aligned slices, spmv.cuh) the direct kernel of the
// u_r = FP32 phase is no longer HBM- but latency-bound: a lane's value loads, its gathers of p and its fma chain
// alternate, so a warp has bytes in flight only part of the time (ncu, c4: DRAM 56 %, issue slots 58 % busy, 18.5
// instructions per entry).  Here the HBM stream is decoupled from the arithmetic:
//   * one block per SM, resident for the whole mat-vec, owns a contiguous range of slices;
//   * ONE producer thread streams that range with cp.async.bulk (the TMA engine, no tensor map needed: the value
//     stream of consecutive slices is one contiguous run) into a ring of shared-memory stages, completion signalled
//     on an mbarrier per stage, L2 evict-first so the matrix does not displace the vectors; the slice table and the
//     per-entry diagonal offsets of the stage's slices ride along in two more small bulk copies, so a consumer has no
//     dependent global load left except the gathers of p;
//   * 15 consumer warps in 3 groups of 5 (stage i belongs to group i mod 3) take the slices of their stages
//     round-robin, read values with conflict-free 128-bit LDS and keep
//     ONE fma chain per row in stored (= CSR) order, so q is bit-identical to the direct kernel and to the oracle;
//   * the work vectors p are allocated with a zero guard band on both sides, so col = row + offset needs no clamp
//     (explicit zeros of boundary rows may point outside [0, n): they read a guard zero).
// With 6 x 32 KB stages about 150 KB per SM are in flight whatever the consumers do.
// Under programmatic dependent launch the producer starts streaming the (constant) matrix BEFORE griddepcontrol.wait,
// i.e. while the p update of the same iteration is still finishing.
#pragma once
#include "async_copy.cuh"
#include "shard.cuh"
#include "spmv.cuh"

namespace amp {

constexpr int kPipeConsumerWarps = 15;                       // + 1 producer warp = 512 threads: 128 registers each
constexpr int kPipeGroups = 3;                               // consumer warps work in 3 groups of 5: stage i belongs to group
constexpr int kPipeGroupWarps = kPipeConsumerWarps / kPipeGroups;  // i mod 3, so a warp visits a third of the stages
constexpr int kPipeThreads = (kPipeConsumerWarps + 1) * 32;  // + one producer warp
constexpr int kPipeChunkW = 256;                             // max summed slice width of one stage
constexpr int kPipeChunkSlices = 64;                         // max slices of one stage
constexpr int kPipeValueBytes = 6 * 32 * kPipeChunkW * 4;    // 196608: 6 FP32 stages
constexpr int kPipeMaxStages = 6;
constexpr int kPipeBaseInts = kPipeChunkW + 8;               // staged diagonal offsets (16-byte aligned window)
constexpr int kPipeWptrInts = kPipeChunkSlices + 8;          // staged slice table window
constexpr int kPipeSmemBytes = kPipeValueBytes + kPipeMaxStages * 4 * (kPipeBaseInts + kPipeWptrInts) +
                               kPipeMaxStages * 16 /* headers */ + 2 * kPipeMaxStages * 8 /* mbarriers */;
constexpr int kPipeMaxGuard = 1 << 22;                       // elements of zero guard band per side we are willing to pay

// gather of p[j] converted to the working type; j may be negative or >= n (guard band)
// COH = true (sharded solve): plain coherent loads, the halo entries were stored by a peer GPU while this kernel ran
template <bool COH, class A, class PT> __device__ __forceinline__ A pipe_gather(const PT* pl, int off) { return gatherA<COH>(A(0), pl, off); }

// one slice from shared memory: this lane's row sum, ONE fma chain in stored order.
// The quads of a slice are taken in trips of up to QT; a trip of NQ quads is straight-line code (template), so only
// instructions of entries that exist are issued (a predicated-off instruction still costs an issue slot): about 5
// per entry — diagonal offset (warp-uniform LDS), address, gather, convert, fma — plus a 128-bit LDS per 4 values.
// All value loads and all gathers of a trip are issued before its first fma.
template <class A> struct PipeTrip;
template <> struct PipeTrip<float> { static constexpr int QT = 4; };
template <> struct PipeTrip<double> { static constexpr int QT = 4; };

template <class A> __device__ __forceinline__ void pipe_ld_quad(const A* sv, int qd, int lane, A (&v)[4]);
template <> __device__ __forceinline__ void pipe_ld_quad<float>(const float* sv, int qd, int lane, float (&v)[4]) {
  const float4 t = *reinterpret_cast<const float4*>(sv + qd * 128 + lane * 4);
  v[0] = t.x; v[1] = t.y; v[2] = t.z; v[3] = t.w;
}
template <> __device__ __forceinline__ void pipe_ld_quad<double>(const double* sv, int qd, int lane, double (&v)[4]) {
  const double2 t0 = *reinterpret_cast<const double2*>(sv + qd * 128 + lane * 2);
  const double2 t1 = *reinterpret_cast<const double2*>(sv + qd * 128 + 64 + lane * 2);
  v[0] = t0.x; v[1] = t0.y; v[2] = t1.x; v[3] = t1.y;
}

template <bool COH, int NQ, class A, class PT>
__device__ __forceinline__ A pipe_trip(const A* sv, const int* sb, int cq, int lane, const PT* pl, A acc) {
  A v[NQ][4], x[NQ][4];
#pragma unroll
  for (int t = 0; t < NQ; ++t) {
    pipe_ld_quad<A>(sv, cq + t, lane, v[t]);
#pragma unroll
    for (int u = 0; u < 4; ++u) x[t][u] = pipe_gather<COH, A>(pl, sb[4 * (cq + t) + u]);
  }
#pragma unroll
  for (int t = 0; t < NQ; ++t) {
#pragma unroll
    for (int u = 0; u < 4; ++u) acc = fma(v[t][u], x[t][u], acc);
  }
  return acc;
}

template <bool COH, class A, class PT>
__device__ __forceinline__ A pipe_slice_sum(const A* sv, const int* sb, int w, int lane, const PT* pl) {
  constexpr int QT = PipeTrip<A>::QT;
  const int a = w >> 2;
  A acc = 0;
  int cq = 0;
  for (; cq + QT <= a; cq += QT) acc = pipe_trip<COH, QT, A, PT>(sv, sb, cq, lane, pl, acc);
  // the last trip: fewer than QT quads, then the pair and the single of the 4a + 2b + c cut
  const bool hp = (w & 2) != 0, hs = (w & 1) != 0;
  A vp[2], xp[2], vs, xs;
  if (hp) {
    if constexpr (sizeof(A) == 4) {
      const float2 t = *reinterpret_cast<const float2*>(sv + a * 128 + lane * 2);
      vp[0] = t.x; vp[1] = t.y;
    } else {
      const double2 t = *reinterpret_cast<const double2*>(sv + a * 128 + lane * 2);
      vp[0] = t.x; vp[1] = t.y;
    }
    xp[0] = pipe_gather<COH, A>(pl, sb[4 * a]);
    xp[1] = pipe_gather<COH, A>(pl, sb[4 * a + 1]);
  }
  if (hs) {
    vs = sv[a * 128 + (hp ? 64 : 0) + lane];
    xs = pipe_gather<COH, A>(pl, sb[w - 1]);
  }
  const int rem = a - cq;
  if constexpr (QT >= 4) {
    if (rem == 3) acc = pipe_trip<COH, 3, A, PT>(sv, sb, cq, lane, pl, acc);
    else if (rem == 2) acc = pipe_trip<COH, 2, A, PT>(sv, sb, cq, lane, pl, acc);
    else if (rem == 1) acc = pipe_trip<COH, 1, A, PT>(sv, sb, cq, lane, pl, acc);
  } else {
    if (rem == 1) acc = pipe_trip<COH, 1, A, PT>(sv, sb, cq, lane, pl, acc);
  }
  if (hp) { acc = fma(vp[0], xp[0], acc); acc = fma(vp[1], xp[1], acc); }
  if (hs) acc = fma(vs, xs, acc);
  return acc;
}

// per-stage descriptor, built once in create(): first slice, first entry column (cumulative width), of stage ch;
// entry nchunks closes the list
struct PipeChunk { int32_t s0, w0; };

template <int UR, bool COH = false, class PT, class PG>
__device__ __forceinline__ double pipe_body(const Ctx& c, const PT* p, const PG* pg, typename Store<UR>::T* q, unsigned char* smem,
                                            unsigned int halo_seq) {
  using A = typename SpmvT<UR>::A;
  constexpr int STAGE = 32 * kPipeChunkW * (int)sizeof(A);
  constexpr int NST = kPipeValueBytes / STAGE;
  static_assert(NST >= 2 && NST <= kPipeMaxStages, "stages");
  unsigned char* sval = smem;
  int* sbase = reinterpret_cast<int*>(smem + kPipeValueBytes);
  int* swptr = sbase + kPipeMaxStages * kPipeBaseInts;
  int4* shdr = reinterpret_cast<int4*>(swptr + kPipeMaxStages * kPipeWptrInts);
  uint64_t* full = reinterpret_cast<uint64_t*>(shdr + kPipeMaxStages);
  uint64_t* empty = full + kPipeMaxStages;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int bid = blockIdx.x;
  const int c0 = __ldg(c.pipe_blk_chunk + bid), c1 = __ldg(c.pipe_blk_chunk + bid + 1);
  const PipeChunk* __restrict__ desc = reinterpret_cast<const PipeChunk*>(c.pipe_chunks);
  if (threadIdx.x == 0) {
#pragma unroll
    for (int s = 0; s < NST; ++s) { mbar_init(full + s, 1); mbar_init(empty + s, kPipeGroupWarps); }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  double gsum = 0.0;
  const int n = (int)c.n;
  if (warp == kPipeConsumerWarps) {
    // ---- producer: the matrix is constant, so streaming starts before the predecessor kernel has finished ----
    if (lane == 0) {
      const A* vals = sell_vals<UR>(c);
      PipeChunk d0 = desc[c0], d1 = desc[min(c0 + 1, c1)];
      for (int ch = c0; ch < c1; ++ch) {
        const PipeChunk d2 = desc[min(ch + 2, c1)];  // descriptor loads stay two stages ahead of their use
        const int i = ch - c0, st = i % NST, round = i / NST;
        if (round > 0) mbar_wait(empty + st, (uint32_t)((round - 1) & 1));
        const uint32_t bytes_v = (uint32_t)(d1.w0 - d0.w0) * 32u * (uint32_t)sizeof(A);
        const int b0 = d0.w0 & ~3, nbi = ((d1.w0 + 3) & ~3) - b0;
        const int p0 = d0.s0 & ~3, npi = ((d1.s0 + 1 + 3) & ~3) - p0;
        shdr[st] = make_int4(d0.s0, d1.s0, d0.w0, 0);
        mbar_arrive_expect_tx(full + st, bytes_v + 4u * (uint32_t)(nbi + npi));
        if (bytes_v) bulk_g2s_stream(sval + (size_t)st * STAGE, vals + (size_t)d0.w0 * 32, bytes_v, full + st);
        if (nbi) bulk_g2s(sbase + st * kPipeBaseInts, c.sell_base + b0, 4u * (uint32_t)nbi, full + st);
        bulk_g2s(swptr + st * kPipeWptrInts, c.sell_wptr + p0, 4u * (uint32_t)npi, full + st);
        d0 = d1;
        d1 = d2;
      }
    }
  } else {
    pdl_wait();  // p (and q's previous readers) belong to the predecessor kernels
    if (c.sh != nullptr) shard_wait_halo_warp(c, halo_seq);  // row-sharded solve: the neighbours' entries of p have arrived
    static_assert(NST % kPipeGroups == 0, "a stage slot must always serve the same group");
    const int grp = warp % kPipeGroups, wg = warp / kPipeGroups;  // this warp's group and its rank inside it
    for (int ch = c0 + grp; ch < c1; ch += kPipeGroups) {
      const int i = ch - c0, st = i % NST, round = i / NST;
      mbar_wait(full + st, (uint32_t)(round & 1));
      const int4 hd = shdr[st];
      const A* sv0 = reinterpret_cast<const A*>(sval + (size_t)st * STAGE);
      const int* sb0 = sbase + st * kPipeBaseInts - (hd.z & ~3);
      const int* sw0 = swptr + st * kPipeWptrInts - (hd.x & ~3);
      for (int sl = hd.x + wg; sl < hd.y; sl += kPipeGroupWarps) {
        const int w0 = sw0[sl] & ~kWptrFlags, w = (sw0[sl + 1] & ~kWptrFlags) - w0;
        const int row = sl * 32 + lane;
        const PT* pl = p + row;
        const double pi = gather64<COH>(pg, row);  // the stored p_i (u_z precision) for gamma
        A acc = 0;
        if (w > 0) acc = pipe_slice_sum<COH, A, PT>(sv0 + (size_t)(w0 - hd.z) * 32, sb0 + w0, w, lane, pl);
        if (row < n) {
          q[row] = acc;
          gsum = fma(pi, (double)acc, gsum);
        }
      }
      __syncwarp();
      if (lane == 0) mbar_arrive(empty + st);
    }
  }
  return gsum;
}

// the loop's SpMV kernel of the u_r = FP32 phases for eligible matrices; dynamic shared memory: kPipeSmemBytes.
// (The u_r = FP64 phases stay with the direct kernel, which already streams at the copy rate there: measured on c4,
// 303 us direct against 327-349 us pipelined, profiles/r02.md.  Both kernels sit in the loop; the one whose phase it
// is not returns at once.)
template <bool COH>
__device__ __forceinline__ void spmv_pipe_kernel(const Ctx& c, int zmode, unsigned char* pipe_smem, double* red) {
  DevState* s = c.st;
  pdl_launch_dependents();
  // Single-GPU loop: done, ur, uz, k were last written by the final kernel of the PREVIOUS iteration (epi_delta), which had
  // completed before the first kernel of this iteration started (plain dependency), and NOTHING between that kernel and
  // this one writes them (epi_rho writes rho / beta only) — an invariant this early read rests on: safe before the wait,
  // so the producer warp streams the matrix while the p update is still finishing.
  // Sharded loop (COH): the block that completes a cross-rank reduction inside k_z / k_p_sh may set done and status
  // (a peer timed out, breakdown on another rank), so there the state is read only after the predecessors have finished.
  if (COH) pdl_wait();
  const int ur = s->ur, uz = s->uz;
  if (s->done || ur != P32) { pdl_wait(); return; }
  const unsigned int hseq = (unsigned int)s->k + 1u;
  double v;
  if (zmode) {  // q = A z inside the Chebyshev-Jacobi preconditioner
    if (uz == P16) v = pipe_body<P32, COH>(c, c.z16, c.z16, c.q32, pipe_smem, hseq);
    else if (uz == P32) v = pipe_body<P32, COH>(c, c.z32, c.z32, c.q32, pipe_smem, hseq);
    else v = pipe_body<P32, COH>(c, c.z64, c.z64, c.q32, pipe_smem, hseq);  // RN32(z_j) per gathered entry
    pdl_wait();
    return;
  }
  if (uz == P16) v = pipe_body<P32, COH>(c, c.p16, c.p16, c.q32, pipe_smem, hseq);
  else if (uz == P32) v = pipe_body<P32, COH>(c, c.p32, c.p32, c.q32, pipe_smem, hseq);
  else v = pipe_body<P32, COH>(c, c.p32, c.p64, c.q32, pipe_smem, hseq);  // gathers the FP32 copy RN32(p) written by the p update
  pdl_wait();  // (the producer warp has not waited yet) before touching the reduction scratch shared with other kernels
  if (c.defer_gamma) { grid_publish<kPipeThreads>(v, c.partials + 1 * kMaxGrid, blockIdx.x, red); return; }
  grid_reduce<kPipeThreads>(v, c.partials + 1 * kMaxGrid, &s->counter[1], blockIdx.x, gridDim.x, red,
                            [&](double tot) { if (c.sh != nullptr) shard_reduce_point(c, kEpiGamma, tot, 0.0); else epi_gamma(epi_ctx(c), tot); });
}

__global__ void __launch_bounds__(kPipeThreads, 1) k_spmv_pipe(const Ctx c, int zmode) {
  extern __shared__ __align__(128) unsigned char pipe_smem[];
  __shared__ double red[32];
  spmv_pipe_kernel<false>(c, zmode, pipe_smem, red);
}
// the same kernel for a handle attached to a shard group (c.sh != nullptr): the halo bands of p are filled by peer GPUs
// while this kernel may already be running, and ld.global.nc is not ordered behind the acquire of the halo flag
__global__ void __launch_bounds__(kPipeThreads, 1) k_spmv_pipe_sh(const Ctx c, int zmode) {
  extern __shared__ __align__(128) unsigned char pipe_smem[];
  __shared__ double red[32];
  spmv_pipe_kernel<true>(c, zmode, pipe_smem, red);
}

}  // namespace amp
