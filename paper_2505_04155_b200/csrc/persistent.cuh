// persistent.cuh — the whole AMP-PCG loop as ONE cooperative kernel (north_star: "a persistent
// cooperative kernel for small n"): every block stays resident and the four synchronisation
// points of an iteration (rho, p complete, gamma, delta; Alg 4.1 lines 6, 10, 13, 17) are grid
// barriers instead of kernel boundaries.
//
// What makes the barrier cheap: the loop scalars are REPLICATED.  Every block keeps its own copy
// of the DevState block in shared memory; at a reduction every block publishes its partial sum,
// arrives (one red.release), waits until all have arrived (one polled ld.acquire), then adds ALL
// partials itself in index order and runs the scalar epilogue on its own copy.  All blocks add
// the same numbers in the same order, so they take identical decisions (precision switches, stop,
// breakdown) without any broadcast: one barrier = arrive + poll + one read of the partials, no
// "last block computes, then releases the others" round trip.  Block 0 writes the state back for
// the host when the loop ends.  The phases are the same device functions the stand-alone kernels
// call; p is gathered with plain (coherent) loads because it is written inside this kernel.
#pragma once
#include <cstddef>

#include "kernels.cuh"

namespace amp {

constexpr int kPersistBIF = 96;  // bytes of loads in flight per thread of the vector phases (register budget: 64)

__device__ __forceinline__ unsigned int ld_acquire_u32(const unsigned int* p) {
  unsigned int v;
  asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ void red_release_add_u32(unsigned int* p, unsigned int v) {
  asm volatile("red.release.gpu.global.add.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}

// Grid barrier fused with a deterministic all-reduce.  `arrivals` counts up over the whole solve
// (reset by the set-up kernel); `target` is this block's running count of expected arrivals.
// SUM = false: plain barrier.  Returns the total in warp 0 (SUM = true).
// `partials` must be a different array at consecutive barriers (a fast block may already publish
// its next partial while a slow one still reads this one).
template <bool SUM, int NT = kPersistThreads>
__device__ __forceinline__ double grid_all_sum(double v, double* partials, unsigned int* arrivals, unsigned int& target,
                                               int bid, int nb, double* red) {
  double bs = 0.0;
  if (SUM) bs = block_sum<NT>(v, red);  // every thread is past its phase's memory accesses
  else __syncthreads();
  target += (unsigned int)nb;
  if (threadIdx.x == 0) {
    if (SUM) __stcg(partials + bid, bs);
    red_release_add_u32(arrivals, 1u);
    while ((int)(ld_acquire_u32(arrivals) - target) < 0) { }
  }
  __syncthreads();
  double tot = 0.0;
  if (SUM) {
    double a = 0.0;
    for (int i = threadIdx.x; i < nb; i += NT) a += __ldcg(partials + i);
    tot = block_sum<NT>(a, red);
  }
  return tot;
}

// the same for two sums (lagged variant: delta^2 and rho), partials interleaved; totals valid in warp 0
template <int NT = kPersistThreads>
__device__ __forceinline__ void grid_all_sum2(double v0, double v1, double* partials, unsigned int* arrivals, unsigned int& target,
                                              int bid, int nb, double* red, double& t0, double& t1) {
  const double b0 = block_sum<NT>(v0, red);
  const double b1 = block_sum<NT>(v1, red);
  target += (unsigned int)nb;
  if (threadIdx.x == 0) {
    __stcg(partials + 2 * bid, b0);
    __stcg(partials + 2 * bid + 1, b1);
    red_release_add_u32(arrivals, 1u);
    while ((int)(ld_acquire_u32(arrivals) - target) < 0) { }
  }
  __syncthreads();
  double a0 = 0.0, a1 = 0.0;
  for (int i = threadIdx.x; i < nb; i += NT) { a0 += __ldcg(partials + 2 * i); a1 += __ldcg(partials + 2 * i + 1); }
  t0 = block_sum<NT>(a0, red);
  t1 = block_sum<NT>(a1, red);
}

// out-of-line copies of the phase dispatchers: each gets its own register allocation instead of
// one allocation for the union of all precision variants
__device__ __noinline__ double pz(const Ctx& c, int rs, int ur, int uz, double omega, int bid, int nb) {
  return dispatch_z<kPersistBIF>(c, rs, ur, uz, omega, bid, nb);
}
__device__ __noinline__ void pp(const Ctx& c, int ps, int uz, int ur, double beta, bool first, int bid, int nb) {
  dispatch_p<kPersistBIF>(c, ps, uz, ur, beta, first, bid, nb);
}
__device__ __noinline__ double ps_(const Ctx& c, int ur, int uz, int bid, int nb, double* red) {
  return dispatch_spmv<true, kPersistThreads>(c, ur, uz, 0, bid, nb, red);
}
__device__ __noinline__ double pxr(const Ctx& c, int ur, int uz, double alpha, double* x, int bid, int nb) {
  return dispatch_xr<kPersistBIF>(c, ur, uz, alpha, x, bid, nb);
}

__device__ __noinline__ void pxrz(const Ctx& c, int ur, int urn, int uz, int uzn, double alpha, double omega_n, double* x,
                                  int bid, int nb, double& rr, double& rz) {
  dispatch_xrz<kPersistBIF>(c, ur, urn, uz, uzn, alpha, omega_n, x, bid, nb, rr, rz);
}

__global__ void __launch_bounds__(kPersistThreads, kPersistMinBlocks) k_persistent(const Ctx cparam) {
  __shared__ double red[32];
  __shared__ DevState ls;  // this block's replica of the loop scalars
  // The out-of-line phase dispatchers take the context by reference.  A reference to the kernel parameter would make
  // every thread keep a 600-byte copy of it on its stack and read every pointer from local memory (round 1: 1.7 KB of
  // stack, 1800 local loads and stores); one copy per block in shared memory is read with plain LDS instead.
  __shared__ Ctx cshared;
  const int bid = blockIdx.x, nb = gridDim.x;
  if (threadIdx.x == 0) cshared = cparam;  // (a plain assignment: taking the parameter's address would spill it again)
  const Ctx& c = cshared;
  {  // replicate the state block (written by the host and the set-up kernel before this launch)
    const int* src = reinterpret_cast<const int*>(cparam.st);
    int* dst = reinterpret_cast<int*>(&ls);
    for (int i = threadIdx.x; i < (int)(sizeof(DevState) / sizeof(int)); i += kPersistThreads) dst[i] = __ldcg(src + i);
  }
  __syncthreads();
  DevState* s = &ls;
  EpiCtx ec = epi_ctx(c);
  ec.st = s;
  ec.use_cond = 0;
  unsigned int* arrivals = &c.st->bar_count;
  unsigned int target = 0u;
  double* x = s->x;
  if (s->amp && s->scale_mode == 4) {
    // lagged variant (reading R17): z_0, rho_0 once, then three phases and three barriers per iteration
    if (!s->done) {
      const double v = pz(c, s->r_store, s->ur, s->uz, s->omega, bid, nb);
      const double t = grid_all_sum<true>(v, c.partials + 0 * kMaxGrid, arrivals, target, bid, nb, red);
      if (threadIdx.x == 0) epi_rho(ec, t);
      __syncthreads();
    }
    while (!s->done) {
      pp(c, s->p_store, s->uz, s->ur, s->beta, s->k == 0, bid, nb);                                  // a3
      grid_all_sum<false>(0.0, nullptr, arrivals, target, bid, nb, red);
      const double v = ps_(c, s->ur, s->uz, bid, nb, red);                                           // a4
      const double t = grid_all_sum<true>(v, c.partials + 1 * kMaxGrid, arrivals, target, bid, nb, red);
      if (threadIdx.x == 0) epi_gamma(ec, t);
      __syncthreads();
      if (s->done) break;  // breakdown
      double rr = 0.0, rz = 0.0, t0, t1;
      pxrz(c, s->ur, s->ur_n, s->uz, s->uz_n, s->alpha, s->omega_n, x, bid, nb, rr, rz);              // a5 + a2
      grid_all_sum2(rr, rz, c.partials + 2 * kMaxGrid, arrivals, target, bid, nb, red, t0, t1);
      if (threadIdx.x == 0) epi_delta_lagged(ec, t0, t1);
      __syncthreads();
    }
  }
  while (!s->done) {
    const int rs = s->r_store, ps = s->p_store, ur = s->ur, uz = s->uz;
    const bool first = (s->k == 0);
    double v = pz(c, rs, ur, uz, s->omega, bid, nb);                                                 // a2
    double t = grid_all_sum<true>(v, c.partials + 0 * kMaxGrid, arrivals, target, bid, nb, red);
    if (threadIdx.x == 0) epi_rho(ec, t);
    __syncthreads();
    pp(c, ps, uz, ur, s->beta, first, bid, nb);                                                      // a3
    grid_all_sum<false>(0.0, nullptr, arrivals, target, bid, nb, red);
    v = ps_(c, ur, uz, bid, nb, red);                                                                // a4
    t = grid_all_sum<true>(v, c.partials + 1 * kMaxGrid, arrivals, target, bid, nb, red);
    if (threadIdx.x == 0) epi_gamma(ec, t);
    __syncthreads();
    if (s->done) break;  // breakdown
    v = pxr(c, ur, uz, s->alpha, x, bid, nb);                                                        // a5
    t = grid_all_sum<true>(v, c.partials + 2 * kMaxGrid, arrivals, target, bid, nb, red);
    if (threadIdx.x == 0) epi_delta(ec, t);
    __syncthreads();
  }
  if (bid == 0) {  // publish the result scalars (not the barrier counter: other blocks may still poll it)
    __syncthreads();
    int* dst = reinterpret_cast<int*>(c.st);
    const int* src = reinterpret_cast<const int*>(&ls);
    // the FP16 counters of the counting build are accumulated in global memory only (other blocks may still be adding)
    const int skip0 = (int)(offsetof(DevState, fp16_subnormal) / sizeof(int));
    const int skip1 = (int)((offsetof(DevState, bar_pad) + sizeof(unsigned int)) / sizeof(int));
    for (int i = threadIdx.x; i < (int)(sizeof(DevState) / sizeof(int)); i += kPersistThreads)
      if (i < skip0 || i >= skip1) dst[i] = src[i];
  }
}

inline void persistent_configure(int num_sms, int* grid, int* ok) {
  *grid = 0;
  *ok = 0;
  int occ = 0, coop = 0, dev = 0;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, dev);
  if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k_persistent, kPersistThreads, 0) != cudaSuccess) {
    cudaGetLastError();
    return;
  }
  if (!coop || occ < 1) return;
  *grid = num_sms * occ;
  if (*grid > kMaxGrid) *grid = (kMaxGrid / num_sms) * num_sms;
  *ok = 1;
}

inline int persistent_launch(const Ctx& c, int grid, cudaStream_t st) {
  Ctx cc = c;
  cc.use_cond = 0;
  void* args[] = {(void*)&cc};
  return (int)cudaLaunchCooperativeKernel((void*)k_persistent, dim3(grid), dim3(kPersistThreads), args, 0, st);
}

}  // namespace amp
