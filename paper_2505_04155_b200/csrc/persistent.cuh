// persistent.cuh — the whole AMP-PCG loop as ONE cooperative kernel (north_star: "a persistent
// cooperative kernel for small n"): every block stays resident, the three reductions of an
// iteration (rho, gamma, delta; Alg 4.1 lines 6, 13, 17) double as grid barriers whose last
// arriver runs the scalar epilogue, and one plain barrier publishes p before the gather.
// The phases are the same device functions the stand-alone kernels call.
#pragma once
#include "kernels.cuh"

namespace amp {


__device__ __forceinline__ unsigned int ld_acquire_u32(const unsigned int* p) {
  unsigned int v;
  asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ void st_release_u32(unsigned int* p, unsigned int v) {
  asm volatile("st.release.gpu.global.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}
template <class T> __device__ __forceinline__ T ldv(const T* p) { return __ldcg(p); }  // L2, never a stale L1 line

// Grid barrier fused with a deterministic reduction: blocks publish partial sums and take a
// ticket; the last arriver adds the partials in index order, runs epi(total) on one thread,
// then opens the barrier by bumping the generation.  SUM = false: plain barrier.
template <bool SUM, class Epi>
__device__ __forceinline__ void grid_sync_reduce(double v, double* partials, DevState* s, int bid, int nb,
                                                 double* red, Epi epi) {
  __shared__ int s_last;
  __shared__ unsigned int s_gen;
  double bs = 0.0;
  if (SUM) bs = block_sum<kPersistThreads>(v, red);
  else __syncthreads();
  if (threadIdx.x == 0) {
    if (SUM) __stcg(partials + bid, bs);
    const unsigned int gen = ld_acquire_u32(&s->bar_gen);
    __threadfence();
    const unsigned int t = atomicAdd(&s->bar_count, 1u);
    s_last = (t == (unsigned int)nb - 1u);
    s_gen = gen;
  }
  __syncthreads();
  if (s_last) {
    double tot = 0.0;
    if (SUM) {
      __threadfence();
      double a = 0.0;
      for (int i = threadIdx.x; i < nb; i += kPersistThreads) a += __ldcg(partials + i);
      tot = block_sum<kPersistThreads>(a, red);
    }
    if (threadIdx.x == 0) {
      if (SUM) epi(tot);
      s->bar_count = 0u;
      __threadfence();
      st_release_u32(&s->bar_gen, s_gen + 1u);
    }
  } else if (threadIdx.x == 0) {
    while (ld_acquire_u32(&s->bar_gen) == s_gen) { }
    __threadfence();
  }
  __syncthreads();
}

// out-of-line copies of the phase dispatchers: each gets its own register allocation instead of
// one allocation for the union of all precision variants
__device__ __noinline__ double pz(const Ctx& c, int rs, int ur, int uz, double omega, int bid, int nb) {
  return dispatch_z(c, rs, ur, uz, omega, bid, nb);
}
__device__ __noinline__ void pp(const Ctx& c, int ps, int uz, double beta, bool first, int bid, int nb) {
  dispatch_p(c, ps, uz, beta, first, bid, nb);
}
__device__ __noinline__ double ps_(const Ctx& c, int ur, int uz, int bid, int nb, double* red) {
  return dispatch_spmv<true, kPersistThreads>(c, ur, uz, bid, nb, red);
}
__device__ __noinline__ double pxr(const Ctx& c, int ur, int uz, double alpha, double* x, int bid, int nb) {
  return dispatch_xr(c, ur, uz, alpha, x, bid, nb);
}

__global__ void __launch_bounds__(kPersistThreads, 1) k_persistent(const Ctx c) {
  __shared__ double red[32];
  DevState* s = c.st;
  const int bid = blockIdx.x, nb = gridDim.x;
  double* x = s->x;  // host-written before the launch, constant during the solve
  auto nop = [](double) {};
  while (true) {
    if (ldv(&s->done)) break;
    const int rs = ldv(&s->r_store), ps = ldv(&s->p_store), ur = ldv(&s->ur), uz = ldv(&s->uz);
    const double omega = ldv(&s->omega);
    const bool first = (ldv(&s->k) == 0);
    double v = pz(c, rs, ur, uz, omega, bid, nb);                                                   // a2
    grid_sync_reduce<true>(v, c.partials + 0 * kMaxGrid, s, bid, nb, red, [&](double t) { epi_rho(epi_ctx(c), t); });
    pp(c, ps, uz, ldv(&s->beta), first, bid, nb);                                                   // a3
    grid_sync_reduce<false>(0.0, nullptr, s, bid, nb, red, nop);
    v = ps_(c, ur, uz, bid, nb, red);                                                        // a4
    grid_sync_reduce<true>(v, c.partials + 1 * kMaxGrid, s, bid, nb, red, [&](double t) { epi_gamma(epi_ctx(c), t); });
    if (ldv(&s->done)) break;  // breakdown
    v = pxr(c, ur, uz, ldv(&s->alpha), x, bid, nb);                                                 // a5
    grid_sync_reduce<true>(v, c.partials + 2 * kMaxGrid, s, bid, nb, red, [&](double t) { epi_delta(epi_ctx(c), t); });
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

inline bool persistent_fits(const Ctx&) { return true; }

inline int persistent_launch(const Ctx& c, int grid, cudaStream_t st) {
  Ctx cc = c;
  cc.use_cond = 0;
  void* args[] = {(void*)&cc};
  return (int)cudaLaunchCooperativeKernel((void*)k_persistent, dim3(grid), dim3(kPersistThreads), args, 0, st);
}

}  // namespace amp
