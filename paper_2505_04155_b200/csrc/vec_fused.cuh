// vec_fused.cuh — the three vector steps between two mat-vecs as ONE kernel: a5 of iteration k (x, r, delta; Alg 4.1
// lines 15-17), then a2 (z, rho; lines 4-6) and a3 (p; line 10) of iteration k + 1, with a grid barrier where Algorithm 4.1
// has a true dependency (delta before the scaling of z, rho before beta).
//
// Why.  At 2-4 M rows a vector kernel moves 13-60 MB, 2-10 us of HBM time, but costs 9-15 us: launch, ramp, reduction
// tail (ncu, profiles/r02.md: c2 k_z 13.3 us for 21 MB, k_p 8.3 us for 12.6 MB, SMs active 54 % of the elapsed time).
// Three kernels pay that three times per iteration.  Here the blocks stay resident; each of the two dependencies costs
// one arrive + poll on a counter (the replicated-scalar barrier of persistent.cuh: every block adds all partial sums in
// index order and runs the scalar step on its own copy of the loop scalars, so nothing is broadcast) instead of a kernel
// boundary.  The phases are the same device functions the stand-alone kernels call, so every vector is bit-identical;
// the sums are added over another grid, i.e. in another fixed order.
// Loop: z_0, p_0 from k_z, k_p before the loop; then per iteration k_spmv (+ k_spmv_pipe), k_vec_fused.
#pragma once
#include "kernels.cuh"
#include "persistent.cuh"

namespace amp {

#ifndef AMP_FUSED_THREADS
#define AMP_FUSED_THREADS 256
#endif
#ifndef AMP_FUSED_BLOCKS
#define AMP_FUSED_BLOCKS 2
#endif
constexpr int kFusedThreads = AMP_FUSED_THREADS;
constexpr int kFusedMinBlocks = AMP_FUSED_BLOCKS;  // 256 x 2: the x/r update needs 128 registers

// LAGGED = false: [xr | sum | z | sum | p];  LAGGED = true (AMP_SCALE_LAGGED): [xrz | sum2 | p]
template <bool LAGGED>
__global__ void __launch_bounds__(kFusedThreads, kFusedMinBlocks) k_vec_fused(const Ctx c) {
  __shared__ double red[32];
  __shared__ DevState ls;  // this block's replica of the loop scalars
  const int bid = blockIdx.x, nb = gridDim.x;
  pdl_launch_dependents();
  pdl_wait();  // alpha comes from the mat-vec's epilogue
  {
    const int* src = reinterpret_cast<const int*>(c.st);
    int* dst = reinterpret_cast<int*>(&ls);
    for (int i = threadIdx.x; i < (int)(sizeof(DevState) / sizeof(int)); i += kFusedThreads) dst[i] = __ldcg(src + i);
  }
  __syncthreads();
  DevState* s = &ls;
  EpiCtx ec = epi_ctx(c);
  ec.st = s;
  ec.use_cond = (bid == 0) ? c.use_cond : 0;  // one block speaks for the WHILE node
  if (s->done) {  // nothing to do
    if (bid == 0 && threadIdx.x == 0) set_loop_cond(ec, 0);
    return;
  }
  if (c.defer_gamma) {
    // gamma = q^T p: the mat-vec left one partial sum per block; every block adds them in index order and runs
    // epi_gamma on its replica (alpha, breakdown test) — the same numbers in the same order everywhere
    const int nbs = (c.use_pipe && s->ur == P32) ? c.spmv_grid_pipe : c.spmv_grid_direct;
    double a = 0.0;
    for (int i = threadIdx.x; i < nbs; i += kFusedThreads) a += __ldcg(c.partials + 1 * kMaxGrid + i);
    const double t = block_sum<kFusedThreads>(a, red);
    if (threadIdx.x == 0) epi_gamma(ec, t);
    __syncthreads();
    if (s->done) {  // breakdown: block 0 publishes status and stops the loop (epi_gamma has set the condition)
      if (bid == 0) {
        int* dst = reinterpret_cast<int*>(c.st);
        const int* src = reinterpret_cast<const int*>(&ls);
        const int skip0 = (int)(offsetof(DevState, fp16_subnormal) / sizeof(int));
        const int skip1 = (int)((offsetof(DevState, bar_pad) + sizeof(unsigned int)) / sizeof(int));
        for (int i = threadIdx.x; i < (int)(sizeof(DevState) / sizeof(int)); i += kFusedThreads)
          if (i < skip0 || i >= skip1) dst[i] = src[i];
      }
      return;
    }
  }
  // arrivals count up over the whole solve: this is launch number k, every earlier launch made `per` barriers
  constexpr unsigned int per = LAGGED ? 1u : 2u;
  unsigned int* arrivals = &c.st->bar_count;
  unsigned int target = (unsigned int)s->k * per * (unsigned int)nb;
  double* x = s->x;
  if constexpr (LAGGED) {
    double rr = 0.0, rz = 0.0, t0, t1;
    dispatch_xrz(c, s->ur, s->ur_n, s->uz, s->uz_n, s->alpha, s->omega_n, x, bid, nb, rr, rz);          // a5 + a2
    grid_all_sum2<kFusedThreads>(rr, rz, c.partials + 2 * kMaxGrid, arrivals, target, bid, nb, red, t0, t1);
    if (threadIdx.x == 0) epi_delta_lagged(ec, t0, t1);
    __syncthreads();
  } else {
    double v = dispatch_xr(c, s->ur, s->uz, s->alpha, x, bid, nb);                                     // a5
    double t = grid_all_sum<true, kFusedThreads>(v, c.partials + 2 * kMaxGrid, arrivals, target, bid, nb, red);
    if (threadIdx.x == 0) epi_delta(ec, t);
    __syncthreads();
    if (!s->done) {
      v = dispatch_z(c, s->r_store, s->ur, s->uz, s->omega, bid, nb);                                  // a2 of iteration k + 1
      t = grid_all_sum<true, kFusedThreads>(v, c.partials + 0 * kMaxGrid, arrivals, target, bid, nb, red);
      if (threadIdx.x == 0) epi_rho(ec, t);
      __syncthreads();
    }
  }
  if (!s->done) dispatch_p(c, s->p_store, s->uz, s->ur, s->beta, false, bid, nb);                      // a3 of iteration k + 1
  if (bid == 0) {  // publish the scalars (not the FP16 counters, accumulated in global memory, nor the barrier counter)
    __syncthreads();
    int* dst = reinterpret_cast<int*>(c.st);
    const int* src = reinterpret_cast<const int*>(&ls);
    const int skip0 = (int)(offsetof(DevState, fp16_subnormal) / sizeof(int));
    const int skip1 = (int)((offsetof(DevState, bar_pad) + sizeof(unsigned int)) / sizeof(int));
    for (int i = threadIdx.x; i < (int)(sizeof(DevState) / sizeof(int)); i += kFusedThreads)
      if (i < skip0 || i >= skip1) dst[i] = src[i];
  }
}

}  // namespace amp
