// kernels.cuh — __global__ entry points: the four loop kernels (precision dispatched at run
// time from the device state, so one static CUDA graph serves every precision phase), the
// set-up / finalisation kernels, the stand-alone SpMV and the one-off kernels of create().
#pragma once
#include "phases.cuh"
#include "shard.cuh"
#include "spmv.cuh"

#ifndef AMP_KZ_BLOCKS
#define AMP_KZ_BLOCKS 3
#endif
#ifndef AMP_KP_BLOCKS
#define AMP_KP_BLOCKS 3
#endif
#ifndef AMP_KXR_BLOCKS
#define AMP_KXR_BLOCKS 2
#endif
#ifndef AMP_VEC_BIF
#define AMP_VEC_BIF 192
#endif

namespace amp {

// ------------------------------------------------------------------ precision dispatch ------
// The precisions in use are device-side scalars (they change inside the loop without the host
// knowing), so every loop kernel branches on them once, uniformly, and runs the templated body.
template <int BIF = kVecBytesInFlight>
__device__ __forceinline__ double dispatch_z(const Ctx& c, int rs, int ur, int uz, double omega, int bid, int nb) {
  if (rs == P64 && ur == P64) {
    if (uz == P64) return phase_z<P64, P64, P64, BIF>(c, omega, bid, nb);
    if (uz == P32) return phase_z<P64, P64, P32, BIF>(c, omega, bid, nb);
    return phase_z<P64, P64, P16, BIF>(c, omega, bid, nb);
  }
  if (rs == P64 && ur == P32) {
    if (uz == P64) return phase_z<P64, P32, P64, BIF>(c, omega, bid, nb);
    if (uz == P32) return phase_z<P64, P32, P32, BIF>(c, omega, bid, nb);
    return phase_z<P64, P32, P16, BIF>(c, omega, bid, nb);
  }
  if (uz == P64) return phase_z<P32, P32, P64, BIF>(c, omega, bid, nb);
  if (uz == P32) return phase_z<P32, P32, P32, BIF>(c, omega, bid, nb);
  return phase_z<P32, P32, P16, BIF>(c, omega, bid, nb);
}

template <int BIF = kVecBytesInFlight, bool PUSH = false>
__device__ __forceinline__ void dispatch_p(const Ctx& c, int ps, int uz, int ur, double beta, bool first, int bid, int nb) {
  if (uz == P64) phase_p<P64, P64, BIF, PUSH>(c, beta, first, ur == P32, bid, nb);
  else if (uz == P32) {
    if (ps == P64) phase_p<P64, P32, BIF, PUSH>(c, beta, first, false, bid, nb);
    else phase_p<P32, P32, BIF, PUSH>(c, beta, first, false, bid, nb);
  } else {
    if (ps == P64) phase_p<P64, P16, BIF, PUSH>(c, beta, first, false, bid, nb);
    else if (ps == P32) phase_p<P32, P16, BIF, PUSH>(c, beta, first, false, bid, nb);
    else phase_p<P16, P16, BIF, PUSH>(c, beta, first, false, bid, nb);
  }
}

// zmode = 0: q = A p (step a4).  zmode = 1: q = A z, the mat-vec inside the Chebyshev-Jacobi preconditioner (the q
// buffers are free between two a4 steps); the returned sum is then not used.
template <bool COH, int NT>
__device__ __forceinline__ double dispatch_spmv(const Ctx& c, int ur, int uz, int zmode, int bid, int nb, double* red) {
  if (zmode) {
    if (ur == P64) {
      if (uz == P64) return phase_spmv<P64, COH, NT>(c, c.z64, c.z64, c.q64, bid, nb, red);
      if (uz == P32) return phase_spmv<P64, COH, NT>(c, c.z32, c.z32, c.q64, bid, nb, red);
      return phase_spmv<P64, COH, NT>(c, c.z16, c.z16, c.q64, bid, nb, red);
    }
    if (uz == P64) return phase_spmv<P32, COH, NT>(c, c.z64, c.z64, c.q32, bid, nb, red);  // RN32(z_j) per gathered entry
    if (uz == P32) return phase_spmv<P32, COH, NT>(c, c.z32, c.z32, c.q32, bid, nb, red);
    return phase_spmv<P32, COH, NT>(c, c.z16, c.z16, c.q32, bid, nb, red);
  }
  if (ur == P64) {
    if (uz == P64) return phase_spmv<P64, COH, NT>(c, c.p64, c.p64, c.q64, bid, nb, red);
    if (uz == P32) return phase_spmv<P64, COH, NT>(c, c.p32, c.p32, c.q64, bid, nb, red);
    return phase_spmv<P64, COH, NT>(c, c.p16, c.p16, c.q64, bid, nb, red);
  }
  // u_z = FP64 with u_r = FP32: the p update left RN32(p) in the FP32 copy (phase_p, shadow32): gather that
  if (uz == P64) return phase_spmv<P32, COH, NT>(c, c.p32, c.p64, c.q32, bid, nb, red);
  if (uz == P32) return phase_spmv<P32, COH, NT>(c, c.p32, c.p32, c.q32, bid, nb, red);
  return phase_spmv<P32, COH, NT>(c, c.p16, c.p16, c.q32, bid, nb, red);
}

template <int BIF = kVecBytesInFlight>
__device__ __forceinline__ double dispatch_xr(const Ctx& c, int ur, int uz, double alpha, double* x, int bid, int nb) {
  if (ur == P64) {
    if (uz == P64) return phase_xr<P64, P64, BIF>(c, alpha, x, bid, nb);
    if (uz == P32) return phase_xr<P64, P32, BIF>(c, alpha, x, bid, nb);
    return phase_xr<P64, P16, BIF>(c, alpha, x, bid, nb);
  }
  if (uz == P64) return phase_xr<P32, P64, BIF>(c, alpha, x, bid, nb);
  if (uz == P32) return phase_xr<P32, P32, BIF>(c, alpha, x, bid, nb);
  return phase_xr<P32, P16, BIF>(c, alpha, x, bid, nb);
}

// ------------------------------------------------------------------ loop kernels ------------
__global__ void __launch_bounds__(kVecThreads, AMP_KZ_BLOCKS) k_z(const Ctx c) {
  __shared__ double red[32];
  DevState* s = c.st;
  pdl_launch_dependents();
  pdl_wait();
  if (s->done) return;
  const int bid = blockIdx.x, nb = gridDim.x;
  const double v = dispatch_z(c, s->r_store, s->ur, s->uz, s->omega, bid, nb);
  // row-sharded solve (c.sh != nullptr): the partial sum goes to every rank's mailbox, k_epi runs the scalar step
  grid_reduce<kVecThreads>(v, c.partials + 0 * kMaxGrid, &s->counter[0], bid, nb, red,
                           [&](double tot) { if (c.sh != nullptr) shard_reduce_point(c, kEpiRho, tot, 0.0); else epi_rho(epi_ctx(c), tot); });
}

__global__ void __launch_bounds__(kVecThreads, AMP_KP_BLOCKS) k_p(const Ctx c) {
  const DevState* s = c.st;
  pdl_launch_dependents();
  pdl_wait();
  if (s->done) return;
  dispatch_p(c, s->p_store, s->uz, s->ur, s->beta, s->k == 0, blockIdx.x, gridDim.x);
}

// the p update of the row-sharded solve: the chunks of the send ranges also go straight into the neighbours' halo bands
// (peer stores), then the block that finishes last raises the neighbours' flags
__global__ void __launch_bounds__(kVecThreads, 2) k_p_sh(const Ctx c) {
  DevState* s = c.st;
  pdl_launch_dependents();
  pdl_wait();
  if (s->done) return;
  const int k = s->k;
  dispatch_p<kVecBytesInFlight, true>(c, s->p_store, s->uz, s->ur, s->beta, k == 0, blockIdx.x, gridDim.x);
  shard_signal_halo(c, (unsigned int)k + 1u, &s->counter[3], (int)gridDim.x);
}

template <bool COH>
__device__ __forceinline__ void spmv_kernel(const Ctx& c, int zmode, double* red) {
  DevState* s = c.st;
  pdl_launch_dependents();
  pdl_wait();
  if (s->done) return;
  if (c.use_pipe && s->ur == P32) return;  // this iteration's mat-vec is k_spmv_pipe's (next in the chain)
  const int bid = blockIdx.x, nb = gridDim.x;
  if (c.sh != nullptr) shard_wait_halo(c, (unsigned int)s->k + 1u);  // the neighbours' entries of p are in the halo bands
  const double v = dispatch_spmv<COH, kSpmvThreads>(c, s->ur, s->uz, zmode, bid, nb, red);
  if (zmode) return;  // q = A z inside M^-1: no inner product
  if (c.defer_gamma) { grid_publish<kSpmvThreads>(v, c.partials + 1 * kMaxGrid, bid, red); return; }
  grid_reduce<kSpmvThreads>(v, c.partials + 1 * kMaxGrid, &s->counter[1], bid, nb, red,
                            [&](double tot) { if (c.sh != nullptr) shard_reduce_point(c, kEpiGamma, tot, 0.0); else epi_gamma(epi_ctx(c), tot); });
}

__global__ void __launch_bounds__(kSpmvThreads, kSpmvMinBlocks) k_spmv(const Ctx c, int zmode) {
  __shared__ double red[32];
  spmv_kernel<false>(c, zmode, red);
}
// Handles attached to a shard group run the _sh twins of the three mat-vec kernels: the halo bands of p are stored by peer
// GPUs while the kernel may already be running (it waits for their flags with ld.acquire.sys), and the PTX memory model
// does not order a non-coherent load (ld.global.nc, __ldg) behind an acquire made by another thread: every gather of p
// is a plain coherent load there.  Same arithmetic, same bits.
__global__ void __launch_bounds__(kSpmvThreads, kSpmvMinBlocks) k_spmv_sh(const Ctx c, int zmode) {
  __shared__ double red[32];
  spmv_kernel<true>(c, zmode, red);
}

// step a4 for uniform-stencil matrices (phase_spmv_uni); takes k_spmv's place in the loop when the handle qualifies
template <int NT, bool COH = false>
__device__ __forceinline__ double dispatch_spmv_uni(const Ctx& c, int ur, int uz, int bid, int nb) {
  if (ur == P64) {
    if (uz == P64) return phase_spmv_uni<P64, NT, COH>(c, c.p64, c.p64, c.q64, bid, nb);
    if (uz == P32) return phase_spmv_uni<P64, NT, COH>(c, c.p32, c.p32, c.q64, bid, nb);
    return phase_spmv_uni<P64, NT, COH>(c, c.p16, c.p16, c.q64, bid, nb);
  }
  if (uz == P64) return phase_spmv_uni<P32, NT, COH>(c, c.p32, c.p64, c.q32, bid, nb);  // gathers RN32(p) (phase_p, shadow32)
  if (uz == P32) return phase_spmv_uni<P32, NT, COH>(c, c.p32, c.p32, c.q32, bid, nb);
  return phase_spmv_uni<P32, NT, COH>(c, c.p16, c.p16, c.q32, bid, nb);
}

#ifndef AMP_SPMV_UNI_BLOCKS
#define AMP_SPMV_UNI_BLOCKS AMP_SPMV_MINBLOCKS
#endif
template <bool COH>
__device__ __forceinline__ void spmv_uni_kernel(const Ctx& c, double* red) {
  DevState* s = c.st;
  pdl_launch_dependents();
  pdl_wait();
  if (s->done) return;
  if (c.use_pipe && s->ur == P32) return;  // this iteration's mat-vec is k_spmv_pipe's (next in the chain)
  const int bid = blockIdx.x, nb = gridDim.x;
  if (c.sh != nullptr) shard_wait_halo(c, (unsigned int)s->k + 1u);
  const double v = dispatch_spmv_uni<kSpmvThreads, COH>(c, s->ur, s->uz, bid, nb);
  if (c.defer_gamma) { grid_publish<kSpmvThreads>(v, c.partials + 1 * kMaxGrid, bid, red); return; }
  grid_reduce<kSpmvThreads>(v, c.partials + 1 * kMaxGrid, &s->counter[1], bid, nb, red,
                            [&](double tot) { if (c.sh != nullptr) shard_reduce_point(c, kEpiGamma, tot, 0.0); else epi_gamma(epi_ctx(c), tot); });
}

__global__ void __launch_bounds__(kSpmvThreads, AMP_SPMV_UNI_BLOCKS) k_spmv_uni(const Ctx c) {
  __shared__ double red[32];
  spmv_uni_kernel<false>(c, red);
}
__global__ void __launch_bounds__(kSpmvThreads, AMP_SPMV_UNI_BLOCKS) k_spmv_uni_sh(const Ctx c) {  // see k_spmv_sh
  __shared__ double red[32];
  spmv_uni_kernel<true>(c, red);
}

__global__ void __launch_bounds__(kVecThreads, AMP_KXR_BLOCKS) k_xr(const Ctx c) {
  __shared__ double red[32];
  DevState* s = c.st;
  pdl_launch_dependents();
  pdl_wait();
  if (s->done) {  // nothing to do (converged at set-up, or breakdown): make sure the WHILE node stops
    if (blockIdx.x == 0 && threadIdx.x == 0) set_loop_cond(epi_ctx(c), 0);
    return;
  }
  const int bid = blockIdx.x, nb = gridDim.x;
  const double v = dispatch_xr(c, s->ur, s->uz, s->alpha, s->x, bid, nb);
  grid_reduce<kVecThreads>(v, c.partials + 2 * kMaxGrid, &s->counter[2], bid, nb, red,
                           [&](double tot) { if (c.sh != nullptr) shard_reduce_point(c, kEpiDelta, tot, 0.0); else epi_delta(epi_ctx(c), tot); });
}

// ------------------------------------------------------------------ Chebyshev-Jacobi kernels --
template <int BIF = kVecBytesInFlight>
__device__ __forceinline__ double dispatch_cheb0(const Ctx& c, int rs, int ur, int uz, double omega, bool with_rho, int bid, int nb) {
  if (rs == P64 && ur == P64) {
    if (uz == P64) return phase_cheb0<P64, P64, P64, BIF>(c, omega, with_rho, bid, nb);
    if (uz == P32) return phase_cheb0<P64, P64, P32, BIF>(c, omega, with_rho, bid, nb);
    return phase_cheb0<P64, P64, P16, BIF>(c, omega, with_rho, bid, nb);
  }
  if (rs == P64 && ur == P32) {
    if (uz == P64) return phase_cheb0<P64, P32, P64, BIF>(c, omega, with_rho, bid, nb);
    if (uz == P32) return phase_cheb0<P64, P32, P32, BIF>(c, omega, with_rho, bid, nb);
    return phase_cheb0<P64, P32, P16, BIF>(c, omega, with_rho, bid, nb);
  }
  if (uz == P64) return phase_cheb0<P32, P32, P64, BIF>(c, omega, with_rho, bid, nb);
  if (uz == P32) return phase_cheb0<P32, P32, P32, BIF>(c, omega, with_rho, bid, nb);
  return phase_cheb0<P32, P32, P16, BIF>(c, omega, with_rho, bid, nb);
}

template <int BIF = kVecBytesInFlight>
__device__ __forceinline__ double dispatch_cheb_step(const Ctx& c, int ur, int uz, double omega, double c1, double c2, bool with_rho,
                                                     int bid, int nb) {
  if (ur == P64) {
    if (uz == P64) return phase_cheb_step<P64, P64, BIF>(c, omega, c1, c2, with_rho, bid, nb);
    if (uz == P32) return phase_cheb_step<P64, P32, BIF>(c, omega, c1, c2, with_rho, bid, nb);
    return phase_cheb_step<P64, P16, BIF>(c, omega, c1, c2, with_rho, bid, nb);
  }
  if (uz == P64) return phase_cheb_step<P32, P64, BIF>(c, omega, c1, c2, with_rho, bid, nb);
  if (uz == P32) return phase_cheb_step<P32, P32, BIF>(c, omega, c1, c2, with_rho, bid, nb);
  return phase_cheb_step<P32, P16, BIF>(c, omega, c1, c2, with_rho, bid, nb);
}

// first sweep of M^-1 (takes k_z's place in the loop); the reduction and epi_rho only when it is also the last sweep
__global__ void __launch_bounds__(kVecThreads, 2) k_cheb0(const Ctx c) {
  __shared__ double red[32];
  DevState* s = c.st;
  pdl_launch_dependents();
  pdl_wait();
  if (s->done) return;
  const int bid = blockIdx.x, nb = gridDim.x;
  const bool last = c.cheb_s == 1;
  const double v = dispatch_cheb0(c, s->r_store, s->ur, s->uz, s->omega, last, bid, nb);
  if (last)
    grid_reduce<kVecThreads>(v, c.partials + 0 * kMaxGrid, &s->counter[0], bid, nb, red,
                             [&](double tot) { epi_rho(epi_ctx(c), tot); });
}

// sweep i (1 <= i < s) of M^-1, after the mat-vec w = A z (k_spmv in mode 1)
__global__ void __launch_bounds__(kVecThreads, 2) k_cheb_step(const Ctx c, int i) {
  __shared__ double red[32];
  DevState* s = c.st;
  pdl_launch_dependents();
  pdl_wait();
  if (s->done) return;
  const int bid = blockIdx.x, nb = gridDim.x;
  const bool last = i == c.cheb_s - 1;
  const double v = dispatch_cheb_step(c, s->ur, s->uz, s->omega, c.cheb_c1[i], c.cheb_c2[i], last, bid, nb);
  if (last)
    grid_reduce<kVecThreads>(v, c.partials + 0 * kMaxGrid, &s->counter[0], bid, nb, red,
                             [&](double tot) { epi_rho(epi_ctx(c), tot); });
}

// ------------------------------------------------------------------ lagged variant: k_xrz ----
template <int UR, int URN, int BIF>
__device__ __forceinline__ void dispatch_xrz_z(const Ctx& c, int uz, int uzn, double alpha, double omega_n, double* x, int bid,
                                               int nb, double& rr, double& rz) {
  if (uz == P64) {
    if (uzn == P64) phase_xrz<UR, URN, P64, P64, BIF>(c, alpha, omega_n, x, bid, nb, rr, rz);
    else if (uzn == P32) phase_xrz<UR, URN, P64, P32, BIF>(c, alpha, omega_n, x, bid, nb, rr, rz);
    else phase_xrz<UR, URN, P64, P16, BIF>(c, alpha, omega_n, x, bid, nb, rr, rz);
  } else if (uz == P32) {
    if (uzn == P32) phase_xrz<UR, URN, P32, P32, BIF>(c, alpha, omega_n, x, bid, nb, rr, rz);
    else phase_xrz<UR, URN, P32, P16, BIF>(c, alpha, omega_n, x, bid, nb, rr, rz);
  } else {
    phase_xrz<UR, URN, P16, P16, BIF>(c, alpha, omega_n, x, bid, nb, rr, rz);
  }
}
template <int BIF = kVecBytesInFlight>
__device__ __forceinline__ void dispatch_xrz(const Ctx& c, int ur, int urn, int uz, int uzn, double alpha, double omega_n,
                                             double* x, int bid, int nb, double& rr, double& rz) {
  if (ur == P64 && urn == P64) dispatch_xrz_z<P64, P64, BIF>(c, uz, uzn, alpha, omega_n, x, bid, nb, rr, rz);
  else if (ur == P64) dispatch_xrz_z<P64, P32, BIF>(c, uz, uzn, alpha, omega_n, x, bid, nb, rr, rz);
  else dispatch_xrz_z<P32, P32, BIF>(c, uz, uzn, alpha, omega_n, x, bid, nb, rr, rz);
}

// a5 of iteration k fused with a2 of iteration k+1 (AMP_SCALE_LAGGED): x, r, delta, z, rho in one pass
__global__ void __launch_bounds__(kVecThreads, 2) k_xrz(const Ctx c) {
  __shared__ double red[32];
  DevState* s = c.st;
  pdl_launch_dependents();
  pdl_wait();
  if (s->done) {
    if (blockIdx.x == 0 && threadIdx.x == 0) set_loop_cond(epi_ctx(c), 0);
    return;
  }
  const int bid = blockIdx.x, nb = gridDim.x;
  double rr = 0.0, rz = 0.0;
  dispatch_xrz(c, s->ur, s->ur_n, s->uz, s->uz_n, s->alpha, s->omega_n, s->x, bid, nb, rr, rz);
  grid_reduce2<kVecThreads>(rr, rz, c.partials + 2 * kMaxGrid, &s->counter[2], bid, nb, red, [&](double t0, double t1) {
    if (c.sh != nullptr) shard_reduce_point(c, kEpiDeltaLagged, t0, t1); else epi_delta_lagged(epi_ctx(c), t0, t1);
  });
}

// ------------------------------------------------------------------ stand-alone SpMV --------
// halo_seq != 0 (row-sharded solve): wait for the neighbours' halo push with that sequence number first
// COH = true whenever a halo is waited for: the gathers are then plain coherent loads (see k_spmv_sh)
template <int UR, class PT, bool COH = false>
__global__ void __launch_bounds__(kSpmvThreads, kSpmvMinBlocks) k_spmv_any(const Ctx c, const PT* p, typename Store<UR>::T* q,
                                                                           unsigned int halo_seq) {
  __shared__ double red[32];
  if (halo_seq != 0u && c.sh != nullptr) shard_wait_halo(c, halo_seq);
  (void)phase_spmv<UR, COH, kSpmvThreads>(c, p, p, q, blockIdx.x, gridDim.x, red);
}

// ------------------------------------------------------------------ set-up / finalise -------
// step a0 (Alg 4.1 line 1): r0 = b - A x0 in FP64 (q64 holds A x0; for x0 = 0: r0 = b, x = 0),
// ||b||, delta_0 = ||r0||, then the selector for k = 0.
__global__ void __launch_bounds__(kVecThreads) k_setup(const Ctx c, int x0_zero) {
  __shared__ double red[32];
  __shared__ int s_last;
  DevState* s = c.st;
  const double* __restrict__ b = s->b;
  double* __restrict__ x = s->x;
  double bb = 0.0, rr = 0.0;
  const int64_t stride = (int64_t)gridDim.x * kVecThreads;
  for (int64_t i = (int64_t)blockIdx.x * kVecThreads + threadIdx.x; i < c.n; i += stride) {
    const double bi = b[i];
    double ri;
    if (x0_zero) { ri = bi; x[i] = 0.0; }
    else ri = bi - c.q64[i];
    c.r64[i] = ri;
    bb = fma(bi, bi, bb);
    rr = fma(ri, ri, rr);
  }
  const double b1 = block_sum<kVecThreads>(bb, red);
  const double b2 = block_sum<kVecThreads>(rr, red);
  double* part = c.partials + 3 * kMaxGrid;
  if (threadIdx.x == 0) {
    __stcg(part + 2 * blockIdx.x, b1);
    __stcg(part + 2 * blockIdx.x + 1, b2);
    __threadfence();
    s_last = (atomicAdd(&s->counter[3], 1u) == gridDim.x - 1);
  }
  __syncthreads();
  if (s_last) {
    __threadfence();
    double s1 = 0.0, s2 = 0.0;
    for (int i = threadIdx.x; i < (int)gridDim.x; i += kVecThreads) {
      s1 += __ldcg(part + 2 * i);
      s2 += __ldcg(part + 2 * i + 1);
    }
    const double t1 = block_sum<kVecThreads>(s1, red);
    const double t2 = block_sum<kVecThreads>(s2, red);
    if (threadIdx.x == 0) {
      s->counter[3] = 0u;
      if (c.sh != nullptr) shard_reduce_point(c, kEpiSetup, t1, t2); else epi_setup(epi_ctx(c), t1, t2);
    }
  }
}

// after the loop: x = 0 if b = 0; optional true residual ||b - A x|| / ||b|| (q64 holds A x)
__global__ void __launch_bounds__(kVecThreads) k_finalize(const Ctx c, int true_residual) {
  __shared__ double red[32];
  DevState* s = c.st;
  const int64_t stride = (int64_t)gridDim.x * kVecThreads;
  if (s->zero_x) {
    for (int64_t i = (int64_t)blockIdx.x * kVecThreads + threadIdx.x; i < c.n; i += stride) s->x[i] = 0.0;
  }
  if (!true_residual) return;
  double rr = 0.0;
  if (!s->zero_x) {
    for (int64_t i = (int64_t)blockIdx.x * kVecThreads + threadIdx.x; i < c.n; i += stride) {
      const double t = s->b[i] - c.q64[i];
      rr = fma(t, t, rr);
    }
  }
  if (c.sh != nullptr && s->zero_x) {  // b = 0 on every rank: no reduction
    if (blockIdx.x == 0 && threadIdx.x == 0) s->relres_true = 0.0;
    return;
  }
  grid_reduce<kVecThreads>(rr, c.partials + 3 * kMaxGrid, &s->counter[3], blockIdx.x, gridDim.x, red, [&](double tot) {
    if (c.sh != nullptr) shard_reduce_point(c, kEpiFinal, tot, 0.0);
    else s->relres_true = (s->bnorm > 0.0) ? sqrt(tot) / s->bnorm : 0.0;
  });
}

// ------------------------------------------------------------------ create() kernels --------
// flags: bit0 rowptr not monotone / out of range, bit1 column out of range,
//        bit2 missing diagonal, bit3 non-positive or non-finite diagonal
// ncols / shift: a block row of a sharded system has n + halo_lo + halo_hi columns and its diagonal at column i + halo_lo
__global__ void k_validate_dinv(int64_t n, int64_t nnz, int64_t ncols, int64_t shift, const int32_t* rowptr, const int32_t* colidx,
                                const double* vals, int jacobi, double* dinv64, float* dinv32, int* flags) {
  const int64_t stride = (int64_t)gridDim.x * blockDim.x;
  int f = 0;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) {
    const int64_t a = rowptr[i], b = rowptr[i + 1];
    if (i == 0 && a != 0) f |= 1;
    if (i == n - 1 && b != nnz) f |= 1;
    if (a < 0 || b < a || b > nnz) { f |= 1; continue; }
    double d = jacobi ? 0.0 : 1.0;
    bool found = !jacobi;
    for (int64_t e = a; e < b; ++e) {
      const int j = colidx[e];
      if (j < 0 || j >= ncols) { f |= 2; continue; }
      if (jacobi && j == i + shift) { d += vals[e]; found = true; }  // duplicates add up, as in the mat-vec
    }
    if (!found) { f |= 4; d = 1.0; }
    else if (!(d > 0.0) || isinf(d)) { f |= 8; d = 1.0; }
    dinv64[i] = 1.0 / d;
    dinv32[i] = __double2float_rn(1.0 / d);
  }
  if (f) atomicOr(flags, f);
}

// max |a_i| of an int32 array (the largest diagonal offset of the aligned slices: size of p's guard band)
__global__ void k_absmax_i32(int64_t n, const int32_t* __restrict__ a, int* __restrict__ out) {
  const int64_t stride = (int64_t)gridDim.x * blockDim.x;
  int m = 0;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) m = max(m, abs(a[i]));
  m = max(m, __shfl_xor_sync(0xffffffffu, m, 16)); m = max(m, __shfl_xor_sync(0xffffffffu, m, 8));
  m = max(m, __shfl_xor_sync(0xffffffffu, m, 4)); m = max(m, __shfl_xor_sync(0xffffffffu, m, 2));
  m = max(m, __shfl_xor_sync(0xffffffffu, m, 1));
  if ((threadIdx.x & 31) == 0 && m > 0) atomicMax(out, m);
}

// max_i (sum_j |a_ij|) / a_ii: Gershgorin bound of the spectrum of D^-1 A (row sums in CSR order, duplicates of the
// diagonal add up); the maximum of positive doubles is the maximum of their bit patterns
__global__ void k_gershgorin(int64_t n, const int32_t* __restrict__ rowptr, const int32_t* __restrict__ colidx,
                             const double* __restrict__ vals, unsigned long long* __restrict__ out) {
  const int64_t stride = (int64_t)gridDim.x * blockDim.x;
  double m = 0.0;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) {
    double d = 0.0, srow = 0.0;
    for (int32_t e = rowptr[i]; e < rowptr[i + 1]; ++e) {
      srow = __dadd_rn(srow, fabs(vals[e]));
      if (colidx[e] == i) d = __dadd_rn(d, vals[e]);
    }
    const double g = __ddiv_rn(srow, d);
    if (g > m) m = g;
  }
  if (m > 0.0) atomicMax(out, (unsigned long long)__double_as_longlong(m));
}

__global__ void k_to_fp32(int64_t n, const double* __restrict__ a, float* __restrict__ o) {
  const int64_t stride = (int64_t)gridDim.x * blockDim.x;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) o[i] = __double2float_rn(a[i]);
}

}  // namespace amp
