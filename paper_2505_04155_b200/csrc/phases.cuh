// phases.cuh — the steps of one AMP-PCG iteration (Algorithm 4.1) as device
// functions over a (block id, block count) work decomposition, so that the same code runs as
// four stand-alone kernels (stream / CUDA-graph loop) or inside the persistent kernel.
//
//   phase_z    a2: y = omega r, z = M^-1 y (fused), one rounding to u_z; rho = r^T z
//   phase_p    a3: p = z + beta p, one rounding to u_z
//   phase_spmv a4: q = A p in u_r, gamma = q^T p  (spmv.cuh)
//   phase_xr   a5: x += alpha p (FP64), r -= alpha q (u_r), delta = ||r||
// and the scalar epilogues (one thread, after each grid reduction):
//   epi_rho    beta = rho_k / rho_{k-1}                       (Alg 4.1 lines 6-9)
//   epi_gamma  alpha = rho / gamma, breakdown test             (lines 13-14)
//   epi_delta  stop test, eta_k and the selector (4.1) for the next iteration (lines 3, 17-20)
#pragma once
#include <math_constants.h>

#include "common.cuh"

namespace amp {

// ------------------------------------------------------------------ scalar epilogues --------
// what the scalar epilogues need from the kernel context (passed by value: the out-of-line
// epilogues must not force a stack copy of the whole Ctx)
struct EpiCtx {
  DevState* st;
  int64_t n;   // rows of the whole system (RMS scale)
  cudaGraphConditionalHandle cond;
  int32_t use_cond;
};
__device__ __forceinline__ EpiCtx epi_ctx(const Ctx& c) { return EpiCtx{c.st, c.n_scale, c.cond, c.use_cond}; }
__device__ __forceinline__ void set_loop_cond(const EpiCtx c, int keep_going) {
  if (c.use_cond) cudaGraphSetConditional(c.cond, keep_going ? 1u : 0u);
}

__device__ __forceinline__ int lower_prec(int a, int b) { return a > b ? a : b; }

// eta_k (4.9)/(4.11) and (u_z,k, u_r,k) = precisionSelector (4.1) for iteration k = s->k, then
// omega_k.  Readings R2 (norms with negative index are ||r_0||), R3 (eta vs tol*||b||, <=) and
// R5 (both switches latched) of DESIGN.md.  hist[t] = ||r_t||.
__device__ __noinline__ void select_precisions(DevState* s, int64_t n) {
  const int k = s->k;
  const double delta = s->delta;
  if (!s->amp) {
    s->omega = 1.0;
    return;
  }
  const double* hist = s->hist;
  if (s->ur == P64 && s->eta_rule != 2) {
    double eta = CUDART_INF;
    const double C = s->C, e32 = s->eps32;
    if (s->eta_rule == 0) {  // (4.9)
      eta = 0.0;
      for (int t = k - s->d; t <= k; ++t) {
        const double hm1 = hist[(t - 1) > 0 ? (t - 1) : 0], h0 = hist[t > 0 ? t : 0];
        eta += e32 * ((3.0 + C) * hm1 + (2.0 + C) * h0);
      }
    } else {  // (4.11)
      const int l = s->ell;
      if (k >= l && hist[k] < hist[k - l]) {
        const double rate = pow(hist[k] / hist[k - l], 1.0 / (double)l);
        eta = e32 * (5.0 + 2.0 * C) * hist[k - 1] / (1.0 - rate);
      }
    }
    if (eta <= s->eta_safety * s->tol * s->bnorm) {  // (4.10)
      s->ur = P32;
      s->it_ur32 = k;
    }
  }
  const double nu = delta / s->bnorm;  // nu_k
  int want = s->u0;
  if (nu < s->tau_zs) want = lower_prec(s->u0, nu >= s->tau_zh ? P32 : P16);
  if (want > s->uz) {
    s->uz = want;
    if (want >= P32 && s->it_uz32 < 0) s->it_uz32 = k;
    if (want == P16 && s->it_uz16 < 0) s->it_uz16 = k;
  }
  double om = 1.0;  // omega_k: Alg 4.1 line 4, or the alternatives allowed by PAPER.md:34, :223
  if (s->scale_mode == 0) om = 1.0 / delta;
  else if (s->scale_mode == 1) om = sqrt((double)n) / delta;
  else if (s->scale_mode == 2) om = ldexp(1.0, (int)rint(log2(1.0 / delta)));
  s->omega = om;
}

__device__ void decide_next(DevState* s, int t);
__device__ __forceinline__ void apply_next(DevState* s);

// after the setup reduction: ||b||, delta_0 = ||r_0||, edge cases, selector for k = 0
__device__ __noinline__ void epi_setup(const EpiCtx c, double bb, double rr) {
  DevState* s = c.st;
  s->bnorm = sqrt(bb);
  s->delta = sqrt(rr);
  s->hist[0] = s->delta;
  s->k = 0;
  s->r_store = P64;
  s->ur = P64;
  s->uz = s->amp ? s->u0 : P64;
  s->p_store = s->uz;
  s->rho_prev = 0.0;
  s->beta = 0.0;
  if (bb == 0.0) {  // b = 0: x = 0 (reading R13)
    s->done = 1; s->status = 0; s->zero_x = 1; s->delta = 0.0;
  } else if (!(s->delta == s->delta) || isinf(s->delta) || isinf(s->bnorm)) {
    s->done = 1; s->status = -2;
  } else if (s->delta <= s->stop_safety * s->tol * s->bnorm && !s->no_stop) {
    s->done = 1; s->status = 0;  // x0 already satisfies the stopping test
  } else if (s->amp && s->scale_mode == 4) {  // lagged: D(0) = D(1) = the decisions from ||r_0||
    decide_next(s, 0);
    apply_next(s);
    s->p_store = s->uz;
  } else {
    select_precisions(s, c.n);
  }
}

__device__ __forceinline__ void epi_rho(const EpiCtx c, double rho) {
  DevState* s = c.st;
  s->rho = rho;
  s->beta = (s->k > 0) ? rho / s->rho_prev : 0.0;  // Alg 4.1 lines 7-9
}

__device__ __forceinline__ void epi_gamma(const EpiCtx c, double gamma) {
  DevState* s = c.st;
  s->gamma = gamma;
  const double rho = s->rho;
  if (!(gamma > 0.0) || !(rho > 0.0) || isinf(gamma) || isinf(rho)) {  // breakdown (reading R13)
    s->status = -2;
    s->done = 1;
    set_loop_cond(c, 0);
  } else {
    s->alpha = rho / gamma;  // line 14
  }
}

__device__ __noinline__ void epi_delta(const EpiCtx c, double rr) {
  DevState* s = c.st;
  const double delta = sqrt(rr);  // line 17
  const int k1 = s->k + 1;
  s->delta = delta;
  s->hist[k1] = delta;
  s->rho_prev = s->rho;
  s->k = k1;
  s->r_store = s->ur;
  s->p_store = s->uz;
  if (!(delta == delta) || isinf(delta)) {
    s->status = -2; s->done = 1;
  } else if (delta <= s->stop_safety * s->tol * s->bnorm && !s->no_stop) {  // line 18
    s->status = 0; s->done = 1;
  } else if (k1 >= s->maxit) {
    s->status = 1; s->done = 1;
  } else {
    select_precisions(s, c.n);  // line 3 of the next iteration
  }
  set_loop_cond(c, !s->done);
}

// ------------------------------------------------------------------ lagged variant ----------
// AMP_SCALE_LAGGED (reading R17): lines 3 and 4 of Alg 4.1 for iteration k are evaluated with
// ||r_{k-1}|| instead of ||r_k|| (other scaling factors are allowed: Thm 3.2).  The decisions
// D(k) = (u_r, u_z, omega) of iteration k are then known one iteration early, so z_{k+1} and rho_{k+1} can be
// produced in the same pass that updates x and r (k_xrz): three kernels and three grid-wide reductions per iteration
// instead of four, and r is not read again.
// decide D(t+1) from hist[0..t] into (ur_n, uz_n, omega_n)
__device__ __noinline__ void decide_next(DevState* s, int t) {
  const double* hist = s->hist;
  int ur_n = s->ur;
  if (ur_n == P64 && s->eta_rule != 2) {
    double eta = CUDART_INF;
    const double C = s->C, e32 = s->eps32;
    if (s->eta_rule == 0) {  // (4.9)
      eta = 0.0;
      for (int u = t - s->d; u <= t; ++u) {
        const double hm1 = hist[(u - 1) > 0 ? (u - 1) : 0], h0 = hist[u > 0 ? u : 0];
        eta += e32 * ((3.0 + C) * hm1 + (2.0 + C) * h0);
      }
    } else {  // (4.11)
      const int l = s->ell;
      if (t >= l && hist[t] < hist[t - l]) {
        const double rate = pow(hist[t] / hist[t - l], 1.0 / (double)l);
        eta = e32 * (5.0 + 2.0 * C) * hist[t - 1] / (1.0 - rate);
      }
    }
    if (eta <= s->eta_safety * s->tol * s->bnorm) ur_n = P32;  // (4.10)
  }
  const double nu = hist[t] / s->bnorm;
  int want = s->u0;
  if (nu < s->tau_zs) want = lower_prec(s->u0, nu >= s->tau_zh ? P32 : P16);
  s->ur_n = ur_n;
  s->uz_n = want > s->uz ? want : s->uz;
  s->omega_n = 1.0 / hist[t];
}

// make D(k) current (k = s->k) and record the switch iterations
__device__ __forceinline__ void apply_next(DevState* s) {
  const int k = s->k;
  if (s->ur_n != s->ur) { s->ur = s->ur_n; s->it_ur32 = k; }
  if (s->uz_n > s->uz) {
    s->uz = s->uz_n;
    if (s->uz >= P32 && s->it_uz32 < 0) s->it_uz32 = k;
    if (s->uz == P16 && s->it_uz16 < 0) s->it_uz16 = k;
  }
  s->omega = s->omega_n;
}

// after k_xrz of iteration k: rr = ||r_{k+1}||^2, rz = r_{k+1}^T z_{k+1}
__device__ __noinline__ void epi_delta_lagged(const EpiCtx c, double rr, double rz) {
  DevState* s = c.st;
  const double delta = sqrt(rr);
  const int k1 = s->k + 1;
  s->delta = delta;
  s->hist[k1] = delta;
  s->rho_prev = s->rho;
  s->rho = rz;
  s->beta = rz / s->rho_prev;
  s->k = k1;
  s->p_store = s->uz;   // p_k is stored in u_z,k
  apply_next(s);        // D(k+1) becomes current; r_{k+1} and z_{k+1} were stored in it
  s->r_store = s->ur;
  if (!(delta == delta) || isinf(delta)) {
    s->status = -2; s->done = 1;
  } else if (delta <= s->stop_safety * s->tol * s->bnorm && !s->no_stop) {
    s->status = 0; s->done = 1;
  } else if (k1 >= s->maxit) {
    s->status = 1; s->done = 1;
  } else {
    decide_next(s, k1);  // D(k+2)
  }
  set_loop_cond(c, !s->done);
}

#ifdef AMP_COUNT_FP16
// counting build: classify every FP16 store of z and p (exact value v, stored value h)
__device__ __forceinline__ void count_fp16(DevState* s, double v, double h) {
  if (v == 0.0) return;
  if (isinf(h) && !isinf(v)) atomicAdd(&s->fp16_inf, 1ull);
  else if (h == 0.0) atomicAdd(&s->fp16_flushed, 1ull);
  else if (fabs(h) < 6.103515625e-05) atomicAdd(&s->fp16_subnormal, 1ull);
}
#endif

// NOTE: the loop vectors (r, z, p, q, x) are deliberately NOT __restrict__/read-only qualified:
// inside the persistent kernel they are written by earlier phases of the same kernel, so they
// must be read with plain coherent loads (ordered by the grid barrier), never ld.global.nc.
// Every thread owns chunks of E consecutive elements (common.cuh: chunk_*), U chunks per trip:
// all loads of a trip are issued before the first use, so a thread keeps about
// kVecBytesInFlight bytes in flight whatever the precisions are.

// ------------------------------------------------------------------ a2: z and rho ------------
// RS: precision r is stored in; UR: precision selected for r (RS != UR only at the iteration of
// the u_r switch, where r <- RN32(r) is fused here, step a6); UZ: precision of z.
// Every vector step below comes as (1) a traits struct with its storage types and chunk size E, (2) a chunk body: the
// arithmetic of ONE chunk of E consecutive elements from raw loaded chunks, shared by (3) the direct driver (every
// thread loads its chunks from global memory, U chunks in flight) and the staged drivers of vec_pipe.cuh (the input
// streams arrive in shared memory through bulk copies).
template <int RS, int UR, int UZ> struct ZT {
  using TR = typename Store<RS>::T;
  using TO = typename Store<UR>::T;
  using TZ = typename Store<UZ>::T;
  using TD = typename Store<(UZ == P64) ? P64 : P32>::T;
  static constexpr int smin = cmin(cmin((int)sizeof(TR), (int)sizeof(TO)), cmin((int)sizeof(TD), (int)sizeof(TZ)));
  static constexpr int smax = cmax(cmax((int)sizeof(TR), (int)sizeof(TO)), cmax((int)sizeof(TD), (int)sizeof(TZ)));
  static constexpr int E = chunk_elems(smin, smax);
  static __device__ __forceinline__ const TD* dinv(const Ctx& c) {
    if constexpr (UZ == P64) return c.dinv64; else return c.dinv32;
  }
};
// z = RN_{u_z}((r omega) dinv) for chunk i; sum += r^T z with the STORED z (Alg 4.1 lines 4-6)
template <int RS, int UR, int UZ>
__device__ __forceinline__ void z_chunk(const Ctx& c, const double omega, const Chunk<typename ZT<RS, UR, UZ>::TR, ZT<RS, UR, UZ>::E>& rr,
                                        const Chunk<typename ZT<RS, UR, UZ>::TD, ZT<RS, UR, UZ>::E>& dd, const int64_t i, double& sum) {
  using T = ZT<RS, UR, UZ>;
  constexpr int E = T::E;
  double a[E], d[E], zz[E];
  chunk_unpack(rr, a);
  chunk_unpack(dd, d);
  if constexpr (RS != UR) {  // r <- RN_{u_r}(r) at the switch iteration
    Chunk<typename T::TO, E> ro;
    chunk_pack(ro, a);
    chunk_store(ro, rvec<UR>(c), i);
    chunk_unpack(ro, a);
  }
#pragma unroll
  for (int e = 0; e < E; ++e) zz[e] = (a[e] * omega) * d[e];
  Chunk<typename T::TZ, E> zo;
  chunk_pack(zo, zz);  // the one rounding to u_z (reading R6)
  chunk_store(zo, zvec<UZ>(c), i);
#ifdef AMP_COUNT_FP16
  double zx[E];
#pragma unroll
  for (int e = 0; e < E; ++e) zx[e] = zz[e];
#endif
  chunk_unpack(zo, zz);
#ifdef AMP_COUNT_FP16
  if (UZ == P16) {
#pragma unroll
    for (int e = 0; e < E; ++e) count_fp16(c.st, zx[e], zz[e]);
  }
#endif
#pragma unroll
  for (int e = 0; e < E; ++e) sum = fma(a[e], zz[e], sum);  // rho uses the stored z
}

template <int RS, int UR, int UZ, int BIF = kVecBytesInFlight>
__device__ __forceinline__ double phase_z(const Ctx& c, const double omega, int bid, int nb) {
  using T = ZT<RS, UR, UZ>;
  using TR = typename T::TR;
  using TD = typename T::TD;
  constexpr int E = T::E;
  constexpr int U = cmax(1, BIF / (E * (int)(sizeof(TR) + sizeof(TD))));
  const TR* rin = rvec<RS>(c);
  const TD* dinv = T::dinv(c);
  const int64_t nchunk = c.npad / E;
  const int64_t stride = (int64_t)nb * blockDim.x;
  double sum = 0.0;
  for (int64_t base = (int64_t)bid * blockDim.x + threadIdx.x; base < nchunk; base += stride * U) {
    Chunk<TR, E> rr[U];
    Chunk<TD, E> dd[U];
#pragma unroll
    for (int u = 0; u < U; ++u) {
      const int64_t i = base + u * stride;
      if (i < nchunk) { chunk_load(rr[u], rin, i); chunk_load(dd[u], dinv, i); }
    }
#pragma unroll
    for (int u = 0; u < U; ++u) {
      const int64_t i = base + u * stride;
      if (i < nchunk) z_chunk<RS, UR, UZ>(c, omega, rr[u], dd[u], i, sum);
    }
  }
  return sum;
}

// ------------------------------------------------------------------ a2 with Chebyshev-Jacobi --
// M^-1 = s sweeps of Chebyshev-accelerated Jacobi (the paper's smoother; reading R18).
// Explicit __dmul_rn / __dsub_rn / __dadd_rn / __fma_rn: the operation order IS the definition (the oracle's
// orc_cheb_first / orc_cheb_step do the same operations), so nothing may be contracted into an fma.
// first sweep: d = z = RN_{u_z}( ((r omega) dinv) / theta ); WITH_RHO (s = 1): rho = r^T z.  RS/UR/UZ as in phase_z.
template <int RS, int UR, int UZ, int BIF = kVecBytesInFlight>
__device__ __forceinline__ double phase_cheb0(const Ctx& c, const double omega, const bool with_rho, int bid, int nb) {
  using TR = typename Store<RS>::T;
  using TO = typename Store<UR>::T;
  using TZ = typename Store<UZ>::T;
  using TD = typename Store<(UZ == P64) ? P64 : P32>::T;
  constexpr int smin = cmin(cmin((int)sizeof(TR), (int)sizeof(TO)), cmin((int)sizeof(TD), (int)sizeof(TZ)));
  constexpr int smax = cmax(cmax((int)sizeof(TR), (int)sizeof(TO)), cmax((int)sizeof(TD), (int)sizeof(TZ)));
  constexpr int E = chunk_elems(smin, smax);
  constexpr int U = cmax(1, BIF / (E * (int)(sizeof(TR) + sizeof(TD))));
  const TR* rin = rvec<RS>(c);
  TO* rout = rvec<UR>(c);
  TZ* z = zvec<UZ>(c);
  TZ* dd_out = dvec<UZ>(c);
  const TD* dinv;
  if constexpr (UZ == P64) dinv = c.dinv64; else dinv = c.dinv32;
  const double inv_theta = c.cheb_inv_theta;
  const int64_t nchunk = c.npad / E;
  const int64_t stride = (int64_t)nb * blockDim.x;
  double sum = 0.0;
  for (int64_t base = (int64_t)bid * blockDim.x + threadIdx.x; base < nchunk; base += stride * U) {
    Chunk<TR, E> rr[U];
    Chunk<TD, E> dd[U];
#pragma unroll
    for (int u = 0; u < U; ++u) {
      const int64_t i = base + u * stride;
      if (i < nchunk) { chunk_load(rr[u], rin, i); chunk_load(dd[u], dinv, i); }
    }
#pragma unroll
    for (int u = 0; u < U; ++u) {
      const int64_t i = base + u * stride;
      if (i < nchunk) {
        double a[E], d[E], zz[E];
        chunk_unpack(rr[u], a);
        chunk_unpack(dd[u], d);
        if constexpr (RS != UR) {  // r <- RN_{u_r}(r) at the switch iteration (step a6)
          Chunk<TO, E> ro;
          chunk_pack(ro, a);
          chunk_store(ro, rout, i);
          chunk_unpack(ro, a);
        }
#pragma unroll
        for (int e = 0; e < E; ++e) zz[e] = __dmul_rn(__dmul_rn(__dmul_rn(a[e], omega), d[e]), inv_theta);
        Chunk<TZ, E> zo;
        chunk_pack(zo, zz);  // one rounding to u_z
        chunk_store(zo, z, i);
        chunk_store(zo, dd_out, i);
        if (with_rho) {
          chunk_unpack(zo, zz);
#pragma unroll
          for (int e = 0; e < E; ++e) sum = fma(a[e], zz[e], sum);
        }
      }
    }
  }
  return sum;
}

// sweep i >= 1, w = A z in u_r (the q buffers): t = r omega - w; u = t dinv; d = RN_{u_z}(fma(c1, d, c2 u));
// z = RN_{u_z}(z + d); with_rho (last sweep): rho = r^T z with the stored z
template <int UR, int UZ, int BIF = kVecBytesInFlight>
__device__ __forceinline__ double phase_cheb_step(const Ctx& c, const double omega, const double c1, const double c2,
                                                  const bool with_rho, int bid, int nb) {
  using TR = typename Store<UR>::T;
  using TZ = typename Store<UZ>::T;
  using TD = typename Store<(UZ == P64) ? P64 : P32>::T;
  constexpr int smin = cmin(cmin((int)sizeof(TR), (int)sizeof(TD)), (int)sizeof(TZ));
  constexpr int smax = cmax(cmax((int)sizeof(TR), (int)sizeof(TD)), (int)sizeof(TZ));
  constexpr int E = chunk_elems(smin, smax);
  constexpr int U = cmax(1, BIF / (E * (int)(2 * sizeof(TR) + sizeof(TD) + 2 * sizeof(TZ))));
  const TR* r = rvec<UR>(c);
  const TR* w = qvec<UR>(c);
  TZ* z = zvec<UZ>(c);
  TZ* dv = dvec<UZ>(c);
  const TD* dinv;
  if constexpr (UZ == P64) dinv = c.dinv64; else dinv = c.dinv32;
  const int64_t nchunk = c.npad / E;
  const int64_t stride = (int64_t)nb * blockDim.x;
  double sum = 0.0;
  for (int64_t base = (int64_t)bid * blockDim.x + threadIdx.x; base < nchunk; base += stride * U) {
    Chunk<TR, E> rr[U], ww[U];
    Chunk<TD, E> ii[U];
    Chunk<TZ, E> dd[U], zz[U];
#pragma unroll
    for (int u = 0; u < U; ++u) {
      const int64_t i = base + u * stride;
      if (i < nchunk) {
        chunk_load(rr[u], r, i); chunk_load(ww[u], w, i); chunk_load(ii[u], dinv, i);
        chunk_load(dd[u], dv, i); chunk_load(zz[u], z, i);
      }
    }
#pragma unroll
    for (int u = 0; u < U; ++u) {
      const int64_t i = base + u * stride;
      if (i < nchunk) {
        double rv[E], wv[E], iv[E], dvv[E], zv[E];
        chunk_unpack(rr[u], rv); chunk_unpack(ww[u], wv); chunk_unpack(ii[u], iv);
        chunk_unpack(dd[u], dvv); chunk_unpack(zz[u], zv);
#pragma unroll
        for (int e = 0; e < E; ++e) {
          const double t = __dsub_rn(__dmul_rn(rv[e], omega), wv[e]);
          const double uu = __dmul_rn(t, iv[e]);
          dvv[e] = __fma_rn(c1, dvv[e], __dmul_rn(c2, uu));
        }
        Chunk<TZ, E> dout;
        chunk_pack(dout, dvv);   // one rounding to u_z
        chunk_store(dout, dv, i);
        chunk_unpack(dout, dvv);
#pragma unroll
        for (int e = 0; e < E; ++e) zv[e] = __dadd_rn(zv[e], dvv[e]);
        Chunk<TZ, E> zout;
        chunk_pack(zout, zv);    // one rounding to u_z
        chunk_store(zout, z, i);
        if (with_rho) {
          chunk_unpack(zout, zv);
#pragma unroll
          for (int e = 0; e < E; ++e) sum = fma(rv[e], zv[e], sum);
        }
      }
    }
  }
  return sum;
}

// ------------------------------------------------------------------ a3: p -------------------
// PS: precision p_{k-1} is stored in; UZ: precision of z_k and p_k (PS != UZ only at a u_z
// switch, where p_{k-1} <- RN_{u_z}(p_{k-1}) is fused here, reading R9).
// shadow32 (only with UZ = P64): also store RN32(p) into the FP32 copy of p.  While u_z = FP64 and u_r = FP32 the
// mat-vec needs RN32(p_j) for every gathered entry (reading R7); rounding each row once here instead of once per
// gather there takes an FP64->FP32 conversion per ENTRY out of the SpMV (c4: 27 per row) for 4 B per row more here.
// PUSH (row-sharded solve, k_p_sh): chunks inside a send range are also stored into the neighbour's halo band, in the
// precision the mat-vec gathers (the FP32 copy in the shadow32 phase).
template <int PS, int UZ> struct PT_ {
  using TP = typename Store<PS>::T;
  using TZ = typename Store<UZ>::T;
  static constexpr int E = chunk_elems(cmin((int)sizeof(TP), (int)sizeof(TZ)), cmax((int)sizeof(TP), (int)sizeof(TZ)));
};
template <int UZ> struct PPush {  // where the chunks of the send ranges go (all null unless PUSH)
  HaloPush<typename Store<UZ>::T> hp{nullptr, nullptr, 0, 0, 0};
  HaloPush<float> hp32{nullptr, nullptr, 0, 0, 0};
};
// p = RN_{u_z}(fma(beta, RN_{u_z}(p), z)) for chunk i (Alg 4.1 line 10); first: p = z
template <int PS, int UZ, bool PUSH>
__device__ __forceinline__ void p_chunk(const Ctx& c, const double beta, const bool first, const bool shadow32, const PPush<UZ>& ph,
                                        const Chunk<typename PT_<PS, UZ>::TZ, PT_<PS, UZ>::E>& zz,
                                        const Chunk<typename PT_<PS, UZ>::TP, PT_<PS, UZ>::E>& pp, const int64_t i) {
  using T = PT_<PS, UZ>;
  constexpr int E = T::E;
  double a[E], zv[E];
  chunk_unpack(zz, zv);
  if (!first) {
    chunk_unpack(pp, a);
    if constexpr (PS != UZ) {
#pragma unroll
      for (int e = 0; e < E; ++e) a[e] = round_to<UZ>(a[e]);
    }
  } else {
#pragma unroll
    for (int e = 0; e < E; ++e) a[e] = 0.0;
  }
#pragma unroll
  for (int e = 0; e < E; ++e) a[e] = fma(beta, a[e], zv[e]);
  Chunk<typename T::TZ, E> po;
  chunk_pack(po, a);
  chunk_store(po, pvec<UZ>(c), i);
  bool pushed = false;
  if constexpr (UZ == P64) {
    if (shadow32) {
      Chunk<float, E> p32;
      chunk_pack(p32, a);
      chunk_store(p32, c.p32, i);
      if constexpr (PUSH) halo_push_chunk(ph.hp32, p32, i);
      pushed = true;
    }
  }
  if constexpr (PUSH) {
    if (!pushed) halo_push_chunk(ph.hp, po, i);
  }
#ifdef AMP_COUNT_FP16
  if (UZ == P16) {
    double h[E];
    chunk_unpack(po, h);
#pragma unroll
    for (int e = 0; e < E; ++e) count_fp16(c.st, a[e], h[e]);
  }
#endif
}

template <int PS, int UZ, int BIF = kVecBytesInFlight, bool PUSH = false>
__device__ __forceinline__ void phase_p(const Ctx& c, const double beta, const bool first, const bool shadow32, int bid, int nb) {
  using T = PT_<PS, UZ>;
  using TP = typename T::TP;
  using TZ = typename T::TZ;
  constexpr int E = T::E;
  constexpr int U = cmax(1, BIF / (E * (int)(sizeof(TP) + sizeof(TZ))));
  const TP* pin = pvec<PS>(c);
  const TZ* z = zvec<UZ>(c);
  const int64_t nchunk = c.npad / E;
  const int64_t stride = (int64_t)nb * blockDim.x;
  PPush<UZ> ph;
  if constexpr (PUSH) { ph.hp = halo_push_of<UZ>(c); ph.hp32 = halo_push_of<P32>(c); }
  for (int64_t base = (int64_t)bid * blockDim.x + threadIdx.x; base < nchunk; base += stride * U) {
    Chunk<TP, E> pp[U];
    Chunk<TZ, E> zz[U];
#pragma unroll
    for (int u = 0; u < U; ++u) {
      const int64_t i = base + u * stride;
      if (i < nchunk) {
        chunk_load(zz[u], z, i);
        if (!first) chunk_load(pp[u], pin, i);
      }
    }
#pragma unroll
    for (int u = 0; u < U; ++u) {
      const int64_t i = base + u * stride;
      if (i < nchunk) p_chunk<PS, UZ, PUSH>(c, beta, first, shadow32, ph, zz[u], pp[u], i);
    }
  }
}

// ------------------------------------------------------------------ a5: x, r, delta ---------
template <int UR, int UZ> struct XRT {
  using TZ = typename Store<UZ>::T;
  using TR = typename Store<UR>::T;
  static constexpr int E = chunk_elems(cmin((int)sizeof(TZ), (int)sizeof(TR)), 8);
};
// chunk i of x, which is caller-owned and exactly n long: the last chunk may be partial
template <int E> __device__ __forceinline__ void x_chunk_load(Chunk<double, E>& k, const double* x, const int64_t i, const int64_t n) {
  if ((i + 1) * E <= n) {
    chunk_load(k, x, i);
  } else {
    double t[E];
#pragma unroll
    for (int e = 0; e < E; ++e) t[e] = (i * E + e < n) ? x[i * E + e] : 0.0;
    chunk_pack(k, t);
  }
}
template <int E> __device__ __forceinline__ void x_chunk_store(const double (&xv)[E], double* x, const int64_t i, const int64_t n) {
  if ((i + 1) * E <= n) {
    Chunk<double, E> xo;
    chunk_pack(xo, xv);
    chunk_store(xo, x, i);
  } else {
#pragma unroll
    for (int e = 0; e < E; ++e)
      if (i * E + e < n) x[i * E + e] = xv[e];
  }
}
// x += alpha p (FP64); r = RN_{u_r}(fma(-alpha, q, r)); sum += r^2 with the stored r (Alg 4.1 lines 15-17)
template <int UR, int UZ>
__device__ __forceinline__ void xr_chunk(const Ctx& c, const double alpha, double* x, const Chunk<double, XRT<UR, UZ>::E>& xx,
                                         const Chunk<typename XRT<UR, UZ>::TZ, XRT<UR, UZ>::E>& pp,
                                         const Chunk<typename XRT<UR, UZ>::TR, XRT<UR, UZ>::E>& qq,
                                         const Chunk<typename XRT<UR, UZ>::TR, XRT<UR, UZ>::E>& rr, const int64_t i, double& sum) {
  using T = XRT<UR, UZ>;
  constexpr int E = T::E;
  double xv[E], pv[E], qv[E], rv[E];
  chunk_unpack(xx, xv);
  chunk_unpack(pp, pv);
  chunk_unpack(qq, qv);
  chunk_unpack(rr, rv);
#pragma unroll
  for (int e = 0; e < E; ++e) xv[e] = fma(alpha, pv[e], xv[e]);  // line 15, FP64
  x_chunk_store<E>(xv, x, i, c.n);
#pragma unroll
  for (int e = 0; e < E; ++e) rv[e] = fma(-alpha, qv[e], rv[e]);  // line 16
  Chunk<typename T::TR, E> ro;
  chunk_pack(ro, rv);  // one rounding to u_r
  chunk_store(ro, rvec<UR>(c), i);
  chunk_unpack(ro, rv);
#pragma unroll
  for (int e = 0; e < E; ++e) sum = fma(rv[e], rv[e], sum);
}

template <int UR, int UZ, int BIF = kVecBytesInFlight>
__device__ __forceinline__ double phase_xr(const Ctx& c, const double alpha, double* x, int bid, int nb) {
  using T = XRT<UR, UZ>;
  using TZ = typename T::TZ;
  using TR = typename T::TR;
  constexpr int E = T::E;
  constexpr int U = cmax(1, BIF / (E * (int)(8 + sizeof(TZ) + 2 * sizeof(TR))));
  const TZ* p = pvec<UZ>(c);
  const TR* q = qvec<UR>(c);
  const TR* r = rvec<UR>(c);
  const int64_t n = c.n;
  const int64_t nchunk = c.npad / E;
  const int64_t stride = (int64_t)nb * blockDim.x;
  double sum = 0.0;
  for (int64_t base = (int64_t)bid * blockDim.x + threadIdx.x; base < nchunk; base += stride * U) {
    Chunk<double, E> xx[U];
    Chunk<TZ, E> pp[U];
    Chunk<TR, E> qq[U], rr[U];
#pragma unroll
    for (int u = 0; u < U; ++u) {
      const int64_t i = base + u * stride;
      if (i < nchunk) {
        x_chunk_load<E>(xx[u], x, i, n);
        chunk_load(pp[u], p, i);
        chunk_load(qq[u], q, i);
        chunk_load(rr[u], r, i);
      }
    }
#pragma unroll
    for (int u = 0; u < U; ++u) {
      const int64_t i = base + u * stride;
      if (i < nchunk) xr_chunk<UR, UZ>(c, alpha, x, xx[u], pp[u], qq[u], rr[u], i, sum);
    }
  }
  return sum;
}

// ------------------------------------------------------------------ lagged: a5 + a2 in one pass
// x += alpha p (FP64); r <- RN_{URN}(r - alpha q); delta^2 += r^2; z = RN_{UZN}((r omega_n) dinv); rho += r z.
// UR / UZ: precisions of iteration k (q, r as read, p); URN / UZN: of iteration k+1 (r as written, z).
template <int UR, int URN, int UZ, int UZN> struct XRZT {
  using TP = typename Store<UZ>::T;
  using TR = typename Store<UR>::T;
  using TO = typename Store<URN>::T;
  using TZ = typename Store<UZN>::T;
  using TD = typename Store<(UZN == P64) ? P64 : P32>::T;
  static constexpr int smin = cmin(cmin((int)sizeof(TP), (int)sizeof(TR)), cmin((int)sizeof(TO), (int)sizeof(TZ)));
  static constexpr int E = chunk_elems(smin, 8);
  static __device__ __forceinline__ const TD* dinv(const Ctx& c) {
    if constexpr (UZN == P64) return c.dinv64; else return c.dinv32;
  }
};
template <int UR, int URN, int UZ, int UZN>
__device__ __forceinline__ void xrz_chunk(const Ctx& c, const double alpha, const double omega_n, double* x,
                                          const Chunk<double, XRZT<UR, URN, UZ, UZN>::E>& xx,
                                          const Chunk<typename XRZT<UR, URN, UZ, UZN>::TP, XRZT<UR, URN, UZ, UZN>::E>& pp,
                                          const Chunk<typename XRZT<UR, URN, UZ, UZN>::TR, XRZT<UR, URN, UZ, UZN>::E>& qq,
                                          const Chunk<typename XRZT<UR, URN, UZ, UZN>::TR, XRZT<UR, URN, UZ, UZN>::E>& rr,
                                          const Chunk<typename XRZT<UR, URN, UZ, UZN>::TD, XRZT<UR, URN, UZ, UZN>::E>& dd, const int64_t i,
                                          double& srr, double& srz) {
  using T = XRZT<UR, URN, UZ, UZN>;
  constexpr int E = T::E;
  double xv[E], pv[E], qv[E], rv[E], dv[E], zv[E];
  chunk_unpack(xx, xv);
  chunk_unpack(pp, pv);
  chunk_unpack(qq, qv);
  chunk_unpack(rr, rv);
  chunk_unpack(dd, dv);
#pragma unroll
  for (int e = 0; e < E; ++e) xv[e] = fma(alpha, pv[e], xv[e]);  // line 15, FP64
  x_chunk_store<E>(xv, x, i, c.n);
#pragma unroll
  for (int e = 0; e < E; ++e) rv[e] = fma(-alpha, qv[e], rv[e]);  // line 16
  Chunk<typename T::TO, E> ro;
  chunk_pack(ro, rv);  // one rounding, to the precision of iteration k+1
  chunk_store(ro, rvec<URN>(c), i);
  chunk_unpack(ro, rv);
#pragma unroll
  for (int e = 0; e < E; ++e) zv[e] = (rv[e] * omega_n) * dv[e];  // lines 4-5 of iteration k+1
  Chunk<typename T::TZ, E> zo;
  chunk_pack(zo, zv);
  chunk_store(zo, zvec<UZN>(c), i);
#ifdef AMP_COUNT_FP16
  double zx[E];
#pragma unroll
  for (int e = 0; e < E; ++e) zx[e] = zv[e];
#endif
  chunk_unpack(zo, zv);
#ifdef AMP_COUNT_FP16
  if (UZN == P16) {
#pragma unroll
    for (int e = 0; e < E; ++e) count_fp16(c.st, zx[e], zv[e]);
  }
#endif
#pragma unroll
  for (int e = 0; e < E; ++e) { srr = fma(rv[e], rv[e], srr); srz = fma(rv[e], zv[e], srz); }
}

template <int UR, int URN, int UZ, int UZN, int BIF = kVecBytesInFlight>
__device__ __forceinline__ void phase_xrz(const Ctx& c, const double alpha, const double omega_n, double* x, int bid, int nb,
                                          double& sum_rr, double& sum_rz) {
  using T = XRZT<UR, URN, UZ, UZN>;
  using TP = typename T::TP;
  using TR = typename T::TR;
  using TD = typename T::TD;
  constexpr int E = T::E;
  constexpr int U = cmax(1, BIF / (E * (int)(8 + sizeof(TP) + 2 * sizeof(TR) + sizeof(TD))));
  const TP* p = pvec<UZ>(c);
  const TR* q = qvec<UR>(c);
  const TR* rin = rvec<UR>(c);
  const TD* dinv = T::dinv(c);
  const int64_t n = c.n;
  const int64_t nchunk = c.npad / E;
  const int64_t stride = (int64_t)nb * blockDim.x;
  double srr = 0.0, srz = 0.0;
  for (int64_t base = (int64_t)bid * blockDim.x + threadIdx.x; base < nchunk; base += stride * U) {
    Chunk<double, E> xx[U];
    Chunk<TP, E> pp[U];
    Chunk<TR, E> qq[U], rr[U];
    Chunk<TD, E> dd[U];
#pragma unroll
    for (int u = 0; u < U; ++u) {
      const int64_t i = base + u * stride;
      if (i < nchunk) {
        x_chunk_load<E>(xx[u], x, i, n);
        chunk_load(pp[u], p, i);
        chunk_load(qq[u], q, i);
        chunk_load(rr[u], rin, i);
        chunk_load(dd[u], dinv, i);
      }
    }
#pragma unroll
    for (int u = 0; u < U; ++u) {
      const int64_t i = base + u * stride;
      if (i < nchunk) xrz_chunk<UR, URN, UZ, UZN>(c, alpha, omega_n, x, xx[u], pp[u], qq[u], rr[u], dd[u], i, srr, srz);
    }
  }
  sum_rr = srr;
  sum_rz = srz;
}

}  // namespace amp
