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
  int64_t n;
  cudaGraphConditionalHandle cond;
  int32_t use_cond;
};
__device__ __forceinline__ EpiCtx epi_ctx(const Ctx& c) { return EpiCtx{c.st, c.n, c.cond, c.use_cond}; }
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

// NOTE: the loop vectors (r, z, p, q, x) are deliberately NOT __restrict__/read-only qualified:
// inside the persistent kernel they are written by earlier phases of the same kernel, so they
// must be read with plain coherent loads (ordered by the grid barrier), never ld.global.nc.
// Loads are grouped ahead of the stores by hand (kVecUnroll chunks in flight per thread).

// ------------------------------------------------------------------ a2: z and rho ------------
// RS: precision r is stored in; UR: precision selected for r (RS != UR only at the iteration of
// the u_r switch, where r <- RN32(r) is fused here, step a6); UZ: precision of z.
template <int RS, int UR, int UZ>
__device__ __forceinline__ double phase_z(const Ctx& c, const double omega, int bid, int nb) {
  using TR = typename Store<RS>::T;
  using TD = typename Store<(UZ == P64) ? P64 : P32>::T;
  const TR* rin = rvec<RS>(c);
  typename Store<UR>::T* rout = rvec<UR>(c);
  typename Store<UZ>::T* z = zvec<UZ>(c);
  const TD* dinv;
  if constexpr (UZ == P64) dinv = c.dinv64; else dinv = c.dinv32;
  const int64_t npair = c.npad >> 1;
  const int64_t stride = (int64_t)nb * blockDim.x;
  constexpr int U = (RS == P64 && UZ == P64) ? kVecUnrollWide : kVecUnrollNarrow;
  double sum = 0.0;
  for (int64_t base = (int64_t)bid * blockDim.x + threadIdx.x; base < npair; base += stride * U) {
    typename Raw2<TR>::T rr[U];
    typename Raw2<TD>::T dd[U];
#pragma unroll
    for (int u = 0; u < U; ++u) {
      const int64_t i = base + u * stride;
      if (i < npair) { rr[u] = load_raw(rin, i); dd[u] = load_raw(dinv, i); }
    }
#pragma unroll
    for (int u = 0; u < U; ++u) {
      const int64_t i = base + u * stride;
      if (i < npair) {
        double a0, a1, d0, d1;
        unpack(rr[u], a0, a1);
        unpack(dd[u], d0, d1);
        if (RS != UR) {  // r <- RN_{u_r}(r) at the switch iteration
          a0 = round_to<UR>(a0); a1 = round_to<UR>(a1);
          store2(rout, i, a0, a1);
        }
        const double z0 = round_to<UZ>((a0 * omega) * d0);
        const double z1 = round_to<UZ>((a1 * omega) * d1);
        store2(z, i, z0, z1);
#ifdef AMP_COUNT_FP16
        if (UZ == P16) { count_fp16(c.st, (a0 * omega) * d0, z0); count_fp16(c.st, (a1 * omega) * d1, z1); }
#endif
        sum = fma(a0, z0, sum);
        sum = fma(a1, z1, sum);
      }
    }
  }
  return sum;
}

// ------------------------------------------------------------------ a3: p -------------------
// PS: precision p_{k-1} is stored in; UZ: precision of z_k and p_k (PS != UZ only at a u_z
// switch, where p_{k-1} <- RN_{u_z}(p_{k-1}) is fused here, reading R9).
template <int PS, int UZ>
__device__ __forceinline__ void phase_p(const Ctx& c, const double beta, const bool first, int bid, int nb) {
  using TP = typename Store<PS>::T;
  using TZ = typename Store<UZ>::T;
  const TP* pin = pvec<PS>(c);
  TZ* pout = pvec<UZ>(c);
  const TZ* z = zvec<UZ>(c);
  const int64_t npair = c.npad >> 1;
  const int64_t stride = (int64_t)nb * blockDim.x;
  constexpr int U = kVecUnrollNarrow;
  for (int64_t base = (int64_t)bid * blockDim.x + threadIdx.x; base < npair; base += stride * U) {
    typename Raw2<TP>::T pp[U];
    typename Raw2<TZ>::T zz[U];
#pragma unroll
    for (int u = 0; u < U; ++u) {
      const int64_t i = base + u * stride;
      if (i < npair) {
        zz[u] = load_raw(z, i);
        if (!first) pp[u] = load_raw(pin, i);
      }
    }
#pragma unroll
    for (int u = 0; u < U; ++u) {
      const int64_t i = base + u * stride;
      if (i < npair) {
        double a0 = 0.0, a1 = 0.0, z0, z1;
        unpack(zz[u], z0, z1);
        if (!first) unpack(pp[u], a0, a1);
        if (PS != UZ) { a0 = round_to<UZ>(a0); a1 = round_to<UZ>(a1); }
        const double n0 = fma(beta, a0, z0), n1 = fma(beta, a1, z1);
        store2(pout, i, n0, n1);
#ifdef AMP_COUNT_FP16
        if (UZ == P16) { count_fp16(c.st, n0, round_to<P16>(n0)); count_fp16(c.st, n1, round_to<P16>(n1)); }
#endif
      }
    }
  }
}

// ------------------------------------------------------------------ a5: x, r, delta ---------
template <int UR, int UZ>
__device__ __forceinline__ double phase_xr(const Ctx& c, const double alpha, double* x, int bid, int nb) {
  using TZ = typename Store<UZ>::T;
  using TR = typename Store<UR>::T;
  const TZ* p = pvec<UZ>(c);
  const TR* q = qvec<UR>(c);
  TR* r = rvec<UR>(c);
  const int64_t n = c.n;
  const int64_t npair = c.npad >> 1;
  const int64_t stride = (int64_t)nb * blockDim.x;
  constexpr int U = kVecUnrollNarrow;
  double sum = 0.0;
  for (int64_t base = (int64_t)bid * blockDim.x + threadIdx.x; base < npair; base += stride * U) {
    double2 xx[U];
    typename Raw2<TZ>::T pp[U];
    typename Raw2<TR>::T qq[U], rr[U];
#pragma unroll
    for (int u = 0; u < U; ++u) {
      const int64_t i = base + u * stride;
      if (i < npair) {
        if (2 * i + 1 < n) xx[u] = load_raw(x, i);
        else xx[u] = make_double2((2 * i < n) ? x[2 * i] : 0.0, 0.0);  // x is caller-owned: exactly n long
        pp[u] = load_raw(p, i);
        qq[u] = load_raw(q, i);
        rr[u] = load_raw(r, i);
      }
    }
#pragma unroll
    for (int u = 0; u < U; ++u) {
      const int64_t i = base + u * stride;
      if (i < npair) {
        double p0, p1, q0, q1, r0, r1;
        unpack(pp[u], p0, p1);
        unpack(qq[u], q0, q1);
        unpack(rr[u], r0, r1);
        const double nx0 = fma(alpha, p0, xx[u].x), nx1 = fma(alpha, p1, xx[u].y);  // line 15, FP64
        if (2 * i + 1 < n) store2(x, i, nx0, nx1);
        else if (2 * i < n) x[2 * i] = nx0;
        const double nr0 = round_to<UR>(fma(-alpha, q0, r0));  // line 16, one rounding to u_r
        const double nr1 = round_to<UR>(fma(-alpha, q1, r1));
        store2(r, i, nr0, nr1);
        sum = fma(nr0, nr0, sum);
        sum = fma(nr1, nr1, sum);
      }
    }
  }
  return sum;
}

}  // namespace amp
