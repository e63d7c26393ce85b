// =========================================================================================
// oracle/amp_pcg_oracle.cpp — TEST INFRASTRUCTURE, NOT PRODUCT CODE.
//
// Plain, slow, CPU-only restatement of the algorithms of arXiv 2505.04155 (Guo, de Sturler,
// Warburton, "An adaptive mixed-precision and dynamically scaled preconditioned conjugate
// gradient algorithm"), written from /root/reference/PAPER.md and nothing else.  It shares no
// code, header, table or constant with the CUDA library under paper_2505_04155_b200/ and is
// only ever called from tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
// --impl reference legs.
//
// What is here, with the passage each piece follows:
//   orc_round_fp16 / orc_round_fp32   IEEE binary16 / binary32 round-to-nearest-even of a
//                                     double (gradual underflow, overflow -> +-inf): the
//                                     storage formats of PAPER.md:236-241, :504.
//   orc_spmv_fp64 / orc_spmv_fp32     q = A p on CSR: row sums in CSR order (an fma chain in
//                                     the working precision u_r, "compute and
//                                     store q_k" in u_r).
//   orc_pcg / orc_amp_pcg             Algorithm 3.1, Algorithm 3.2
//                                     (:184-221, via scale modes) and Algorithm 4.1
//                                     (:264-309) with the precision selector (4.1)
//                                     (:245-253) and the indicators (4.9)/(4.10) (:359-366)
//                                     and (4.11) (:370-375).  x, all inner products, norms
//                                     and scalars are FP64.
//   orc_eta_posteriori                the a-posteriori indicator eta_hat_m(k) of (4.7) (:350-354).
//   orc_cheb_*                        Chebyshev-accelerated Jacobi preconditioner (the paper's smoother, :461; reading R18).
//   orc_step_z / orc_step_p / orc_step_xr   the vector steps of the loop body (Alg 4.1 lines 4-5, 10, 15-16),
//                                     called by orc_amp_pcg and, one at a time, by the per-step GPU parity tests.
//
// Low-precision STORAGE is emulated by explicit rounding: every vector is a double array that
// holds values exactly representable in its storage format.  Readings of the garbled or
// silent places of the paper are those of DESIGN.md ("Readings", R1..R16).
//
// Reductions (dot products, norms) are FP64 sums of FP64 products, accumulated in fixed
// chunks of ORC_CHUNK elements whose partial sums are added in index order, so the result
// does not depend on the OpenMP thread count.  (A sum has no order in the paper.)
//
// Parity status: every function below is pinned by tests/test_oracle_*.py against facts the
// paper or mathematics fix.  The exact AMP iteration counts on
// the five BASELINE configs are "parity unpinned" by the paper (it prints none).
// =========================================================================================
#include <cmath>
#include <cstdint>
#include <cstdlib>
#include <cstring>
#include <limits>
#include <vector>

#define ORC_CHUNK 4096

extern "C" {

// ---------------------------------------------------------------- storage rounding -------
// binary32: the hardware cast is IEEE round-to-nearest-even, with gradual underflow and
// overflow to infinity.
double orc_round_fp32(double v) { return (double)(float)v; }

// binary16, directly from the double (no double rounding through float):
//   normal range   |v| in [2^-14, 65520): spacing 2^(e-10) with e = floor(log2|v|)
//   subnormal      |v| < 2^-14: spacing 2^-24 (so |v| <= 2^-25 rounds to 0, ties-to-even)
//   overflow       |v| >= 65520 (the midpoint of 65504 and 2^16, which ties to even = 2^16)
double orc_round_fp16(double v) {
  if (std::isnan(v) || std::isinf(v) || v == 0.0) return v;
  double a = std::fabs(v), r;
  if (a >= 65520.0) {
    r = std::numeric_limits<double>::infinity();
  } else if (a < 6.103515625e-05) {                        // 2^-14
    const double q = 5.9604644775390625e-08;               // 2^-24
    r = std::nearbyint(a / q) * q;                         // exact scaling; nearbyint = RN-even
  } else {
    int e;
    std::frexp(a, &e);                                     // a = f * 2^e, f in [0.5,1)
    const double q = std::ldexp(1.0, e - 1 - 10);          // spacing in this binade
    r = std::nearbyint(a / q) * q;
  }
  return std::copysign(r, v);
}

void orc_round_array(int64_t n, const double* in, double* out, int prec) {   // prec: 1 FP32, 2 FP16
  for (int64_t i = 0; i < n; ++i) out[i] = (prec == 2) ? orc_round_fp16(in[i]) : (prec == 1 ? orc_round_fp32(in[i]) : in[i]);
}

static inline double round_store(double v, int prec) {     // prec: 0 FP64, 1 FP32, 2 FP16
  return prec == 0 ? v : (prec == 1 ? orc_round_fp32(v) : orc_round_fp16(v));
}

// ---------------------------------------------------------------- reductions --------------
static double dot_fp64(int64_t n, const double* a, const double* b) {
  const int64_t nchunk = (n + ORC_CHUNK - 1) / ORC_CHUNK;
  std::vector<double> part((size_t)nchunk);
#pragma omp parallel for schedule(static)
  for (int64_t c = 0; c < nchunk; ++c) {
    const int64_t lo = c * ORC_CHUNK, hi = (lo + ORC_CHUNK < n) ? lo + ORC_CHUNK : n;
    double s = 0.0;
    for (int64_t i = lo; i < hi; ++i) s += a[i] * b[i];
    part[(size_t)c] = s;
  }
  double s = 0.0;
  for (int64_t c = 0; c < nchunk; ++c) s += part[(size_t)c];
  return s;
}

double orc_dot(int64_t n, const double* a, const double* b) { return dot_fp64(n, a, b); }

// ---------------------------------------------------------------- SpMV --------------------
// q_i = sum_{j in row i, CSR order} a_ij p_j, FP64 fma chain ("q <- A p").
void orc_spmv_fp64(int64_t n, const int32_t* rowptr, const int32_t* colidx, const double* vals,
                   const double* p, double* q) {
#pragma omp parallel for schedule(static)
  for (int64_t i = 0; i < n; ++i) {
    double s = 0.0;
    for (int32_t e = rowptr[i]; e < rowptr[i + 1]; ++e) s = std::fma(vals[e], p[colidx[e]], s);
    q[i] = s;
  }
}

// u_r = FP32: matrix values are the FP32-rounded copy, p_j is converted to
// float (exact when p is stored in FP16/FP32, one rounding when stored in FP64), the row sum is
// a float fma chain in CSR order; q is returned as doubles holding float values.
// accumulate64 != 0 selects the diagnostic variant: FP64 fma chain of (float a)*(float p),
// rounded once to FP32.
void orc_spmv_fp32(int64_t n, const int32_t* rowptr, const int32_t* colidx, const float* vals32,
                   const double* p, double* q, int accumulate64) {
#pragma omp parallel for schedule(static)
  for (int64_t i = 0; i < n; ++i) {
    if (accumulate64) {
      double s = 0.0;
      for (int32_t e = rowptr[i]; e < rowptr[i + 1]; ++e)
        s = std::fma((double)vals32[e], (double)(float)p[colidx[e]], s);
      q[i] = (double)(float)s;
    } else {
      float s = 0.0f;
      for (int32_t e = rowptr[i]; e < rowptr[i + 1]; ++e) s = std::fmaf(vals32[e], (float)p[colidx[e]], s);
      q[i] = (double)s;
    }
  }
}

// ---------------------------------------------------------------- policy / stats ----------
enum { ORC_FP64 = 0, ORC_FP32 = 1, ORC_FP16 = 2 };
enum { ORC_ETA_DELAY = 0, ORC_ETA_LINEAR = 1, ORC_ETA_NEVER = 2 };
enum { ORC_SCALE_NORM2 = 0, ORC_SCALE_RMS = 1, ORC_SCALE_POW2 = 2, ORC_SCALE_NONE = 3, ORC_SCALE_LAGGED = 4 };

struct orc_policy {
  int32_t amp;              // 0: Algorithm 3.1 literally; 1: Algorithm 4.1
  int32_t u0;               // initial / maximum precision of z, p
  int32_t eta_rule;         // (4.9)+(4.10), (4.11), or never (u_r stays FP64)
  int32_t d, ell;           // delay d of (4.9), window ell of (4.11)
  int32_t scale_mode;       // omega_k: 1/||r_k|| (Alg 4.1 l.4), sqrt(n)/||r_k||, 2^round(log2(1/||r_k||)), 1
  int32_t no_stop;          // 1: ignore the stopping test, run maxit iterations
  int32_t strict_rounding;  // diagnostic R6: y and M^-1 stored in u_z, two roundings
  int32_t accumulate64;     // diagnostic R7: FP32-phase SpMV accumulated in FP64
  int32_t precond;          // 0: M = I ; 1: Jacobi, M = diag(A) ; 2: Chebyshev-accelerated Jacobi (reading R18)
  int32_t cheb_degree;      // number of Jacobi sweeps s >= 1 of one application (s - 1 mat-vecs); "second-order": 2
  int32_t pad0;
  double cheb_lmin, cheb_lmax;  // bounds of the spectrum of D^-1 A the polynomial is built for; 0, 0: orc_cheb_default_bounds
  double C;                 // constant of Assumption 4.1, default 1
  double tau_zs, tau_zh;    // thresholds (5.1)
  double eps32;             // unit roundoff of FP32, 2^-24
  double eta_safety, stop_safety;  // 1,1 = paper; theta, 1-theta = strict split of (3.10)
};

struct orc_stats {
  int32_t status;           // 0 converged, 1 maxit reached, -2 breakdown
  int32_t iters, it_ur32, it_uz32, it_uz16;
  double bnorm, relres_updated, relres_true;
  int64_t fp16_subnormal, fp16_flushed, fp16_inf, fp16_stored;   // z and p stores in FP16
};

// trace callback: called once per iteration after step O11 with the vectors of that iteration.
// scal = {rho, beta, gamma, alpha, delta_k, delta_{k+1}, omega, eta_k, u_r, u_z}
typedef void (*orc_trace_fn)(int32_t k, const double* x, const double* r, const double* z,
                             const double* p, const double* q, const double* scal, void* user);

// A-posteriori attainable-accuracy indicator eta_hat_m(k), PAPER.md:350-354 (4.7), written out as
// the two sums of its definition for one k (m = final iteration index, hist[t] = ||r_t||, t = 0..m):
//   sum_{t=0}^{k} eps64 ((3+C)||r_{t-1}|| + (2+C)||r_t||) + sum_{t=k}^{m} eps32 ((3+C)||r_{t-1}|| + (2+C)||r_t||)
// Reading R2: ||r_{-1}|| is taken as ||r_0||.  Diagnostic only (needs the whole history).
double orc_eta_posteriori(const double* hist, int32_t m, int32_t k, double C, double eps32, double eps64) {
  double s64 = 0.0, s32 = 0.0;
  for (int32_t t = 0; t <= k; ++t) s64 += eps64 * ((3.0 + C) * hist[t > 0 ? t - 1 : 0] + (2.0 + C) * hist[t]);
  for (int32_t t = k; t <= m; ++t) s32 += eps32 * ((3.0 + C) * hist[t > 0 ? t - 1 : 0] + (2.0 + C) * hist[t]);
  return s64 + s32;
}

// eta_k, PAPER.md:361-362 (4.9) and :372-373 (4.11).  hist[t] = ||r_t||, t = 0..k.
// Reading R2: for t < 0 the norm is taken as ||r_0||.
double orc_eta(const orc_policy* pol, const double* hist, int32_t k) {
  const double inf = std::numeric_limits<double>::infinity();
  if (pol->eta_rule == ORC_ETA_NEVER) return inf;
  const double C = pol->C, e32 = pol->eps32;
  if (pol->eta_rule == ORC_ETA_DELAY) {
    double s = 0.0;
    for (int32_t t = k - pol->d; t <= k; ++t) {
      const double hm1 = hist[(t - 1) > 0 ? (t - 1) : 0], h0 = hist[t > 0 ? t : 0];
      s += e32 * ((3.0 + C) * hm1 + (2.0 + C) * h0);
    }
    return s;
  }
  const int32_t l = pol->ell;
  if (k >= l && l >= 1 && hist[k] < hist[k - l]) {
    const double rate = std::pow(hist[k] / hist[k - l], 1.0 / (double)l);
    return e32 * (5.0 + 2.0 * C) * hist[k - 1] / (1.0 - rate);
  }
  return inf;
}

static inline int lower_prec(int a, int b) { return a > b ? a : b; }  // larger code = lower precision

// u_z by the selector (4.1)
int32_t orc_select_uz(const orc_policy* pol, double nu) {
  if (nu >= pol->tau_zs) return pol->u0;
  if (nu >= pol->tau_zh) return lower_prec(pol->u0, ORC_FP32);
  return lower_prec(pol->u0, ORC_FP16);
}

static double scale_factor(const orc_policy* pol, double delta, int64_t n) {
  switch (pol->scale_mode) {
    case ORC_SCALE_NORM2: return 1.0 / delta;                               // Alg 4.1 line 4
    case ORC_SCALE_LAGGED: return 1.0 / delta;                              // called with ||r_{k-1}|| (see the loop)
    case ORC_SCALE_RMS:   return std::sqrt((double)n) / delta;
    case ORC_SCALE_POW2:  return std::ldexp(1.0, (int)std::nearbyint(std::log2(1.0 / delta)));
    default:              return 1.0;
  }
}

// classification of one FP16 store: 1 = became inf, 2 = flushed to zero, 3 = subnormal, 0 = other
static inline int classify_fp16(double unrounded, double stored) {
  if (std::isinf(stored) && !std::isinf(unrounded)) return 1;
  if (stored == 0.0 && unrounded != 0.0) return 2;
  if (stored != 0.0 && std::fabs(stored) < 6.103515625e-05) return 3;
  return 0;
}

// ---------------------------------------------------------------- the vector steps ---------
// One function per vector step of the loop body, in the paper's notation; orc_amp_pcg below calls exactly these,
// and the per-step GPU parity tests call them one at a time.  Vectors are double arrays holding values that are
// exactly representable in their storage precision; counts (may be NULL) = {became inf, flushed to zero, subnormal}
// of the FP16 stores of this call (only counted when uz = FP16).

// O2, Alg 4.1 lines 4-5 (PAPER.md:274-276; Alg 3.2 line 3; scaling fused with the preconditioner, :223), M = diag:
//   z_i = RN_{u_z}( (r_i * omega) * dinv_i )                 FP64 arithmetic, ONE rounding (reading R6)
// strict != 0 is the diagnostic of reading R6: y = RN_{u_z}(RN_{u_r}(r omega)), M^-1 rounded to u_z, z = RN_{u_z}(y M^-1)
// (dinv must then be the FP64 1/a_ii).
void orc_step_z(int64_t n, const double* r, double omega, const double* dinv, int32_t ur, int32_t uz, int32_t strict,
                double* z, int64_t* counts) {
  int64_t c_inf = 0, c_flush = 0, c_sub = 0;
#pragma omp parallel for schedule(static) reduction(+ : c_inf, c_flush, c_sub)
  for (int64_t i = 0; i < n; ++i) {
    double zi;
    if (strict) {
      const double y = round_store(round_store(r[i] * omega, ur), uz);
      zi = y * round_store(dinv[i], uz);
    } else {
      zi = (r[i] * omega) * dinv[i];
    }
    const double zs = round_store(zi, uz);
    if (uz == ORC_FP16) { const int c = classify_fp16(zi, zs); c_inf += (c == 1); c_flush += (c == 2); c_sub += (c == 3); }
    z[i] = zs;
  }
  if (counts) { counts[0] += c_inf; counts[1] += c_flush; counts[2] += c_sub; }
}

// O5, Alg 4.1 line 10: p_i = RN_{u_z}( fma(beta, p_i, z_i) ), one rounding
void orc_step_p(int64_t n, double beta, const double* z, int32_t uz, double* p, int64_t* counts) {
  int64_t c_inf = 0, c_flush = 0, c_sub = 0;
#pragma omp parallel for schedule(static) reduction(+ : c_inf, c_flush, c_sub)
  for (int64_t i = 0; i < n; ++i) {
    const double pi = std::fma(beta, p[i], z[i]);
    const double ps = round_store(pi, uz);
    if (uz == ORC_FP16) { const int c = classify_fp16(pi, ps); c_inf += (c == 1); c_flush += (c == 2); c_sub += (c == 3); }
    p[i] = ps;
  }
  if (counts) { counts[0] += c_inf; counts[1] += c_flush; counts[2] += c_sub; }
}

// O9, O10, Alg 4.1 lines 15-16: x_i = fma(alpha, p_i, x_i) in FP64 (:241);
// r_i = RN_{u_r}( fma(-alpha, q_i, r_i) ), FP64 arithmetic on the stored values, one rounding (reading R8)
void orc_step_xr(int64_t n, double alpha, const double* p, const double* q, int32_t ur, double* x, double* r) {
#pragma omp parallel for schedule(static)
  for (int64_t i = 0; i < n; ++i) {
    x[i] = std::fma(alpha, p[i], x[i]);
    r[i] = round_store(std::fma(-alpha, q[i], r[i]), ur);
  }
}

// classification of one FP16 store (see classify_fp16), exported for its pin
int32_t orc_classify_fp16(double unrounded, double stored) { return classify_fp16(unrounded, stored); }

// ---------------------------------------------------------------- Chebyshev-accelerated Jacobi ----
// The paper's smoother ("second-order Chebyshev-accelerated Jacobi smoother [35]"; stronger
// preconditioners are its stated remedy for hard spectra, :584) used as the preconditioner M^-1 of the loop.  The paper
// gives no formulas; this is the textbook Chebyshev iteration for A z = y with the Jacobi splitting, started from
// z = 0 and stopped after s sweeps (reading R18 of DESIGN.md), D = diag(A), [lmin, lmax] bounds of the spectrum of
// D^-1 A:   theta = (lmax+lmin)/2, dc = (lmax-lmin)/2, sigma = theta/dc, rho_0 = 1/sigma,
//   d_0 = D^-1 y / theta,                     z_1 = d_0
//   for i = 1 .. s-1:  rho_i = 1/(2 sigma - rho_{i-1}),  t = y - A z_i,
//                      d_i = rho_i rho_{i-1} d_{i-1} + (2 rho_i / dc) D^-1 t,   z_{i+1} = z_i + d_i
// i.e. z_s = (I - q_s(D^-1 A)) A^-1 y with q_s(l) = T_s((theta - l)/dc) / T_s(sigma) (T_s: Chebyshev polynomial).
// In the mixed-precision loop y = omega r is never stored (recomputed from the stored r in FP64), d and z are stored in
// u_z with ONE rounding per update, w = A z is computed and stored in u_r like q, all scalars FP64.

// lmax = max_i (sum_j |a_ij|) / a_ii  (Gershgorin bound of D^-1 A, sums in CSR order), lmin = lmax / ratio
void orc_cheb_default_bounds(int64_t n, const int32_t* rowptr, const int32_t* colidx, const double* vals, double ratio,
                             double* lmin, double* lmax) {
  double m = 0.0;
  for (int64_t i = 0; i < n; ++i) {
    double d = 0.0, srow = 0.0;
    for (int32_t e = rowptr[i]; e < rowptr[i + 1]; ++e) {
      srow += std::fabs(vals[e]);
      if (colidx[e] == i) d += vals[e];
    }
    const double g = srow / d;
    if (g > m) m = g;
  }
  *lmax = m;
  *lmin = m / ratio;
}

// inv_theta = 1/theta; c1[i] = rho_i rho_{i-1}, c2[i] = 2 rho_i / dc for i = 1 .. s-1 (index 0 unused)
void orc_cheb_coeffs(int32_t s, double lmin, double lmax, double* inv_theta, double* c1, double* c2) {
  const double theta = (lmax + lmin) / 2.0, dc = (lmax - lmin) / 2.0, sigma = theta / dc;
  *inv_theta = 1.0 / theta;
  double rho_prev = 1.0 / sigma;
  c1[0] = c2[0] = 0.0;
  for (int32_t i = 1; i < s; ++i) {
    const double rho = 1.0 / (2.0 * sigma - rho_prev);
    c1[i] = rho * rho_prev;
    c2[i] = 2.0 * rho / dc;
    rho_prev = rho;
  }
}

// first sweep: d_i = RN_{u_z}( ((r_i omega) dinv_i) inv_theta ), z = d
void orc_cheb_first(int64_t n, const double* r, double omega, const double* dinv, double inv_theta, int32_t uz,
                    double* d, double* z) {
#pragma omp parallel for schedule(static)
  for (int64_t i = 0; i < n; ++i) {
    const double v = round_store(((r[i] * omega) * dinv[i]) * inv_theta, uz);
    d[i] = v;
    z[i] = v;
  }
}

// sweep i >= 1, given w = A z: t = r omega - w; u = t dinv; d = RN_{u_z}(fma(c1, d, c2 u)); z = RN_{u_z}(z + d)
void orc_cheb_step(int64_t n, const double* r, double omega, const double* w, const double* dinv, double c1, double c2,
                   int32_t uz, double* d, double* z) {
#pragma omp parallel for schedule(static)
  for (int64_t i = 0; i < n; ++i) {
    const double t = r[i] * omega - w[i];
    const double u = t * dinv[i];
    const double dn = round_store(std::fma(c1, d[i], c2 * u), uz);
    d[i] = dn;
    z[i] = round_store(z[i] + dn, uz);
  }
}

// one whole application z = M^-1 (omega r) in precisions (u_z, u_r); vals32 (FP32-rounded values) is read when ur = FP32;
// dinv = 1/a_ii in FP64 when uz = FP64, else its FP32-rounded copy (reading R6); work: d, w of length n
void orc_cheb_apply(int64_t n, const int32_t* rowptr, const int32_t* colidx, const double* vals, const float* vals32,
                    const double* r, double omega, const double* dinv, int32_t s, double lmin, double lmax, int32_t uz,
                    int32_t ur, double* z, double* d, double* w) {
  std::vector<double> c1((size_t)s + 1), c2((size_t)s + 1);
  double inv_theta;
  orc_cheb_coeffs(s, lmin, lmax, &inv_theta, c1.data(), c2.data());
  orc_cheb_first(n, r, omega, dinv, inv_theta, uz, d, z);
  for (int32_t i = 1; i < s; ++i) {
    if (ur == ORC_FP64) orc_spmv_fp64(n, rowptr, colidx, vals, z, w);
    else orc_spmv_fp32(n, rowptr, colidx, vals32, z, w, 0);
    orc_cheb_step(n, r, omega, w, dinv, c1[(size_t)i], c2[(size_t)i], uz, d, z);
  }
}

// ---------------------------------------------------------------- the solver --------------
// Algorithm 4.1 (amp=1) / Algorithm 3.1 (amp=0), step by step in the paper's order.
// x: in = x0, out = x_m.  hist (may be NULL) receives ||r_t||, t = 0..iters.
int32_t orc_amp_pcg(int64_t n, const int32_t* rowptr, const int32_t* colidx, const double* vals,
                    const double* b, double* x, double tol, int32_t maxit, const orc_policy* pol,
                    orc_stats* st, double* hist_out, orc_trace_fn trace, void* user) {
  std::memset(st, 0, sizeof(*st));
  st->it_ur32 = st->it_uz32 = st->it_uz16 = -1;
  std::vector<double> r((size_t)n), z((size_t)n), p((size_t)n, 0.0), q((size_t)n), dinv((size_t)n), dinv32((size_t)n);
  std::vector<float> vals32;
  std::vector<double> hist((size_t)maxit + 2, 0.0);
  const int64_t nnz = rowptr[n];

  for (int64_t i = 0; i < n; ++i) {
    double d = 1.0;
    if (pol->precond >= 1) {
      d = 0.0;   // M = diag(A) (Jacobi); duplicate entries add up, as they do in the mat-vec
      for (int32_t e = rowptr[i]; e < rowptr[i + 1]; ++e) if (colidx[e] == i) d += vals[e];
      if (!(d > 0.0)) { st->status = -1; return -1; }
    }
    dinv[(size_t)i] = 1.0 / d;
    dinv32[(size_t)i] = orc_round_fp32(1.0 / d);
  }

  const bool cheb = pol->precond == 2;
  double cheb_lmin = pol->cheb_lmin, cheb_lmax = pol->cheb_lmax;
  std::vector<double> cheb_d, cheb_w;
  if (cheb) {
    if (pol->cheb_degree < 1 || pol->cheb_degree > 16 || (pol->amp && pol->scale_mode == ORC_SCALE_LAGGED) || pol->strict_rounding) {
      st->status = -1; return -1;
    }
    if (!(cheb_lmax > 0.0)) orc_cheb_default_bounds(n, rowptr, colidx, vals, 30.0, &cheb_lmin, &cheb_lmax);
    if (!(cheb_lmin > 0.0) || !(cheb_lmax > cheb_lmin)) { st->status = -1; return -1; }
    cheb_d.resize((size_t)n); cheb_w.resize((size_t)n);
    if (vals32.empty()) { vals32.resize((size_t)nnz); for (int64_t e = 0; e < nnz; ++e) vals32[(size_t)e] = (float)vals[e]; }
  }

  // O0: r0 = b - A x0 in FP64, delta0 = ||r0||   (Alg 4.1 line 1)
  const double nb = std::sqrt(dot_fp64(n, b, b));
  st->bnorm = nb;
  orc_spmv_fp64(n, rowptr, colidx, vals, x, q.data());
  for (int64_t i = 0; i < n; ++i) r[(size_t)i] = b[i] - q[(size_t)i];
  double delta = std::sqrt(dot_fp64(n, r.data(), r.data()));
  hist[0] = delta;
  int32_t ur = ORC_FP64, uz = pol->amp ? pol->u0 : ORC_FP64;
  double rho_prev = 0.0;
  const bool lag = pol->amp && pol->scale_mode == ORC_SCALE_LAGGED;
  int32_t ur_n = ur, uz_n = uz;   // lagged variant: decisions for the next iteration
  double omega_n = 1.0;
  int32_t k = 0, status = 1;
  if (nb == 0.0) {                          // R13: b = 0 -> x = 0
    for (int64_t i = 0; i < n; ++i) x[i] = 0.0;
    delta = 0.0; status = 0; maxit = 0;
  } else if (delta <= pol->stop_safety * tol * nb && !pol->no_stop) {
    status = 0; maxit = 0;                  // R13: x0 already satisfies the test
  }

  for (k = 0; k < maxit; ++k) {
    double eta = std::numeric_limits<double>::infinity();
    double omega_lag = 1.0;
    if (pol->amp && !lag) {
      // O1: eta_k and the precision selector (4.1), Alg 4.1 line 3.
      // Reading R5: both switches are latched (precision never goes back up).
      eta = orc_eta(pol, hist.data(), k);
      if (ur == ORC_FP64 && eta <= pol->eta_safety * tol * nb) {      // (4.10)
        ur = ORC_FP32; st->it_ur32 = k;
        for (int64_t i = 0; i < n; ++i) r[(size_t)i] = orc_round_fp32(r[(size_t)i]);
        if (vals32.empty()) { vals32.resize((size_t)nnz); for (int64_t e = 0; e < nnz; ++e) vals32[(size_t)e] = (float)vals[e]; }
      }
      const int32_t want = orc_select_uz(pol, delta / nb);
      if (want > uz) {
        uz = want;
        if (uz >= ORC_FP32 && st->it_uz32 < 0) st->it_uz32 = k;
        if (uz == ORC_FP16 && st->it_uz16 < 0) st->it_uz16 = k;
        for (int64_t i = 0; i < n; ++i) p[(size_t)i] = round_store(p[(size_t)i], uz);   // R9
      }
    } else if (pol->amp) {
      // Lagged variant (reading R17): lines 3 and 4 of Alg 4.1 for iteration k are evaluated with
      // ||r_{k-1}|| instead of ||r_k|| ("other scaling factors can be used"; Thm 3.2), i.e. the
      // decisions D(k) = (u_r, u_z, omega) of iteration k were taken one iteration earlier, from hist[0..k-1]
      // (k = 0: from hist[0]).  r_k was therefore already stored in u_r,k by line 16 of iteration k-1.
      auto decide = [&](int32_t t) {  // D(t+1) from hist[0..t]
        const double e = orc_eta(pol, hist.data(), t);
        ur_n = (ur == ORC_FP32 || e <= pol->eta_safety * tol * nb) ? ORC_FP32 : ORC_FP64;
        const int32_t want = orc_select_uz(pol, hist[(size_t)t] / nb);
        uz_n = want > uz ? want : uz;
        omega_n = scale_factor(pol, hist[(size_t)t], n);
        return e;
      };
      if (k == 0) decide(0);
      if (ur_n != ur) {
        ur = ur_n; st->it_ur32 = k;
        for (int64_t i = 0; i < n; ++i) r[(size_t)i] = orc_round_fp32(r[(size_t)i]);  // only changes r at k = 0
        if (vals32.empty()) { vals32.resize((size_t)nnz); for (int64_t e = 0; e < nnz; ++e) vals32[(size_t)e] = (float)vals[e]; }
      }
      if (uz_n > uz) {
        uz = uz_n;
        if (uz >= ORC_FP32 && st->it_uz32 < 0) st->it_uz32 = k;
        if (uz == ORC_FP16 && st->it_uz16 < 0) st->it_uz16 = k;
        for (int64_t i = 0; i < n; ++i) p[(size_t)i] = round_store(p[(size_t)i], uz);   // R9
      }
      omega_lag = omega_n;
      eta = decide(k);  // D(k+1)
    }
    // O2: y = omega r, z = M^-1 y  (Alg 4.1 lines 4-5; Alg 3.2 line 3; fused)
    const double omega = !pol->amp ? 1.0 : (lag ? omega_lag : scale_factor(pol, delta, n));
    const bool strict = pol->strict_rounding && pol->amp;
    const double* dv = (uz == ORC_FP64 || strict) ? dinv.data() : dinv32.data();            // R6
    int64_t counts[3] = {0, 0, 0};
    if (cheb)   // M^-1 = s sweeps of Chebyshev-accelerated Jacobi (reading R18); needs s - 1 mat-vecs in u_r
      orc_cheb_apply(n, rowptr, colidx, vals, vals32.data(), r.data(), omega, dv, pol->cheb_degree, cheb_lmin, cheb_lmax, uz, ur,
                     z.data(), cheb_d.data(), cheb_w.data());
    else
      orc_step_z(n, r.data(), omega, dv, ur, uz, strict ? 1 : 0, z.data(), counts);
    // O3: rho = r^T z (Alg 4.1 line 6), FP64, with the stored z
    const double rho = dot_fp64(n, r.data(), z.data());
    // O4: beta (lines 7-9)
    const double beta = (k > 0) ? rho / rho_prev : 0.0;
    // O5: p = z + beta p (line 10), one rounding to u_z
    orc_step_p(n, beta, z.data(), uz, p.data(), counts);
    if (uz == ORC_FP16) { st->fp16_inf += counts[0]; st->fp16_flushed += counts[1]; st->fp16_subnormal += counts[2]; st->fp16_stored += 2 * n; }
    // O6: q = A p in u_r (line 11)
    if (ur == ORC_FP64) orc_spmv_fp64(n, rowptr, colidx, vals, p.data(), q.data());
    else orc_spmv_fp32(n, rowptr, colidx, vals32.data(), p.data(), q.data(), pol->accumulate64);
    // O7: gamma = q^T p (line 13)
    const double gamma = dot_fp64(n, q.data(), p.data());
    if (!(gamma > 0.0) || !(rho > 0.0) || !std::isfinite(gamma) || !std::isfinite(rho)) { status = -2; break; }
    // O8: alpha (line 14)
    const double alpha = rho / gamma;
    // O9: x += alpha p in FP64 (line 15); O10: r -= alpha q in u_r (line 16), one rounding
    orc_step_xr(n, alpha, p.data(), q.data(), lag ? ur_n : ur, x, r.data());
    // O11: delta_{k+1} = ||r_{k+1}|| (line 17)
    const double delta_k = delta;
    delta = std::sqrt(dot_fp64(n, r.data(), r.data()));
    hist[(size_t)k + 1] = delta;
    rho_prev = rho;
    if (trace) {
      const double scal[10] = {rho, beta, gamma, alpha, delta_k, delta, omega, eta, (double)ur, (double)uz};
      trace(k, x, r.data(), z.data(), p.data(), q.data(), scal, user);
    }
    if (!std::isfinite(delta)) { status = -2; ++k; break; }
    // O12: stopping test (lines 18-20)
    if (delta <= pol->stop_safety * tol * nb && !pol->no_stop) { status = 0; ++k; break; }
  }
  st->status = status;
  st->iters = k;
  st->relres_updated = (nb > 0.0) ? delta / nb : 0.0;
  orc_spmv_fp64(n, rowptr, colidx, vals, x, q.data());
  for (int64_t i = 0; i < n; ++i) q[(size_t)i] = b[i] - q[(size_t)i];
  st->relres_true = (nb > 0.0) ? std::sqrt(dot_fp64(n, q.data(), q.data())) / nb : 0.0;
  if (hist_out) for (int32_t t = 0; t <= k && t <= maxit; ++t) hist_out[t] = hist[(size_t)t];
  return status;
}

int32_t orc_sizeof_policy() { return (int32_t)sizeof(orc_policy); }
int32_t orc_sizeof_stats() { return (int32_t)sizeof(orc_stats); }

}  // extern "C"
