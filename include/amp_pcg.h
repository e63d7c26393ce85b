/* ===========================================================================================
 * amp_pcg.h — C ABI of the B200-native AMP-PCG iteration loop.
 *
 * Method: Guo, de Sturler, Warburton, "An adaptive mixed-precision and dynamically scaled
 * preconditioned conjugate gradient algorithm", arXiv 2505.04155 (PAPER.md in this task):
 *   problem statement  SPD  A x = b, preconditioner M, x0, relative-residual tol, maxit
 *   PCG                Algorithm 3.1
 *   dynamic scaling    Algorithm 3.2, Theorem 3.2
 *   AMP-PCG(u0)        Algorithm 4.1
 *   precision selector eq. (4.1)
 *   indicators eta_k   eq. (4.9)+(4.10) "delay", eq. (4.11) "linear"
 *   defaults           d=10, C=1, ell=5, tau_zs=1e-4, tau_zh=1e-6
 *
 * Every step of the loop (SpMV, Jacobi apply + scaling + cast + (r,z), p update, x/r update +
 * ||r|| + precision bookkeeping) runs in hand-written sm_100a CUDA kernels inside this
 * library; convergence, precision switches and breakdown are decided from device-side scalars
 * and the loop is one CUDA-graph launch (WHILE conditional node) or one persistent
 * cooperative kernel, so the host is not synchronised until the solve has ended.
 * There is no CPU fallback: every entry point fails with AMP_ERR_CUDA if no device is usable.
 *
 * Pointer convention: unless a parameter is marked HOST, every pointer is a DEVICE pointer
 * (e.g. torch-allocated), 16-byte aligned, valid on the device current at amp_pcg_create().
 * All functions are thread-compatible (one handle = one thread at a time), not thread-safe.
 * =========================================================================================== */
#ifndef AMP_PCG_H_
#define AMP_PCG_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct amp_pcg amp_pcg_t; /* opaque solver handle */

/* preconditioner M: the paper uses M = I for its small examples and Jacobi for
 * the timed GPU example */
enum {
  AMP_PRECOND_NONE = 0,
  AMP_PRECOND_JACOBI = 1,
  /* s sweeps of Chebyshev-accelerated Jacobi, the paper's smoother ("second-order Chebyshev-accelerated
   * Jacobi smoother [35]"; stronger preconditioning is what the paper asks for when the spectrum is hard, :584), used as
   * M^-1 of the loop (reading R18): with D = diag(A), [lmin, lmax] bounds of the spectrum of D^-1 A,
   * theta = (lmax+lmin)/2, dc = (lmax-lmin)/2, sigma = theta/dc, rho_0 = 1/sigma and y = omega r (Alg 4.1 line 4):
   *   d = D^-1 y / theta, z = d;   then for i = 1..s-1:  rho_i = 1/(2 sigma - rho_{i-1}),
   *   d = rho_i rho_{i-1} d + (2 rho_i/dc) D^-1 (y - A z),  z = z + d.
   * d, z are stored in u_z (one rounding per update), A z is computed and stored in u_r (like q), scalars FP64.
   * Costs s - 1 extra mat-vecs per iteration and divides the iteration count by about s.  Needs amp_pcg_create_ex
   * (cheb_degree, bounds); not available with AMP_SCALE_LAGGED or AMP_LOOP_PERSISTENT. */
  AMP_PRECOND_CHEBJACOBI = 2
};
/* column-index form of the SELL-32 repack.  AUTO takes the most compact form the matrix
 * allows; the other two force a more general form on the same matrix (testing / tuning) */
enum {
  AMP_INDEX_AUTO = 0,     /* diagonal-aligned slices where possible, else 16-bit offsets if they fit, else 32-bit */
  AMP_INDEX_NO_ALIGN = 1, /* never diagonal-aligned: 16-bit offsets if they fit, else 32-bit */
  AMP_INDEX_FORCE32 = 2   /* never diagonal-aligned, always 32-bit column indices */
};
/* which SpMV kernel the loop uses in the u_r = FP32 phase (execution choice; same arithmetic, same bits) */
enum {
  AMP_SPMV_AUTO = 0,      /* bulk-copy pipelined kernel when the matrix is eligible (every slice diagonal-aligned,
                             natural row order, no long rows), else the direct kernel */
  AMP_SPMV_DIRECT = 1,    /* every lane streams its row with 128-bit loads (round-1 kernel) */
  AMP_SPMV_PIPELINED = 2  /* value stream staged through shared memory by cp.async.bulk + mbarrier ring */
};
/* which vector kernels (steps a2, a3, a5) the loop uses (execution choice; same arithmetic, same bits) */
enum {
  AMP_VEC_AUTO = 0,       /* from 4 M rows on the z and p updates are staged, the x/r update stays direct; below: all direct */
  AMP_VEC_DIRECT = 1,     /* every thread loads its chunks of the vectors from global memory */
  AMP_VEC_STAGED = 2      /* persistent blocks; the input vectors are streamed into a shared-memory ring by cp.async.bulk */
};
/* whether the three vector steps between two mat-vecs run as ONE cooperative kernel with two grid barriers
 * (execution choice; the vectors are bit-identical, the inner products are added in another fixed order) */
enum { AMP_FUSE_AUTO = 0 /* on wherever it can run: Jacobi / no preconditioner, not a block row of a sharded system */,
       AMP_FUSE_OFF = 1, AMP_FUSE_ON = 2 };
/* storage / working precisions u_z, u_r */
enum { AMP_FP64 = 0, AMP_FP32 = 1, AMP_FP16 = 2 };
/* indicator used by the u_r switch */
enum { AMP_ETA_DELAY = 0 /* (4.9)+(4.10) */, AMP_ETA_LINEAR = 1 /* (4.11) */, AMP_ETA_NEVER = 2 /* u_r stays FP64 */ };
/* scaling factor omega_k of Algorithm 3.2 ("other scaling factors can be used") */
enum {
  AMP_SCALE_NORM2 = 0, /* omega = 1/||r_k||                 (Algorithm 4.1 line 4) — default */
  AMP_SCALE_RMS = 1,   /* omega = sqrt(n)/||r_k||            */
  AMP_SCALE_POW2 = 2,  /* omega = 2^round(log2(1/||r_k||))   (exact scaling) */
  AMP_SCALE_NONE = 3,  /* omega = 1                          (diagnostic: naive low precision) */
  AMP_SCALE_LAGGED = 4 /* omega_k = 1/||r_{k-1}|| (omega_0 = 1/||r_0||) AND the selector (4.1)/(4.10) of iteration k
                          evaluated with the norms up to ||r_{k-1}||: every decision of iteration k is known one
                          iteration early, so z_{k+1} and rho_{k+1} are produced in the pass that updates x and r —
                          three kernels and reductions per iteration instead of four.  Same iterates in exact
                          arithmetic (Theorem 3.2); switch iterations move by +1. */
};
/* how the iteration loop is driven (execution choice; does not change the arithmetic) */
enum {
  AMP_LOOP_AUTO = 0,       /* persistent kernel for small systems (n <= 2^20 rows), else graph */
  AMP_LOOP_STREAM = 1,     /* plain stream launches in batches; host polls a device flag between batches */
  AMP_LOOP_GRAPH = 2,      /* one CUDA graph launch: WHILE conditional node around the 4 kernels */
  AMP_LOOP_PERSISTENT = 3  /* one cooperative kernel, grid barriers between the phases */
};

/* return / status codes */
enum {
  AMP_OK = 0,             /* converged: ||r_k|| <= stop_safety * tol * ||b||  (Alg 4.1 line 18) */
  AMP_MAXIT = 1,          /* maxit reached; x holds the last iterate, stats are valid */
  AMP_ERR_INVALID = -1,   /* invalid argument (see each function) */
  AMP_ERR_BREAKDOWN = -2, /* gamma <= 0, rho <= 0 or a non-finite scalar: A not SPD, or FP16 overflow */
  AMP_ERR_CUDA = -3,      /* CUDA error or no usable device; see amp_pcg_last_error() */
  AMP_ERR_NOMEM = -4      /* device allocation failed */
};

/* Policy of one solve.  A NULL policy means AMP-PCG(FP64) with the paper's defaults and
 * the delay indicator.  Use amp_policy_default() to fill a struct and then edit fields. */
typedef struct {
  int32_t amp;        /* 0: PCG(FP64), Algorithm 3.1 exactly (no scaling, no switching); 1: Algorithm 4.1 */
  int32_t u0;         /* AMP_FP64 -> AMP-PCG(FP64): z,p start FP64 and step down by (4.1);
                         AMP_FP16 -> AMP-PCG(FP16): z,p in FP16 throughout */
  int32_t eta_rule;   /* AMP_ETA_* */
  int32_t d;          /* delay of (4.9), default 10 (1 <= d <= 64) */
  int32_t ell;        /* window of (4.11), default 5 (1 <= ell <= 64) */
  int32_t scale_mode; /* AMP_SCALE_* */
  int32_t no_stop;    /* 1: ignore the stopping test, run maxit iterations (attainable-accuracy runs) */
  int32_t x0_zero;    /* 1: caller promises x0 = 0; x is zero-filled and r0 = b without a mat-vec */
  int32_t true_residual; /* 1: after the loop compute ||b - A x||/||b|| in FP64 (one extra FP64 SpMV, not in solve_ms) */
  int32_t loop_mode;  /* AMP_LOOP_* */
  int32_t profile_kernels; /* 1 (AMP_LOOP_STREAM only): bracket every loop kernel with CUDA events on the solve stream;
                              read the per-kernel, per-phase sums with amp_pcg_kernel_times().  Plain launches (no
                              programmatic overlap) so that each duration belongs to one kernel */
  int32_t reserved0;  /* 0 */
  double C;           /* constant of Assumption 4.1, default 1 */
  double tau_zs;      /* u_z: FP64 -> FP32 when ||r_k||/||b|| < tau_zs, default 1e-4 (5.1) */
  double tau_zh;      /* u_z: FP32 -> FP16 when ||r_k||/||b|| < tau_zh, default 1e-6 (5.1); 0 = never FP16 */
  double eps32;       /* unit roundoff of FP32 in eta_k; 0 means 2^-24 */
  double eta_safety;  /* switch u_r when eta_k <= eta_safety * tol * ||b||; 0 means 1 (paper, (4.10)) */
  double stop_safety; /* stop when ||r_k|| <= stop_safety * tol * ||b||; 0 means 1 (paper). eta_safety = theta,
                         stop_safety = 1 - theta enforces (3.10): ||zeta|| + ||r|| <= tol ||b|| */
} amp_policy_t;

/* Result of one solve. */
typedef struct {
  int32_t status;           /* same value amp_pcg_solve returns */
  int32_t iters;            /* iterations performed (k+1 of the last executed loop index) */
  int32_t it_ur32;          /* iteration index k at which u_r became FP32, -1 if never */
  int32_t it_uz32;          /* iteration index k at which u_z became FP32 (or lower), -1 if never */
  int32_t it_uz16;          /* iteration index k at which u_z became FP16, -1 if never */
  int32_t loop_mode;        /* AMP_LOOP_* actually used */
  double bnorm;             /* ||b||_2 */
  double relres_updated;    /* ||r_m|| / ||b|| of the recursively updated residual */
  double relres_true;       /* ||b - A x_m|| / ||b|| in FP64 if policy.true_residual, else -1 */
  double solve_ms;          /* device time of setup + loop (CUDA events on the solve stream) */
  double algorithmic_bytes; /* compulsory bytes moved by the loop: sum over iterations of
                               amp_pcg_iteration_bytes() for the precisions in use at each iteration */
  uint64_t fp16_subnormal;  /* FP16 stores of z,p that were subnormal / flushed to 0 / overflowed; */
  uint64_t fp16_flushed;    /* filled only when the library is built with -DAMP_COUNT_FP16, else 0 */
  uint64_t fp16_inf;
} amp_stats_t;

/* Fill *p with the paper's defaults: amp=1, u0=FP64, eta_rule=DELAY, d=10, ell=5, C=1,
 * tau=(1e-4,1e-6), eps32=2^-24, safeties 1, scale NORM2, x0_zero=0, true_residual=0, loop AUTO, profile_kernels=0. */
void amp_policy_default(amp_policy_t *p);

/* Build a solver for the SPD matrix A given in CSR (CSR per BASELINE.json).
 *   n, nnz      rows (= columns) and stored entries; 0 < n, 0 <= nnz < 2^31
 *   rowptr      int32[n+1], rowptr[0] = 0, non-decreasing, rowptr[n] = nnz
 *   colidx      int32[nnz], 0 <= colidx < n (any order within a row; duplicates are summed by the mat-vec)
 *   vals        float64[nnz]
 *   precond     AMP_PRECOND_NONE (M = I) or AMP_PRECOND_JACOBI (M = diag(A); every row needs a
 *               stored, positive diagonal entry)
 * rowptr/colidx/vals are BORROWED: they must stay valid and unchanged until amp_pcg_destroy()
 * (rows longer than max(256, 8 nnz/n) entries are read from them by every mat-vec).
 * The handle owns everything derived (SELL-32 repack of A: indices, FP64 values and the FP32 value
 * copy; 1/diag in FP64 and FP32; work vectors in FP64/FP32/FP16; device state; captured graph).
 * Symmetry is not verified.
 * Returns NULL on failure; amp_pcg_last_error() says why (invalid structure, CUDA, memory). */
amp_pcg_t *amp_pcg_create(int64_t n, int64_t nnz, const int32_t *rowptr, const int32_t *colidx,
                          const double *vals, int precond);

/* Create-time options.  amp_create_opts_default() fills the defaults; amp_pcg_create(..., precond) is
 * amp_pcg_create_ex() with the defaults and the given preconditioner. */
typedef struct {
  int32_t struct_bytes;   /* sizeof(amp_create_opts_t) as the caller compiled it (ABI growth check) */
  int32_t precond;        /* AMP_PRECOND_* */
  int32_t index_format;   /* AMP_INDEX_*, default AUTO */
  int32_t spmv_kernel;    /* AMP_SPMV_*, default AUTO */
  int32_t spmv_grid_mult; /* upper bound on resident SpMV blocks per SM for the direct kernel's grid; 0 = automatic */
  int32_t pdl;            /* 1 (default): launch the loop kernels as programmatic dependents (griddepcontrol), 0: plain */
  int32_t cheb_degree;    /* AMP_PRECOND_CHEBJACOBI: sweeps s, 1 <= s <= 16; default 2 (the paper's "second-order") */
  int32_t reserved0;      /* 0 */
  double cheb_lmin;       /* bounds of the spectrum of D^-1 A the polynomial is built for; cheb_lmax = 0 (default): */
  double cheb_lmax;       /*   lmax = max_i sum_j |a_ij| / a_ii (Gershgorin), lmin = lmax / 30, computed in create() */
  void *stream;           /* cudaStream_t the create() kernels run on and the handle starts with (NULL = legacy
                             default stream); the caller's CSR arrays must be complete in this stream's order */
  int64_t halo_lo;        /* row-sharded solve (see "row-sharded solve" below): the matrix is one block row of a larger */
  int64_t halo_hi;        /*   system, n rows by halo_lo + n + halo_hi columns; column index halo_lo + i is the diagonal of
                               row i, columns below halo_lo / from halo_lo + n on are the neighbour ranks' entries of p
                               (filled by the halo exchange).  Both 0 (default): an ordinary square matrix */
  int32_t vec_kernel;     /* AMP_VEC_*, default AUTO */
  int32_t fuse_vec;       /* AMP_FUSE_*, default AUTO */
} amp_create_opts_t;
void amp_create_opts_default(amp_create_opts_t *o);
amp_pcg_t *amp_pcg_create_ex(int64_t n, int64_t nnz, const int32_t *rowptr, const int32_t *colidx,
                             const double *vals, const amp_create_opts_t *opts);

/* Solve A x = b to ||r_k|| <= tol ||b|| (Algorithm 3.1 or 4.1 by policy).
 *   b        float64[n], read-only
 *   x        float64[n], in: initial guess x0, out: x_m (FP64 always)
 *   tol      > 0 relative residual tolerance;  maxit >= 1 (<= 2^24)
 *   policy   HOST pointer or NULL;  stats  HOST pointer or NULL
 * ||b|| = 0 gives x = 0, status AMP_OK, 0 iterations.  If x0 already satisfies the stopping test,
 * 0 iterations are made.  Returns the status (also in stats->status).  The call synchronises the
 * stream once, after the loop has ended, to read the result scalars. */
int amp_pcg_solve(amp_pcg_t *h, const double *b, double *x, double tol, int32_t maxit,
                  const amp_policy_t *policy, amp_stats_t *stats);

/* Same as amp_pcg_solve but b and x are HOST buffers (pinned memory recommended): b and x0 are
 * copied to the device, the solve runs, x is copied back; all three inside the call. */
int amp_pcg_solve_host(amp_pcg_t *h, const double *b_host, double *x_host, double tol, int32_t maxit,
                       const amp_policy_t *policy, amp_stats_t *stats);

/* q = A p with the loop's own SpMV kernel (step a4, Alg 4.1 line 11).
 *   mat_prec  AMP_FP64 (original values, FP64 accumulation) or AMP_FP32 (FP32 value copy, FP32 arithmetic)
 *   vec_prec  storage type of p: AMP_FP64 double[n], AMP_FP32 float[n], AMP_FP16 __half[n rounded up to 8]
 *   q         mat_prec type: double[n] or float[n]
 * Returns AMP_OK, AMP_ERR_INVALID or AMP_ERR_CUDA.  Asynchronous on the handle's stream. */
int amp_spmv(amp_pcg_t *h, int mat_prec, int vec_prec, const void *p, void *q);

/* Copy the residual-norm history ||r_t||, t = 0..iters of the last solve into HOST out[0..count);
 * returns the number of values written (<= iters+1), or a negative error code. */
int32_t amp_pcg_residual_history(amp_pcg_t *h, double *out_host, int32_t count);

/* A-posteriori attainable-accuracy indicator of the last solve, eq. (4.7):
 *   out[k] = eta_hat_m(k) = sum_{t=0..k} eps64 ((3+C)||r_{t-1}|| + (2+C)||r_t||) + sum_{t=k..m} eps32 ((3+C)||r_{t-1}|| + (2+C)||r_t||)
 * for k = 0..min(count, m+1)-1, m = iterations of the last solve, ||r_{-1}|| := ||r_0||, eps64 = 2^-53, eps32 = 0 -> 2^-24:
 * the accuracy the run could have attained had u_r been switched to FP32 at iteration k (the dotted curves of the
 * paper's Fig. 3 and 8).  Host post-processing of the stored history (HOST out); returns the number of values
 * written or a negative error code. */
int32_t amp_pcg_eta_posteriori(amp_pcg_t *h, double C, double eps32, double *out_host, int32_t count);

/* Run all work of this handle on the given cudaStream_t (NULL = legacy default stream). */
int amp_pcg_set_stream(amp_pcg_t *h, void *cuda_stream);

/* Number of kernel launches (graph launches count their kernel nodes once per loop iteration)
 * made by the last solve / spmv call of this handle: bench.py's gpu_launches. */
int64_t amp_pcg_last_launch_count(const amp_pcg_t *h);

/* Release the handle and everything it owns (not the borrowed CSR arrays). NULL is ignored. */
void amp_pcg_destroy(amp_pcg_t *h);

/* Thread-local message of the last failure in this library ("" if none). */
const char *amp_pcg_last_error(void);

/* Per-row bytes of one iteration for m = nnz/n and the given (u_z, u_r) in the paper-style CSR
 * reference accounting (Table 2 :524-537 for the vector kernels; CSR values + 4-byte
 * column index + 4-byte row pointer for the mat-vec; every vector read/written once per pass).
 * A format-independent yardstick; what THIS library moves is amp_pcg_iteration_bytes(). */
double amp_pcg_bytes_per_row(double m, int uz, int ur);

/* Compulsory bytes ONE mat-vec q = A p of this handle moves with the matrix format it built
 * (SELL-32 repack): stored values (zero padding included) in mat_prec, the index
 * data actually read (slice table, per-entry 32- or 16-bit columns of general slices, 4 bytes per
 * 32 entries for diagonal-aligned slices, row order if rows were sorted), p read once in vec_prec,
 * q written once in mat_prec.  The roofline numerator of bench.py for the SpMV kernel. */
double amp_pcg_spmv_bytes(const amp_pcg_t *h, int mat_prec, int vec_prec);

/* Compulsory bytes of one whole iteration in phase (u_z, u_r): amp_pcg_spmv_bytes(h, u_r, u_z) plus
 * the three vector kernels (z: r, 1/diag -> z; p: z, p -> p; x/r: x, p, q, r -> x, r).  In phase (FP64, FP32) the p
 * update also writes RN32(p) (4 B per row) and the mat-vec gathers that copy instead of converting every gathered entry.
 * amp_stats_t.algorithmic_bytes is the sum of this over the iterations of a solve. */
double amp_pcg_iteration_bytes(const amp_pcg_t *h, int uz, int ur);

/* What create() built for this matrix: for tests, tuning and reports. */
typedef struct {
  int64_t slices;          /* SELL-32 slices */
  int64_t aligned_slices;  /* diagonal-aligned slices (no per-entry column index) */
  int64_t uniform_slices;  /* of those: slices of the uniform stencil (columns = row + a constant of the handle) */
  int64_t stored_entries;  /* entries of the repack, zero padding included */
  int64_t long_rows;       /* rows kept out of the slices (summed from the CSR arrays) */
  int64_t guard;           /* zero guard band (entries) on each side of p and z */
  int32_t index_bits;      /* 0: every slice aligned; 16 / 32: width of the per-entry column data of the general slices */
  int32_t rows_sorted;     /* 1: rows sorted by length inside windows of 1024 */
  int32_t spmv_pipelined;  /* 1: the u_r = FP32 phases run the bulk-copy pipelined mat-vec */
  int32_t vec_staged;      /* bit 0: z and p updates, bit 1: x/r update run the bulk-copy staged kernels */
  int32_t uniform_width;   /* entries per row of the uniform stencil, 0 if none */
  int32_t reserved0;
} amp_format_info_t;
int amp_pcg_format_info(const amp_pcg_t *h, amp_format_info_t *out_host);

/* ---- measurement: per-kernel device times of the last solve made with policy.profile_kernels = 1 ---------- */
enum { AMP_K_Z = 0, AMP_K_P = 1, AMP_K_SPMV = 2, AMP_K_XR = 3, AMP_K_XRZ = 4,
       AMP_K_CHEB0 = 5 /* first Chebyshev sweep */, AMP_K_CHEBSTEP = 6 /* further sweeps */,
       AMP_K_VEC_FUSED = 7 /* a5 of iteration k + a2, a3 of iteration k + 1 in one kernel (AMP_FUSE_ON) */, AMP_K_COUNT = 8 };
typedef struct {
  int32_t kernel;          /* AMP_K_*: step a2, a3, a4, a5 of SURVEY.md section 8(a) (XRZ: a5 + a2 of the lagged variant;
                              with AMP_PRECOND_CHEBJACOBI step a2 is CHEB0 + (s-1) x (SPMV + CHEBSTEP), all mat-vecs under SPMV) */
  int32_t uz, ur;          /* precision phase (u_z, u_r) of the iterations summed here */
  int32_t launches;        /* launches of this kernel in this phase */
  double total_ms;         /* sum over those launches of (event after - event before) on the solve stream */
  double bytes_per_launch; /* compulsory bytes of one launch: amp_pcg_spmv_bytes() for AMP_K_SPMV, n times the
                              per-row figures of DESIGN.md section 5 for the vector kernels */
} amp_kernel_time_t;
/* Writes up to cap records (one per kernel and phase that occurred) to HOST out; returns the count, 0 if the last
 * solve was not profiled, or a negative error code. */
int32_t amp_pcg_kernel_times(amp_pcg_t *h, amp_kernel_time_t *out_host, int32_t cap);

/* ---- row-sharded solve over several GPUs ------------------------------------
 * The paper runs on one GPU; how Algorithm 4.1 shards follows from its data flow: the rows of A, and
 * with them r, z, p, q, x, are split into contiguous blocks, one per rank.  Per iteration the only data that crosses ranks
 * are  (1) the entries of p the local block row touches outside its own rows (the halo), needed by q = A p (line 11) —
 * exchanged in the precision the mat-vec gathers (u_z; RN32(p) while u_z = FP64 and u_r = FP32), so AMP shrinks it up
 * to 4x;  (2) the three inner products rho = r^T z, gamma = q^T p, ||r||^2 (lines 6, 13, 17): every rank publishes its
 * partial sum to every rank and each adds all partials in rank order, so all ranks hold bit-identical scalars and take
 * the same decisions (stop, switches, breakdown) without any broadcast.
 * Both exchanges are done by the loop kernels themselves over peer-mapped device memory (NVLink / NVSwitch stores, or
 * plain stores when the ranks share a device): the p update writes the boundary entries straight into the neighbours'
 * halo bands and then raises their flags, the mat-vec waits for its two flags, the reducing kernels post their partial
 * sums into every rank's mailbox and a one-warp kernel per reduction point adds them and runs the scalar step.  No NCCL
 * call, no host on the data path; the host launches the same graph / stream loop as in the single-GPU solve.
 *
 * Partition: contiguous row blocks whose boundaries are multiples of 32 rows (whole SELL-32 slices), balanced by stored
 * entries.  A rank's halo must lie inside its two neighbour ranks (banded coupling: stencils, c5's 50 000-row band).
 * All pointers of amp_shard_plan / amp_shard_extract are HOST pointers; they do not touch the device. */
typedef struct {
  int64_t row0, row1;       /* this rank owns the global rows [row0, row1) */
  int64_t halo_lo, halo_hi; /* entries of p needed below row0 / from row1 on (rounded up to multiples of 8) */
  int64_t nnz;              /* stored entries of the block row */
} amp_shard_t;
/* Plan the block-row partition of an n x n CSR pattern over `world` ranks (1 <= world <= 16) into out[world].
 * Returns AMP_OK, or AMP_ERR_INVALID (bad arguments; fewer than 32 rows per rank; a halo reaching past the neighbour). */
int amp_shard_plan(int64_t n, const int32_t *rowptr, const int32_t *colidx, int32_t world, amp_shard_t *out);
/* Extract the block row `s` as a CSR of s->row1 - s->row0 rows whose column indices are shifted to the extended vector
 * [halo_lo | owned | halo_hi] (global column j becomes j - row0 + halo_lo) — the arrays amp_pcg_create_ex takes together
 * with opts.halo_lo / halo_hi.  rowptr_out: int32[rows + 1]; colidx_out / vals_out: s->nnz entries, CSR order kept. */
int amp_shard_extract(int64_t n, const int32_t *rowptr, const int32_t *colidx, const double *vals, const amp_shard_t *s,
                      int32_t *rowptr_out, int32_t *colidx_out, double *vals_out);

/* Wiring.  Every rank creates its handle with amp_pcg_create_ex (opts.halo_lo / halo_hi from the plan), then either
 *  (a) one process drives all ranks (handles on one device — the testable emulation — or on peer-accessible devices):
 *      amp_pcg_shard_attach_local(handles, world), handles[r] = rank r; or
 *  (b) one process per GPU: every rank fills an amp_shard_export_t (amp_pcg_shard_export), the blobs are all-gathered by
 *      the caller (torch.distributed: plumbing), and every rank calls amp_pcg_shard_attach(h, rank, world, blobs), which
 *      opens its neighbours' buffers with CUDA IPC.
 * Handles of one group must agree in preconditioner (NONE / JACOBI) and be created from one amp_shard_plan. */
#define AMP_SHARD_MAX_WORLD 16
typedef struct {
  int64_t n, halo_lo, halo_hi, guard; /* geometry of this rank's extended p vectors */
  unsigned char mem[4][64];           /* cudaIpcMemHandle_t of: the exchange block (mailboxes + flags), p64, p32, p16 */
  int64_t off[4];                     /* byte offset of each object inside its allocation */
} amp_shard_export_t;
int amp_pcg_shard_export(amp_pcg_t *h, amp_shard_export_t *out_host);
int amp_pcg_shard_attach(amp_pcg_t *h, int32_t rank, int32_t world, const amp_shard_export_t *all_host);
int amp_pcg_shard_attach_local(amp_pcg_t *const *handles, int32_t world);

/* Solve the sharded system: handles[0..nlocal) are the ranks this process drives (nlocal = world after
 * amp_pcg_shard_attach_local, 1 after amp_pcg_shard_attach), b[i] / x[i] their DEVICE block rows of b and x (x: x0 in,
 * x_m out), stats[i] HOST (may be NULL).  Same policy semantics as amp_pcg_solve; every rank must pass the same tol,
 * maxit and policy.  Not available with AMP_PRECOND_CHEBJACOBI and AMP_LOOP_PERSISTENT; AMP_LOOP_AUTO = graph when
 * nlocal = 1, else stream (the ranks of one process are launched in lock step).  In mode (b) no rank may start a
 * solve before every rank has returned from the previous one (a host barrier between solves).
 * A rank that waits longer than ~10 s for a peer gives up with AMP_ERR_CUDA.  Returns the common status. */
int amp_pcg_solve_sharded(amp_pcg_t *const *handles, int32_t nlocal, const double *const *b, double *const *x, double tol,
                          int32_t maxit, const amp_policy_t *policy, amp_stats_t *stats);
/* q = A p on the sharded system (mat_prec / vec_prec as amp_spmv; p[i]: this rank's n entries, q[i]: its rows): halo
 * exchange of p, then the loop's mat-vec.  For tests and for callers that need the operator alone. */
int amp_spmv_sharded(amp_pcg_t *const *handles, int32_t nlocal, int mat_prec, int vec_prec, const void *const *p, void *const *q);

/* ---- diagnostic entry points (parity tests; not on the hot path) ------------------------------------------
 * Run ONE step of the loop with caller-given scalars and precisions through the SAME __global__ kernel, grid and
 * reduction the stream / graph loop launches, on the handle's own work vectors, so that a test can compare z, p, r,
 * x element by element with the formulas of Algorithm 4.1.
 * Work vectors: which = AMP_VEC_*; prec = storage precision of the copy addressed (r, q: FP64/FP32; z, p:
 * FP64/FP32/FP16; 1/diag: FP64/FP32).  src/dst are DEVICE arrays of n elements of that storage type; the library's
 * zero padding to a multiple of 8 is kept. */
enum { AMP_VEC_R = 0, AMP_VEC_Q = 1, AMP_VEC_Z = 2, AMP_VEC_P = 3, AMP_VEC_DINV = 4 /* get only */,
       AMP_VEC_D = 5 /* Chebyshev direction d (AMP_PRECOND_CHEBJACOBI handles only), stored like z */ };
int amp_pcg_debug_set_vector(amp_pcg_t *h, int which, int prec, const void *src);
int amp_pcg_debug_get_vector(amp_pcg_t *h, int which, int prec, void *dst);
enum {
  AMP_STEP_Z = 0,    /* a2 (+a6): z = RN_uz((r omega) dinv), rho = r^T z; r <- RN_ur(r) first if rs != ur   (lines 4-6) */
  AMP_STEP_P = 1,    /* a3 (+a6): p = RN_uz(fma(beta, RN_uz(p), z)); first != 0: p = z                      (line 10) */
  AMP_STEP_SPMV = 2, /* a4: q = A p in u_r, gamma = q^T p                                                   (lines 11-13) */
  AMP_STEP_XR = 3,   /* a5: x += alpha p (FP64), r = RN_ur(fma(-alpha, q, r)), delta = ||r||               (lines 15-17) */
  AMP_STEP_XRZ = 4,  /* lagged a5 + a2: x, r = RN_ur_n(..), z = RN_uz_n((r omega_n) dinv), ||r|| and r^T z */
  /* AMP_PRECOND_CHEBJACOBI handles only: */
  AMP_STEP_CHEB0 = 5,    /* d = z = RN_uz(((r omega) dinv) / theta) (+a6 as AMP_STEP_Z); rho = r^T z if s = 1 */
  AMP_STEP_SPMV_Z = 6,   /* q = A z in u_r (the mat-vec inside M^-1; no reduction) */
  AMP_STEP_CHEBSTEP = 7  /* sweep i = `first` (1 <= i < s): d = RN_uz(fma(c1_i, d, c2_i ((r omega - q) dinv))), z = RN_uz(z + d);
                            rho = r^T z if i = s - 1 */
};
typedef struct {
  int32_t step;            /* AMP_STEP_* */
  int32_t rs, ur, uz;      /* precision r is stored in on entry; u_r and u_z of this iteration */
  int32_t ps;              /* precision p is stored in on entry (AMP_STEP_P) */
  int32_t ur_n, uz_n;      /* precisions of the next iteration (AMP_STEP_XRZ) */
  int32_t first;           /* AMP_STEP_P: iteration k = 0 (p_{-1} is not read); AMP_STEP_CHEBSTEP: sweep index i */
  double omega, beta, alpha, omega_n; /* scalars the step reads */
  double sum0, sum1;       /* out: the step's scalar(s) after its grid reduction: Z: rho = r^T z | SPMV: gamma = q^T p |
                              XR: delta = ||r||_2 | XRZ: delta = ||r||_2 and sum1 = r^T z */
} amp_debug_step_t;
/* x: DEVICE float64[n], read and written by AMP_STEP_XR / AMP_STEP_XRZ only (may be NULL otherwise).
 * Synchronises the stream.  Returns AMP_OK, AMP_ERR_INVALID or AMP_ERR_CUDA. */
int amp_pcg_debug_step(amp_pcg_t *h, amp_debug_step_t *io, double *x);

/* ---- step a5 without any device allocation ------------------------------------------------------------------------
 * x += alpha p,  r -= alpha q,  *delta_out = ||r||_2   (Algorithm 4.1 lines 15-17), all FP64, in one
 * kernel, for callers that can't let this library allocate: every other entry point works on a handle, and
 * amp_pcg_create() calls cudaMalloc.  That is no option for a process that gave the whole device memory to its own pool
 * at start-up (a later cudaMalloc fails there, or takes memory the pool's owner counted on), nor for a loop with a
 * latency bound (cudaMalloc and cudaFree may synchronise the device and have no time bound).  This call needs no handle
 * and makes no cudaMalloc, cudaFree or other allocating call: the scratch memory of its grid reduction is a static
 * device array of 131 328 bytes inside the library image, which every GPU that loads the library holds until exit.
 *   n          elements, 0 < n <= AMP_XR_STATIC_MAX_N (what the fixed array serves; beyond it: AMP_ERR_INVALID, nothing runs)
 *   alpha      step length (HOST value)
 *   p, q       float64[n] DEVICE, read-only, 16-byte aligned
 *   x, r       float64[n] DEVICE, updated in place, 16-byte aligned
 *   delta_out  float64[1] DEVICE: ||r||_2 after the update, written by the kernel (no host synchronisation)
 *   cuda_stream  cudaStream_t the work is queued on (NULL = legacy default stream); the call is asynchronous
 * The arrays must live on the device that is current at the call.  x and r come out bit-identical to the handle path's
 * FP64 x / r update (k_xr); the norm is added in another fixed order (agreement to n 2^-53 relative).
 * Sharing: all calls on a device use the one array, which keeps the previous call's contents; the call clears what has
 * to start at zero itself, in stream order.  Calls that can overlap on one GPU (different streams without an order
 * between them) race on the array: order them.
 * Set-up: the first call on each device looks up the array's device address (cudaGetSymbolAddress, once per device,
 * thread-safe); make that first call before beginning any stream capture.
 * Returns AMP_OK, AMP_ERR_INVALID (size, null or misaligned pointer) or AMP_ERR_CUDA; amp_pcg_last_error() says why. */
#define AMP_XR_STATIC_MAX_N 67108864
int amp_xr_update_static(int64_t n, double alpha, const double *p, const double *q, double *x, double *r,
                         double *delta_out, void *cuda_stream);

#ifdef __cplusplus
}
#endif
#endif /* AMP_PCG_H_ */
