// amp_pcg.cu — host side of the C ABI declared in include/amp_pcg.h: handle management,
// validation, the solve drivers (stream batches / CUDA-graph WHILE loop / persistent kernel)
// and result read-back.  All arithmetic of the method runs in the kernels of kernels.cuh.
#include "../../include/amp_pcg.h"

#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <string>
#include <vector>

#include "kernels.cuh"
#include "persistent.cuh"
#include "spmv_pipe.cuh"
#include "vec_fused.cuh"
#include "vec_pipe.cuh"

using namespace amp;

static thread_local std::string g_last_error;

static void set_error(const char* fmt, ...) {
  char buf[512];
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(buf, sizeof(buf), fmt, ap);
  va_end(ap);
  g_last_error = buf;
}
namespace amp {
void set_error_text(const char* msg) { g_last_error = msg; }  // for the library's other translation units (xr_static.cu)
}

#define CU_TRY(call, onfail)                                                                  \
  do {                                                                                        \
    cudaError_t e_ = (call);                                                                  \
    if (e_ != cudaSuccess) {                                                                  \
      set_error("%s failed: %s (%s:%d)", #call, cudaGetErrorString(e_), __FILE__, __LINE__);   \
      onfail;                                                                                 \
    }                                                                                         \
  } while (0)

struct amp_pcg {
  int64_t n = 0, nnz = 0, npad = 0;
  int precond = 0, device = 0, num_sms = 0;
  cudaStream_t stream = nullptr;
  Ctx ctx{};
  std::vector<void*> owned;     // device allocations released in destroy
  DevState* h_state = nullptr;  // pinned staging for the state block
  int* h_flag = nullptr;        // pinned: done flag polled by the stream loop
  double* hist = nullptr;
  int64_t hist_cap = 0;
  int vec_grid = 1, grid_z = 1, grid_p = 1, grid_p_sh = 1, grid_xr = 1, spmv_grid = 1, persist_grid = 0, persist_ok = 0;
  // graph loop
  cudaGraph_t graph = nullptr;
  cudaGraphExec_t graph_exec = nullptr;
  cudaGraphConditionalHandle cond{};
  // graph loop of the lagged variant (k_p, k_spmv, k_xrz)
  cudaGraph_t graph_lag = nullptr;
  cudaGraphExec_t graph_lag_exec = nullptr;
  cudaGraphConditionalHandle cond_lag{};
  int grid_xrz = 1;
  // host-buffer staging for amp_pcg_solve_host
  double* d_b_stage = nullptr;
  double* d_x_stage = nullptr;
  cudaEvent_t ev0 = nullptr, ev1 = nullptr;
  int64_t launches = 0;
  int pdl = 0;                // graph loop built with programmatic dependent launches
  int32_t last_iters = -1;
  double m_avg = 0.0;
  double idx_bytes_total = 0.0;  // bytes of index data one SpMV reads (slice table, bases, per-entry indices, row order)
  double long_bytes_idx = 0.0, long_entries = 0.0;  // long rows, read from the CSR arrays (4 B index per entry)
  int64_t sell_entries = 0;   // stored entries of the SELL-32 repack (padding included)
  int use_pipe = 0;           // the loop's SpMV is the bulk-copy pipelined kernel (spmv_pipe.cuh)
  int pipe_grid = 0;
  int64_t pipe_chunks = 0;
  int64_t guard = 0;          // zero guard band (elements) on both sides of the p (and z) vectors
  int cheb_s = 0;             // sweeps of the Chebyshev-Jacobi preconditioner (0: not in use)
  double cheb_lmin = 0.0, cheb_lmax = 0.0;
  int grid_cheb0 = 1, grid_cheb_step = 1;
  // per-kernel event profile of the last solve (policy.profile_kernels, stream loop)
  std::vector<cudaEvent_t> prof_events;  // pool, grown on demand
  size_t prof_used = 0;
  std::vector<int8_t> prof_kernel;       // kernel id of the launch that FOLLOWS event i (-1: end of an iteration)
  std::vector<int32_t> prof_iter;        // iteration index the launch belongs to
  std::vector<amp_kernel_time_t> prof_result;
  // row-sharded solve (block row of a larger system; include/amp_pcg.h "row-sharded solve")
  int64_t halo_lo = 0, halo_hi = 0;
  void* p_base[3] = {nullptr, nullptr, nullptr};  // allocations behind ctx.p64 / p32 / p16 (guard band included)
  char* xchg = nullptr;                  // exchange block: mailbox [kMailEntries] then 2 halo flags (owned, zeroed once)
  ShardCtx* d_shard = nullptr;           // device copy of the peer table (owned)
  int shard_rank = -1, shard_world = 0;  // set by amp_pcg_shard_attach*
  int64_t nslices_aligned = 0, nslices_uniform = 0;
  int index_bits = 0, rows_sorted = 0;
  int use_uni_kernel = 0;                // the loop's direct mat-vec is k_spmv_uni (every slice aligned, natural order, no long rows)
  int use_fused = 0, grid_fused = 1;     // the loop runs k_vec_fused (vec_fused.cuh) instead of k_xr, k_z, k_p
  cudaGraph_t graph_fu[2] = {nullptr, nullptr};          // [lagged] graph loops with the fused vector kernel
  cudaGraphExec_t graph_fu_exec[2] = {nullptr, nullptr};
  cudaGraphConditionalHandle cond_fu[2] = {};
  int use_vstage = 0;                    // bit 0: k_z and k_p, bit 1: k_xr and k_xrz are the bulk-copy staged kernels (vec_pipe.cuh)
  int shard_inline = 0;                  // the reducing kernels also collect and step (ranks run concurrently): no k_epi launches
  bool h_state_upload_queued = false;    // an asynchronous upload of h_state may still be queued (amp_spmv_sharded returns without
                                         // synchronising): staging_ready() waits for it before the pinned buffer is rewritten
  unsigned int shard_epoch = 0;          // sharded solves / mat-vecs made so far (identical on all ranks of the group)
  std::vector<void*> ipc_opened;         // peer allocations opened with cudaIpcOpenMemHandle
  cudaGraph_t graph_sh[2] = {nullptr, nullptr};          // [lagged] graph loops of the sharded solve
  cudaGraphExec_t graph_sh_exec[2] = {nullptr, nullptr};
  cudaGraphConditionalHandle cond_sh[2] = {};
};
#ifndef AMP_GRAPH_UNROLL
#define AMP_GRAPH_UNROLL 4
#endif
constexpr int kGraphUnroll = AMP_GRAPH_UNROLL;  // iterations per body of a graph loop (measured on the fused loop, us per iteration for 1 / 2 / 4:
                                                // c2 47.1 / 45.0 / 44.4, c3 79.7 / 77.9 / 76.3, 262 K rows 23.9 / 21.9 / 20.9: the WHILE node costs
                                                // about 2.7 us per evaluation)
constexpr int64_t kVecStagedAutoMinRows = 4000000;  // AMP_VEC_AUTO stages the z and p updates from here on
constexpr size_t kXchgBytes = sizeof(Mail) * kMailEntries + 64;

// The pinned staging copy of the device state is rewritten by every solve / step / sharded mat-vec.  A call that queued an
// upload from it and returned without synchronising must be waited for first, else the next call's host writes race with
// the copy engine (ranks would upload different epochs and wait 10 s for halo tags that never come).
static cudaError_t staging_ready(amp_pcg* h) {
  if (!h->h_state_upload_queued) return cudaSuccess;
  h->h_state_upload_queued = false;
  return cudaStreamSynchronize(h->stream);
}

template <class T> static T* dev_alloc(amp_pcg* h, size_t count, bool zero) {
  void* p = nullptr;
  cudaError_t e = cudaMalloc(&p, std::max<size_t>(count, 1) * sizeof(T));
  if (e != cudaSuccess) {
    set_error("cudaMalloc of %zu bytes failed: %s", count * sizeof(T), cudaGetErrorString(e));
    cudaGetLastError();
    return nullptr;
  }
  h->owned.push_back(p);
  if (zero && cudaMemsetAsync(p, 0, std::max<size_t>(count, 1) * sizeof(T), h->stream) != cudaSuccess) return nullptr;
  return static_cast<T*>(p);
}

extern "C" const char* amp_pcg_last_error(void) { return g_last_error.c_str(); }

extern "C" void amp_policy_default(amp_policy_t* p) {
  if (!p) return;
  std::memset(p, 0, sizeof(*p));
  p->amp = 1; p->u0 = AMP_FP64; p->eta_rule = AMP_ETA_DELAY; p->d = 10; p->ell = 5;
  p->scale_mode = AMP_SCALE_NORM2; p->loop_mode = AMP_LOOP_AUTO;
  p->C = 1.0; p->tau_zs = 1e-4; p->tau_zh = 1e-6; p->eps32 = std::ldexp(1.0, -24);
  p->eta_safety = 1.0; p->stop_safety = 1.0;
}

extern "C" double amp_pcg_bytes_per_row(double m, int uz, int ur) {
  const double sA = (ur == AMP_FP64) ? 8.0 : 4.0, sr = sA;
  const double sz = (uz == AMP_FP64) ? 8.0 : (uz == AMP_FP32 ? 4.0 : 2.0);
  const double sd = (uz == AMP_FP64) ? 8.0 : 4.0;          // 1/diag copy read by the z kernel
  const double k_spmv = m * (sA + 4.0) + 4.0 + sz + sr;    // values+indices, rowptr, p, q
  const double k_z = sr + sd + sz;                         // r, 1/diag -> z
  const double k_p = 3.0 * sz;                             // z, p -> p
  const double k_xr = 16.0 + sz + sr + 2.0 * sr;           // x (r/w FP64), p, q, r (r/w)
  return k_spmv + k_z + k_p + k_xr;
}

static double vec_size(int prec) { return prec == AMP_FP64 ? 8.0 : (prec == AMP_FP32 ? 4.0 : 2.0); }

extern "C" double amp_pcg_spmv_bytes(const amp_pcg_t* h, int mat_prec, int vec_prec) {
  if (!h) return 0.0;
  const double sA = (mat_prec == AMP_FP64) ? 8.0 : 4.0;
  return (double)h->sell_entries * sA + h->idx_bytes_total + h->long_bytes_idx + h->long_entries * sA +
         (double)h->n * (vec_size(vec_prec) + sA);  // p read once, q written once
}

// phase (u_z = FP64, u_r = FP32): the p update also writes RN32(p) (4 B per row) and the mat-vec gathers that copy
static bool shadow_phase(int uz, int ur) { return uz == AMP_FP64 && ur == AMP_FP32; }
static double loop_spmv_bytes(const amp_pcg_t* h, int uz, int ur) {
  return amp_pcg_spmv_bytes(h, ur, shadow_phase(uz, ur) ? AMP_FP32 : uz);
}

extern "C" double amp_pcg_iteration_bytes(const amp_pcg_t* h, int uz, int ur) {
  if (!h) return 0.0;
  const double sr = (ur == AMP_FP64) ? 8.0 : 4.0, sz = vec_size(uz), sd = (uz == AMP_FP64) ? 8.0 : 4.0;
  double k_z = sr + sd + sz;
  const double k_p = 3.0 * sz + (shadow_phase(uz, ur) ? 4.0 : 0.0), k_xr = 16.0 + sz + 3.0 * sr;
  double spmv = loop_spmv_bytes(h, uz, ur);
  if (h->cheb_s > 0) {  // first sweep: r, 1/diag -> d, z; each further sweep: a mat-vec (z -> w) and r, w, 1/diag, d, z -> d, z
    k_z = (sr + sd + 2.0 * sz) + (double)(h->cheb_s - 1) * (2.0 * sr + sd + 4.0 * sz);
    spmv += (double)(h->cheb_s - 1) * amp_pcg_spmv_bytes(h, ur, uz);
  }
  return spmv + (double)h->n * (k_z + k_p + k_xr);
}

extern "C" void amp_pcg_destroy(amp_pcg_t* h) {
  if (!h) return;
  cudaSetDevice(h->device);
  cudaStreamSynchronize(h->stream);
  if (h->graph_exec) cudaGraphExecDestroy(h->graph_exec);
  if (h->graph) cudaGraphDestroy(h->graph);
  if (h->graph_lag_exec) cudaGraphExecDestroy(h->graph_lag_exec);
  if (h->graph_lag) cudaGraphDestroy(h->graph_lag);
  for (int i = 0; i < 2; ++i) {
    if (h->graph_sh_exec[i]) cudaGraphExecDestroy(h->graph_sh_exec[i]);
    if (h->graph_sh[i]) cudaGraphDestroy(h->graph_sh[i]);
    if (h->graph_fu_exec[i]) cudaGraphExecDestroy(h->graph_fu_exec[i]);
    if (h->graph_fu[i]) cudaGraphDestroy(h->graph_fu[i]);
  }
  for (void* p : h->ipc_opened) cudaIpcCloseMemHandle(p);
  for (void* p : h->owned) cudaFree(p);
  if (h->hist) cudaFree(h->hist);
  if (h->h_state) cudaFreeHost(h->h_state);
  if (h->h_flag) cudaFreeHost(h->h_flag);
  if (h->ev0) cudaEventDestroy(h->ev0);
  if (h->ev1) cudaEventDestroy(h->ev1);
  for (cudaEvent_t e : h->prof_events) cudaEventDestroy(e);
  delete h;
}

static bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

extern "C" void amp_create_opts_default(amp_create_opts_t* o) {
  if (!o) return;
  std::memset(o, 0, sizeof(*o));
  o->struct_bytes = (int32_t)sizeof(*o);
  o->precond = AMP_PRECOND_JACOBI;
  o->index_format = AMP_INDEX_AUTO;
  o->spmv_kernel = AMP_SPMV_AUTO;
  o->spmv_grid_mult = 0;
  o->pdl = 1;
  o->cheb_degree = 2;
  o->cheb_lmin = 0.0;
  o->cheb_lmax = 0.0;
  o->stream = nullptr;
  o->halo_lo = 0;
  o->halo_hi = 0;
  o->vec_kernel = AMP_VEC_AUTO;
  o->fuse_vec = AMP_FUSE_AUTO;
}

extern "C" amp_pcg_t* amp_pcg_create(int64_t n, int64_t nnz, const int32_t* rowptr, const int32_t* colidx,
                                     const double* vals, int precond) {
  amp_create_opts_t o;
  amp_create_opts_default(&o);
  o.precond = precond;
  return amp_pcg_create_ex(n, nnz, rowptr, colidx, vals, &o);
}

extern "C" amp_pcg_t* amp_pcg_create_ex(int64_t n, int64_t nnz, const int32_t* rowptr, const int32_t* colidx,
                                        const double* vals, const amp_create_opts_t* opts) {
  g_last_error.clear();
  amp_create_opts_t o;
  amp_create_opts_default(&o);
  if (opts) {
    if (opts->struct_bytes != (int32_t)sizeof(amp_create_opts_t)) {
      set_error("amp_pcg_create_ex: opts->struct_bytes = %d, this library expects %d (use amp_create_opts_default)",
                opts->struct_bytes, (int)sizeof(amp_create_opts_t));
      return nullptr;
    }
    o = *opts;
  }
  const int precond = o.precond;
  if (o.index_format < AMP_INDEX_AUTO || o.index_format > AMP_INDEX_FORCE32 || o.spmv_kernel < AMP_SPMV_AUTO ||
      o.spmv_kernel > AMP_SPMV_PIPELINED || o.spmv_grid_mult < 0 || (o.pdl != 0 && o.pdl != 1) || o.vec_kernel < AMP_VEC_AUTO ||
      o.vec_kernel > AMP_VEC_STAGED || o.fuse_vec < AMP_FUSE_AUTO || o.fuse_vec > AMP_FUSE_ON) {
    set_error("amp_pcg_create_ex: invalid index_format / spmv_kernel / vec_kernel / spmv_grid_mult / pdl");
    return nullptr;
  }
  if (o.halo_lo < 0 || o.halo_hi < 0 || (o.halo_lo & 7) || (o.halo_hi & 7) || o.halo_lo > (1 << 26) || o.halo_hi > (1 << 26) ||
      ((o.halo_lo > 0 || o.halo_hi > 0) && precond == AMP_PRECOND_CHEBJACOBI)) {
    set_error("amp_pcg_create_ex: halo_lo / halo_hi must be multiples of 8 in [0, 2^26] (not available with AMP_PRECOND_CHEBJACOBI)");
    return nullptr;
  }
  if (n <= 0 || n > (int64_t)0x7fffffff - 64 || nnz < 0 || nnz > (int64_t)0x7fffffff - 64) {
    set_error("amp_pcg_create: n and nnz must satisfy 0 < n, 0 <= nnz < 2^31 (got n=%lld nnz=%lld)", (long long)n, (long long)nnz);
    return nullptr;
  }
  if (!rowptr || (nnz > 0 && (!colidx || !vals)) || precond < AMP_PRECOND_NONE || precond > AMP_PRECOND_CHEBJACOBI) {
    set_error("amp_pcg_create: null pointer or unknown preconditioner %d", precond);
    return nullptr;
  }
  if (precond == AMP_PRECOND_CHEBJACOBI &&
      (o.cheb_degree < 1 || o.cheb_degree > kMaxChebDegree || !(o.cheb_lmax >= 0.0) || !(o.cheb_lmin >= 0.0) ||
       (o.cheb_lmax > 0.0 && !(o.cheb_lmin > 0.0 && o.cheb_lmin < o.cheb_lmax)))) {
    set_error("amp_pcg_create_ex: Chebyshev-Jacobi needs 1 <= cheb_degree <= %d and 0 < cheb_lmin < cheb_lmax (or both 0)", kMaxChebDegree);
    return nullptr;
  }
  if (!aligned16(rowptr) || !aligned16(colidx) || !aligned16(vals)) {
    set_error("amp_pcg_create: rowptr, colidx and vals must be 16-byte aligned device pointers");
    return nullptr;
  }
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) {
    cudaGetLastError();
    set_error("amp_pcg_create: no usable CUDA device (this library has no CPU fallback)");
    return nullptr;
  }
  amp_pcg* h = new amp_pcg();
  h->stream = static_cast<cudaStream_t>(o.stream);
  h->pdl = o.pdl;
  CU_TRY(cudaGetDevice(&h->device), { delete h; return nullptr; });
  cudaDeviceProp prop;
  CU_TRY(cudaGetDeviceProperties(&prop, h->device), { delete h; return nullptr; });
  h->num_sms = prop.multiProcessorCount;
  h->n = n; h->nnz = nnz; h->npad = (n + 7) & ~(int64_t)7; h->precond = precond;
  h->m_avg = (double)nnz / (double)n;
  h->halo_lo = o.halo_lo; h->halo_hi = o.halo_hi;
  Ctx& c = h->ctx;
  c.n = n; c.npad = h->npad; c.nnz = nnz;
  c.col_shift = (int32_t)o.halo_lo;
  c.n_scale = n;
  c.rowptr = rowptr; c.colidx = colidx; c.vals64 = vals;

#define ALLOC(dst, T, count)                                            \
  do {                                                                  \
    dst = dev_alloc<T>(h, (count), true);                               \
    if (!dst) { amp_pcg_destroy(h); return nullptr; }                   \
  } while (0)
  const size_t np = (size_t)h->npad;
  double* dinv64; float* dinv32; int* flags;
  ALLOC(dinv64, double, np); ALLOC(dinv32, float, np);
  ALLOC(c.r64, double, np); ALLOC(c.r32, float, np);
  ALLOC(c.q64, double, np); ALLOC(c.q32, float, np);
  ALLOC(c.partials, double, (size_t)4 * kMaxGrid);
  ALLOC(c.st, DevState, 1);
  ALLOC(flags, int, 1);
  ALLOC(h->d_b_stage, double, np);
  ALLOC(h->d_x_stage, double, np);
  c.dinv64 = dinv64; c.dinv32 = dinv32; c.vals32 = nullptr;
  CU_TRY(cudaMallocHost(&h->h_state, sizeof(DevState)), { amp_pcg_destroy(h); return nullptr; });
  CU_TRY(cudaMallocHost(&h->h_flag, 64), { amp_pcg_destroy(h); return nullptr; });
  CU_TRY(cudaEventCreate(&h->ev0), { amp_pcg_destroy(h); return nullptr; });
  CU_TRY(cudaEventCreate(&h->ev1), { amp_pcg_destroy(h); return nullptr; });

  // structure check + 1/diag, FP32 value copy
  const int vgrid = (int)std::min<int64_t>((n + 255) / 256, (int64_t)h->num_sms * 16);
  k_validate_dinv<<<vgrid, 256, 0, h->stream>>>(n, nnz, n + o.halo_lo + o.halo_hi, o.halo_lo, rowptr, colidx, vals,
                                                precond != AMP_PRECOND_NONE, dinv64, dinv32, flags);
  std::vector<int32_t> rp((size_t)n + 1);
  int hflags = 0;
  CU_TRY(cudaMemcpyAsync(&hflags, flags, sizeof(int), cudaMemcpyDeviceToHost, h->stream), { amp_pcg_destroy(h); return nullptr; });
  CU_TRY(cudaMemcpyAsync(rp.data(), rowptr, sizeof(int32_t) * ((size_t)n + 1), cudaMemcpyDeviceToHost, h->stream),
         { amp_pcg_destroy(h); return nullptr; });
  CU_TRY(cudaStreamSynchronize(h->stream), { amp_pcg_destroy(h); return nullptr; });
  if (hflags) {
    set_error("amp_pcg_create: invalid matrix:%s%s%s%s", (hflags & 1) ? " rowptr not monotone or rowptr[n] != nnz;" : "",
              (hflags & 2) ? " column index out of range;" : "", (hflags & 4) ? " missing diagonal entry (Jacobi);" : "",
              (hflags & 8) ? " non-positive diagonal entry (Jacobi);" : "");
    amp_pcg_destroy(h);
    return nullptr;
  }

  // ---- SELL-32 repack of A (spmv.cuh): slice widths, optional windowed row sort, long rows ----
  {
    const int64_t nsl = (n + 31) / 32;
    const int long_min = (int)std::max<int64_t>(256, 8 * (int64_t)std::ceil(h->m_avg));
    std::vector<int32_t> long_rows;
    auto row_len = [&](int64_t r) -> int {  // length inside the slices
      if (r < 0 || r >= n) return 0;
      const int len = rp[(size_t)r + 1] - rp[(size_t)r];
      return len > long_min ? 0 : len;
    };
    int64_t nnz_sell = 0;
    for (int64_t r = 0; r < n; ++r) {
      const int len = rp[(size_t)r + 1] - rp[(size_t)r];
      if (len > long_min) long_rows.push_back((int32_t)r); else nnz_sell += len;
    }
    c.long_min = long_min;
    if (!long_rows.empty()) {  // long rows are summed from the CSR arrays: they need the FP32-rounded CSR values too
      float* vals32;
      ALLOC(vals32, float, (size_t)nnz + 8);
      const int cgrid = (int)std::min<int64_t>((nnz + 255) / 256, (int64_t)h->num_sms * 16);
      k_to_fp32<<<cgrid, 256, 0, h->stream>>>(nnz, vals, vals32);
      c.vals32 = vals32;
    }
    std::vector<int32_t> wptr((size_t)nsl + 1, 0), perm;
    auto build_widths = [&]() -> int64_t {
      int64_t tot = 0;
      for (int64_t sl = 0; sl < nsl; ++sl) {
        int w = 0;
        for (int l = 0; l < 32; ++l) {
          const int64_t slot = sl * 32 + l;
          const int64_t r = perm.empty() ? slot : (int64_t)perm[(size_t)slot];
          w = std::max(w, row_len(r));
        }
        wptr[(size_t)sl] = (int32_t)tot;
        tot += w;
      }
      wptr[(size_t)nsl] = (int32_t)tot;
      return tot;
    };
    int64_t wsum = build_widths();
    if ((double)wsum * 32.0 > 1.03 * (double)nnz_sell + 4096.0) {
      // row lengths vary: sort rows by length (descending, stable) inside windows of kSortWindow rows
      const int64_t kSortWindow = 1024;
      perm.assign((size_t)nsl * 32, -1);
      for (int64_t r = 0; r < n; ++r) perm[(size_t)r] = (int32_t)r;
      for (int64_t w0 = 0; w0 < n; w0 += kSortWindow) {
        const int64_t w1 = std::min(n, w0 + kSortWindow);
        std::stable_sort(perm.begin() + w0, perm.begin() + w1,
                         [&](int32_t x, int32_t y) { return row_len(x) > row_len(y); });
      }
      wsum = build_widths();
    }
    // pass 1 on the device: final width of every slice and whether it is stored diagonal-aligned
    int32_t *wptr_d, *cols_d, *perm_d = nullptr, *long_d, *base_d, *width_d;
    ALLOC(wptr_d, int32_t, wptr.size() + 8);
    ALLOC(width_d, int32_t, (size_t)nsl + 1);
    ALLOC(long_d, int32_t, long_rows.size() + 1);
    if (!perm.empty()) ALLOC(perm_d, int32_t, perm.size());
    if (!long_rows.empty())
      CU_TRY(cudaMemcpyAsync(long_d, long_rows.data(), sizeof(int32_t) * long_rows.size(), cudaMemcpyHostToDevice, h->stream),
             { amp_pcg_destroy(h); return nullptr; });
    if (perm_d)
      CU_TRY(cudaMemcpyAsync(perm_d, perm.data(), sizeof(int32_t) * perm.size(), cudaMemcpyHostToDevice, h->stream),
             { amp_pcg_destroy(h); return nullptr; });
    const int pgrid = (int)((nsl * 32 + 255) / 256);
    const int allow_aligned = (o.index_format == AMP_INDEX_AUTO) ? 1 : 0;
    k_sell_scan<<<pgrid, 256, 0, h->stream>>>((int)n, (int)nsl, long_min, allow_aligned, (int)o.halo_lo, rowptr, colidx, perm_d,
                                             width_d);
    std::vector<int32_t> width((size_t)nsl);
    CU_TRY(cudaMemcpyAsync(width.data(), width_d, sizeof(int32_t) * (size_t)nsl, cudaMemcpyDeviceToHost, h->stream),
           { amp_pcg_destroy(h); return nullptr; });
    CU_TRY(cudaStreamSynchronize(h->stream), { amp_pcg_destroy(h); return nullptr; });
    CU_TRY(cudaGetLastError(), { amp_pcg_destroy(h); return nullptr; });
    wsum = 0;
    int64_t w_aligned = 0;
    for (int64_t sl = 0; sl < nsl; ++sl) {
      const int32_t wv = width[(size_t)sl];
      const int32_t w = wv & 0x7fffffff;
      wptr[(size_t)sl] = (int32_t)wsum | (wv & (int32_t)0x80000000u);
      wsum += w;
      if (wv < 0) w_aligned += w;
      if (wsum * 32 + 256 > (int64_t)0x7fffffff) break;
    }
    wptr[(size_t)nsl] = (int32_t)wsum;
    if (wsum * 32 + 256 > (int64_t)0x7fffffff) {
      set_error("amp_pcg_create: padded SELL-32 storage exceeds 2^31 entries");
      amp_pcg_destroy(h);
      return nullptr;
    }
    const size_t total = (size_t)wsum * 32 + 256;
    uint16_t* cols16_d;
    int* flag16_d;
    double* v64_d; float* v32_d;
    ALLOC(cols_d, int32_t, total);
    ALLOC(cols16_d, uint16_t, total);
    ALLOC(base_d, int32_t, (size_t)wsum + 64);
    ALLOC(flag16_d, int, 1);
    ALLOC(v64_d, double, total);
    ALLOC(v32_d, float, total);
    CU_TRY(cudaMemcpyAsync(wptr_d, wptr.data(), sizeof(int32_t) * wptr.size(), cudaMemcpyHostToDevice, h->stream),
           { amp_pcg_destroy(h); return nullptr; });
    k_sell_pack<<<pgrid, 256, 0, h->stream>>>((int)n, (int)nsl, long_min, (int)o.halo_lo, rowptr, colidx, vals, wptr_d, perm_d,
                                             cols_d, cols16_d, base_d, v64_d, v32_d, flag16_d);
    int wide = 0, maxbase = 0;
    int* maxbase_d;
    ALLOC(maxbase_d, int, 1);
    if (wsum > 0) k_absmax_i32<<<(int)std::min<int64_t>((wsum + 255) / 256, 4096), 256, 0, h->stream>>>(wsum, base_d, maxbase_d);
    CU_TRY(cudaMemcpyAsync(&wide, flag16_d, sizeof(int), cudaMemcpyDeviceToHost, h->stream), { amp_pcg_destroy(h); return nullptr; });
    CU_TRY(cudaMemcpyAsync(&maxbase, maxbase_d, sizeof(int), cudaMemcpyDeviceToHost, h->stream), { amp_pcg_destroy(h); return nullptr; });
    CU_TRY(cudaStreamSynchronize(h->stream), { amp_pcg_destroy(h); return nullptr; });
    CU_TRY(cudaGetLastError(), { amp_pcg_destroy(h); return nullptr; });
    if (o.index_format == AMP_INDEX_FORCE32) wide = 1;
    auto release = [&](void* ptr) {
      cudaFree(ptr);
      h->owned.erase(std::find(h->owned.begin(), h->owned.end(), ptr));
    };
    release(width_d);
    if (wide) {  // some offset needs more than 16 bits: keep the 32-bit indices
      release(cols16_d);
      cols16_d = nullptr;
    } else {
      release(cols_d);
      cols_d = nullptr;
    }
    // bytes of index data the SpMV reads: slice table + bases + per-entry indices of the general slices
    h->idx_bytes_total = 4.0 * (double)(nsl + 1) + 4.0 * (double)wsum + (wide ? 4.0 : 2.0) * 32.0 * (double)(wsum - w_aligned) +
                         (perm.empty() ? 0.0 : 4.0 * 32.0 * (double)nsl);
    c.sell_wptr = wptr_d; c.sell_cols = cols_d; c.sell_cols16 = cols16_d; c.sell_base = base_d;
    c.sell_vals64 = v64_d; c.sell_vals32 = v32_d; c.sell_perm = perm_d;
    c.long_rows = long_d; c.nslices = (int32_t)nsl; c.nlong = (int32_t)long_rows.size();
    h->long_entries = (double)(nnz - nnz_sell);
    h->long_bytes_idx = 4.0 * h->long_entries + 12.0 * (double)long_rows.size();
    h->sell_entries = wsum * 32;
    for (int64_t sl = 0; sl < nsl; ++sl) h->nslices_aligned += width[(size_t)sl] < 0 ? 1 : 0;
    h->index_bits = (w_aligned == wsum) ? 0 : (wide ? 32 : 16);
    h->rows_sorted = perm.empty() ? 0 : 1;

    // ---- uniform stencil (spmv.cuh, narrow_uniform_sum): narrow diagonal-aligned slices that share one set of offsets ----
    {
      int wmax_all = 0;
      for (int64_t sl = 0; sl < nsl; ++sl) wmax_all = std::max(wmax_all, (int)(width[(size_t)sl] & 0x7fffffff));
      // reference slice: the first diagonal-aligned slice of full width from the middle of the matrix on (boundary slices
      // of a grid lack some diagonals)
      int64_t ref = -1;
      for (int64_t sl = nsl / 2; sl < nsl && ref < 0; ++sl)
        if (width[(size_t)sl] < 0 && (int)(width[(size_t)sl] & 0x7fffffff) == wmax_all) ref = sl;
      const int ref_w = wmax_all;
      if (o.index_format == AMP_INDEX_AUTO && wmax_all >= 1 && wmax_all <= 7 && ref >= 0) {
        const int ref_w0 = wptr[(size_t)ref] & 0x7fffffff;
        int* cnt_d;
        ALLOC(cnt_d, int, 1);
        k_mark_uniform<<<(int)((nsl + 255) / 256), 256, 0, h->stream>>>((int)nsl, wptr_d, base_d, ref_w0, ref_w, cnt_d);
        int cnt = 0;
        int32_t ub[8] = {0, 0, 0, 0, 0, 0, 0, 0};
        CU_TRY(cudaMemcpyAsync(&cnt, cnt_d, sizeof(int), cudaMemcpyDeviceToHost, h->stream), { amp_pcg_destroy(h); return nullptr; });
        CU_TRY(cudaMemcpyAsync(ub, base_d + ref_w0, sizeof(int32_t) * (size_t)ref_w, cudaMemcpyDeviceToHost, h->stream),
               { amp_pcg_destroy(h); return nullptr; });
        CU_TRY(cudaStreamSynchronize(h->stream), { amp_pcg_destroy(h); return nullptr; });
        CU_TRY(cudaGetLastError(), { amp_pcg_destroy(h); return nullptr; });
        h->nslices_uniform = cnt;
        if (cnt > 0) {  // (slices that do not match keep the general aligned path: the flag is per slice)
          int maxoff = 0;
          for (int k = 0; k < ref_w; ++k) { c.uni_base[k] = ub[k]; maxoff = std::max(maxoff, std::abs(ub[k])); }
          c.uni_w = ref_w;
          const int64_t uguard = (((int64_t)maxoff + 64 + 127) / 128) * 128;
          if (uguard <= kPipeMaxGuard) { h->guard = std::max(h->guard, uguard); c.uni_noclamp = 1; }
          h->use_uni_kernel = perm.empty() && long_rows.empty() && w_aligned == wsum;
        }
      }
    }
    // ---- bulk-copy pipelined SpMV (spmv_pipe.cuh): eligibility, zero guard band of p, stage plan ----
    {
      bool eligible = o.spmv_kernel != AMP_SPMV_DIRECT && perm.empty() && long_rows.empty() && w_aligned == wsum;
      int wmax = 0;
      for (int64_t sl = 0; sl < nsl; ++sl) wmax = std::max(wmax, (int)(width[(size_t)sl] & 0x7fffffff));
      const int64_t guard = (((int64_t)maxbase + 64 + 127) / 128) * 128;
      if (wmax > kPipeChunkW || guard > kPipeMaxGuard) eligible = false;
      // measured (B200, profiles/r02.md): the pipelined kernel wins for wide slices (c4, 27 entries per row: 181 vs 210 us
      // in the FP32 phase) and loses for narrow ones (c2/c3, 7 per row: 43 vs 29 us), where the per-slice bookkeeping of
      // a consumer warp outweighs its 7 entries; AUTO therefore takes it from an average slice width of 12
      // (also tried for narrow uniform stencils with a consumer path that takes four slices at once with constant
      // offsets: c2 41.5 vs 25.0 us, c3 66.0 vs 39.3 us against the direct k_spmv_uni — 15 consumer warps per SM cannot keep
      // enough gathers of p in flight; dropped)
      if (o.spmv_kernel == AMP_SPMV_AUTO && (double)wsum < 12.0 * (double)nsl) eligible = false;
      if (eligible) {
        cudaError_t ea = cudaFuncSetAttribute((const void*)k_spmv_pipe, cudaFuncAttributeMaxDynamicSharedMemorySize, kPipeSmemBytes);
        if (ea == cudaSuccess)
          ea = cudaFuncSetAttribute((const void*)k_spmv_pipe_sh, cudaFuncAttributeMaxDynamicSharedMemorySize, kPipeSmemBytes);
        if (ea != cudaSuccess) { cudaGetLastError(); eligible = false; }
      }
      if (!eligible && o.spmv_kernel == AMP_SPMV_PIPELINED) {
        set_error("amp_pcg_create_ex: AMP_SPMV_PIPELINED needs a matrix whose SELL-32 slices are all diagonal-aligned "
                  "(natural row order, no long rows, slice width <= %d)", kPipeChunkW);
        amp_pcg_destroy(h);
        return nullptr;
      }
      if (eligible) {
        auto wof = [&](int64_t sl) { return (int)(width[(size_t)sl] & 0x7fffffff); };
        const int cap = (int)std::min<int64_t>(kPipeChunkW, std::max<int64_t>(std::max(wmax, 1), wsum / ((int64_t)h->num_sms * 6)));
        std::vector<int32_t> chunks;       // {first slice, first entry column} per stage
        std::vector<int64_t> cost;         // per stage
        for (int64_t sl = 0; sl < nsl;) {
          chunks.push_back((int32_t)sl);
          chunks.push_back(wptr[(size_t)sl] & 0x7fffffff);
          int acc = 0, cnt = 0;
          while (sl < nsl && cnt < kPipeChunkSlices && acc + wof(sl) <= cap) { acc += wof(sl); ++cnt; ++sl; }
          cost.push_back((int64_t)acc + 2 * cnt);
        }
        const int64_t nch = (int64_t)cost.size();
        chunks.push_back((int32_t)nsl);
        chunks.push_back((int32_t)wsum);
        const int nb = (int)std::max<int64_t>(1, std::min<int64_t>(h->num_sms, nch));
        int64_t total = 0;
        for (int64_t v : cost) total += v;
        std::vector<int32_t> blk((size_t)nb + 1, 0);
        {  // contiguous stage ranges of (nearly) equal cost
          int64_t run = 0;
          int b = 1;
          for (int64_t ch = 0; ch < nch && b < nb; ++ch) {
            run += cost[(size_t)ch];
            while (b < nb && run * nb >= total * b) blk[(size_t)b++] = (int32_t)(ch + 1);
          }
          for (; b <= nb; ++b) blk[(size_t)b] = (int32_t)nch;
        }
        int32_t *chunks_d, *blk_d;
        ALLOC(chunks_d, int32_t, chunks.size());
        ALLOC(blk_d, int32_t, blk.size());
        CU_TRY(cudaMemcpyAsync(chunks_d, chunks.data(), sizeof(int32_t) * chunks.size(), cudaMemcpyHostToDevice, h->stream),
               { amp_pcg_destroy(h); return nullptr; });
        CU_TRY(cudaMemcpyAsync(blk_d, blk.data(), sizeof(int32_t) * blk.size(), cudaMemcpyHostToDevice, h->stream),
               { amp_pcg_destroy(h); return nullptr; });
        CU_TRY(cudaStreamSynchronize(h->stream), { amp_pcg_destroy(h); return nullptr; });
        c.pipe_chunks = chunks_d; c.pipe_blk_chunk = blk_d; c.use_pipe = 1;
        h->use_pipe = 1; h->pipe_grid = nb; h->pipe_chunks = nch; h->guard = std::max(h->guard, guard);
        h->idx_bytes_total += 8.0 * (double)(nch + 1) + 4.0 * (double)(nb + 1);  // stage descriptors
      }
    }
    {  // p and z (both are gathered by a mat-vec: z inside the Chebyshev-Jacobi preconditioner) in their three storage
       // precisions, with the zero guard band on both sides (0 elements unless pipelined); a block row of a sharded
       // system keeps its halo bands there (the guard covers them)
      const int64_t halo = ((std::max(o.halo_lo, o.halo_hi) + 127) / 128) * 128;
      h->guard = std::max(h->guard, halo);
      const size_t g = (size_t)h->guard;
      c.col_min = -(int32_t)h->guard;
      c.col_max = (int32_t)(n - 1 + h->guard);
      double* b64; float* b32; __half* b16;
      ALLOC(b64, double, np + 2 * g); ALLOC(b32, float, np + 2 * g); ALLOC(b16, __half, np + 2 * g);
      h->p_base[0] = b64; h->p_base[1] = b32; h->p_base[2] = b16;
      c.p64 = b64 + g; c.p32 = b32 + g; c.p16 = b16 + g;
      ALLOC(b64, double, np + 2 * g); ALLOC(b32, float, np + 2 * g); ALLOC(b16, __half, np + 2 * g);
      c.z64 = b64 + g; c.z32 = b32 + g; c.z16 = b16 + g;
    }
    if (precond == AMP_PRECOND_CHEBJACOBI) {  // direction vector d, spectrum bounds, recurrence coefficients
      ALLOC(c.d64, double, np); ALLOC(c.d32, float, np); ALLOC(c.d16, __half, np);
      double lmin = o.cheb_lmin, lmax = o.cheb_lmax;
      if (!(lmax > 0.0)) {  // Gershgorin bound of D^-1 A (row sums in CSR order: the same number the oracle computes)
        unsigned long long* gmax_d;
        ALLOC(gmax_d, unsigned long long, 1);
        k_gershgorin<<<vgrid, 256, 0, h->stream>>>(n, rowptr, colidx, vals, gmax_d);
        unsigned long long bits = 0;
        CU_TRY(cudaMemcpyAsync(&bits, gmax_d, sizeof(bits), cudaMemcpyDeviceToHost, h->stream), { amp_pcg_destroy(h); return nullptr; });
        CU_TRY(cudaStreamSynchronize(h->stream), { amp_pcg_destroy(h); return nullptr; });
        std::memcpy(&lmax, &bits, sizeof(double));
        lmin = lmax / 30.0;
      }
      if (!(lmin > 0.0) || !(lmax > lmin) || std::isinf(lmax)) {
        set_error("amp_pcg_create_ex: Chebyshev-Jacobi spectrum bounds are not usable (lmin %g, lmax %g)", lmin, lmax);
        amp_pcg_destroy(h);
        return nullptr;
      }
      h->cheb_s = o.cheb_degree; h->cheb_lmin = lmin; h->cheb_lmax = lmax;
      const double theta = (lmax + lmin) / 2.0, dc = (lmax - lmin) / 2.0, sigma = theta / dc;
      c.cheb_s = o.cheb_degree;
      c.cheb_inv_theta = 1.0 / theta;
      double rho_prev = 1.0 / sigma;
      for (int i = 1; i < o.cheb_degree; ++i) {
        const double rho = 1.0 / (2.0 * sigma - rho_prev);
        c.cheb_c1[i] = rho * rho_prev;
        c.cheb_c2[i] = 2.0 * rho / dc;
        rho_prev = rho;
      }
    }

    // SpMV grid: a warp takes a group of up to kSpmvGroupMax slices per pass; blocks make a whole number of
    // (nearly) equal passes, at most `mult` blocks per SM (AMP_SPMV_GRID_MULT: tuning aid)
    int mult = perm.empty() ? 4 : 55;  // sorted (irregular) matrices: small blocks even out the slice widths
    if (o.spmv_grid_mult > 0) mult = o.spmv_grid_mult;
    const int64_t max_grid = std::min<int64_t>((int64_t)h->num_sms * mult, kMaxGrid);
    const int64_t nblk = (nsl + kSpmvWarps * kSpmvGroupMax - 1) / (kSpmvWarps * kSpmvGroupMax);
    const int64_t passes = std::max<int64_t>(1, (nblk + max_grid - 1) / max_grid);
    h->spmv_grid = (int)std::max<int64_t>(1, (nblk + passes - 1) / passes);
  }

  // persistent kernel and vector kernels: whole multiples of the SM count
  persistent_configure(h->num_sms, &h->persist_grid, &h->persist_ok);
  if (h->persist_ok) {  // small problems: no more blocks than there are SpMV groups for their warps (cheaper barriers)
    const int64_t want = (c.nslices + 2 * (kPersistThreads / 32) - 1) / (2 * (kPersistThreads / 32));
    h->persist_grid = (int)std::max<int64_t>(1, std::min<int64_t>(h->persist_grid, want));
  }
  // vector kernels: one full wave of blocks (grid-stride loops inside); small problems get fewer blocks
  // (at least 2 chunks of 8 elements per thread)
  auto vec_grid_for = [&](const void* kern) -> int {
    int occ = 1;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kern, kVecThreads, 0) != cudaSuccess) { cudaGetLastError(); occ = 1; }
    const int64_t max_grid = std::min<int64_t>((int64_t)h->num_sms * std::max(occ, 1), (int64_t)kMaxGrid);
    const int64_t want = (h->npad / 16 + kVecThreads - 1) / kVecThreads;
    return (int)std::max<int64_t>(1, std::min(max_grid, want));
  };
  h->grid_z = vec_grid_for((const void*)k_z);
  h->grid_p = vec_grid_for((const void*)k_p);
  h->grid_p_sh = vec_grid_for((const void*)k_p_sh);
  h->grid_xr = vec_grid_for((const void*)k_xr);
  h->grid_xrz = vec_grid_for((const void*)k_xrz);
  h->grid_cheb0 = vec_grid_for((const void*)k_cheb0);
  h->grid_cheb_step = vec_grid_for((const void*)k_cheb_step);
  h->vec_grid = vec_grid_for((const void*)k_setup);
  c.spmv_grid_direct = h->spmv_grid;
  c.spmv_grid_pipe = h->pipe_grid;
  // fused vector kernel (vec_fused.cuh): one cooperative kernel per iteration instead of k_xr, k_z, k_p
  {
    int occ = 0, coop = 0;
    cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, h->device);
    const bool ok = coop && cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k_vec_fused<false>, kFusedThreads, 0) == cudaSuccess &&
                    occ >= 1;
    int occ2 = occ;
    if (ok && cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ2, k_vec_fused<true>, kFusedThreads, 0) != cudaSuccess) occ2 = 0;
    cudaGetLastError();
    const int64_t cap = (int64_t)h->num_sms * std::min(occ, occ2);
    const int64_t want = (h->npad / 16 + kFusedThreads - 1) / kFusedThreads;
    h->grid_fused = (int)std::max<int64_t>(1, std::min<int64_t>(std::min<int64_t>(cap, kMaxGrid), want));
    const bool can = ok && occ2 >= 1 && h->cheb_s == 0 && h->halo_lo == 0 && h->halo_hi == 0;
    if (o.fuse_vec == AMP_FUSE_ON && !can) {
      set_error("amp_pcg_create_ex: AMP_FUSE_ON needs cooperative launch and is not available with Chebyshev-Jacobi or block rows");
      amp_pcg_destroy(h);
      return nullptr;
    }
    // measured (B200, profiles/r02.md, ms per solve fused vs unfused): c2 20.98 vs 23.92, c3 78.6 vs 82.6, c4 113.6 vs 119.4;
    // the fused kernel reaches 0.75-0.97 of the copy rate on c4 where k_z / k_p alone sat at 0.45: AUTO = on wherever it can run
    h->use_fused = can && o.fuse_vec != AMP_FUSE_OFF;
  }
  // bulk-copy staged vector kernels (vec_pipe.cuh).  Measured on B200 (profiles/r02.md, us per launch, staged vs direct):
  // c4 (8 M rows) k_z 23.1 vs 27.4 (FP16 phase), 25.1 vs 31.8 (FP32 phase), k_p 18.5 vs 20.5, but k_xr 47.8 vs 44.6; c3
  // (4.1 M) k_z 16.9 vs 21.0, k_p 12.5 vs 14.5, k_xr 29.1 vs 28.4; c2 (2.1 M) a tie.  AUTO therefore stages the z and p
  // updates from 4 M rows on and keeps the direct x/r update; STAGED stages all four (tests, tuning).
  h->use_vstage = o.vec_kernel == AMP_VEC_STAGED ? 3 : ((o.vec_kernel == AMP_VEC_AUTO && n >= kVecStagedAutoMinRows) ? 1 : 0);
  if (h->use_vstage) {
    const void* ks[4] = {(const void*)k_z_st, (const void*)k_p_st, (const void*)k_xr_st, (const void*)k_xrz_st};
    for (const void* k : ks) {
      if (cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, kVpSmemBytes) != cudaSuccess) {
        cudaGetLastError();
        if (o.vec_kernel == AMP_VEC_STAGED) {
          set_error("amp_pcg_create_ex: AMP_VEC_STAGED needs %d bytes of shared memory per block", kVpSmemBytes);
          amp_pcg_destroy(h);
          return nullptr;
        }
        h->use_vstage = 0;
      }
    }
  }
#undef ALLOC
  return h;
}

extern "C" int amp_pcg_set_stream(amp_pcg_t* h, void* cuda_stream) {
  if (!h) return AMP_ERR_INVALID;
  h->stream = static_cast<cudaStream_t>(cuda_stream);
  return AMP_OK;
}

extern "C" int64_t amp_pcg_last_launch_count(const amp_pcg_t* h) { return h ? h->launches : 0; }

extern "C" int amp_pcg_format_info(const amp_pcg_t* h, amp_format_info_t* out) {
  if (!h || !out) return AMP_ERR_INVALID;
  std::memset(out, 0, sizeof(*out));
  out->slices = h->ctx.nslices; out->aligned_slices = h->nslices_aligned; out->uniform_slices = h->nslices_uniform;
  out->stored_entries = h->sell_entries; out->long_rows = h->ctx.nlong; out->guard = h->guard;
  out->index_bits = h->index_bits; out->rows_sorted = h->rows_sorted; out->spmv_pipelined = h->use_pipe;
  out->vec_staged = h->use_vstage; out->uniform_width = h->ctx.uni_w;
  return AMP_OK;
}

// ------------------------------------------------------------------ SpMV entry --------------
template <int UR, class PT>
static void launch_spmv_any(amp_pcg* h, const void* p, void* q, unsigned int halo_seq) {
  Ctx c = h->ctx;
  if (halo_seq == 0u) {  // p is a caller's vector of exactly n entries: no halo bands, no guard band around it
    c.col_min = 0;
    c.col_max = (int32_t)(h->n - 1);
    c.uni_noclamp = 0;
  }
  if (halo_seq == 0u)
    k_spmv_any<UR, PT, false><<<h->spmv_grid, kSpmvThreads, 0, h->stream>>>(
        c, static_cast<const PT*>(p), static_cast<typename Store<UR>::T*>(q), halo_seq);
  else  // peers store into the halo bands while the kernel may already run: coherent gathers
    k_spmv_any<UR, PT, true><<<h->spmv_grid, kSpmvThreads, 0, h->stream>>>(
        c, static_cast<const PT*>(p), static_cast<typename Store<UR>::T*>(q), halo_seq);
}

// halo_seq != 0 (row-sharded solve): p is the handle's own extended p vector; wait for the neighbours' push first
static int spmv_dispatch(amp_pcg* h, int mat_prec, int vec_prec, const void* p, void* q, unsigned int halo_seq = 0u) {
  if (mat_prec == AMP_FP64) {
    if (vec_prec == AMP_FP64) launch_spmv_any<P64, double>(h, p, q, halo_seq);
    else if (vec_prec == AMP_FP32) launch_spmv_any<P64, float>(h, p, q, halo_seq);
    else if (vec_prec == AMP_FP16) launch_spmv_any<P64, __half>(h, p, q, halo_seq);
    else return AMP_ERR_INVALID;
  } else if (mat_prec == AMP_FP32) {
    if (vec_prec == AMP_FP64) launch_spmv_any<P32, double>(h, p, q, halo_seq);
    else if (vec_prec == AMP_FP32) launch_spmv_any<P32, float>(h, p, q, halo_seq);
    else if (vec_prec == AMP_FP16) launch_spmv_any<P32, __half>(h, p, q, halo_seq);
    else return AMP_ERR_INVALID;
  } else {
    return AMP_ERR_INVALID;
  }
  h->launches += 1;
  return AMP_OK;
}

extern "C" int amp_spmv(amp_pcg_t* h, int mat_prec, int vec_prec, const void* p, void* q) {
  g_last_error.clear();
  if (!h || !p || !q) { set_error("amp_spmv: null argument"); return AMP_ERR_INVALID; }
  if (h->halo_lo > 0 || h->halo_hi > 0 || h->shard_world > 0) {
    set_error("amp_spmv: this handle is a block row of a sharded system; use amp_spmv_sharded");
    return AMP_ERR_INVALID;
  }
  CU_TRY(cudaSetDevice(h->device), return AMP_ERR_CUDA);
  h->launches = 0;
  const int rc = spmv_dispatch(h, mat_prec, vec_prec, p, q);
  if (rc != AMP_OK) { set_error("amp_spmv: mat_prec must be FP64/FP32 and vec_prec FP64/FP32/FP16"); return rc; }
  CU_TRY(cudaGetLastError(), return AMP_ERR_CUDA);
  return AMP_OK;
}

// ------------------------------------------------------------------ graph loop --------------
template <class K, class... Args>
static cudaError_t launch_loop_kernel_ex(K kern, int grid, int threads, cudaStream_t s, bool pdl, size_t smem, Args... args) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3((unsigned)grid);
  cfg.blockDim = dim3((unsigned)threads);
  cfg.dynamicSmemBytes = smem;
  cfg.stream = s;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr;
  cfg.numAttrs = pdl ? 1 : 0;
  return cudaLaunchKernelEx(&cfg, kern, args...);
}
// a kernel whose blocks wait for one another at a grid barrier: cooperative launch (all blocks resident or the launch fails)
template <class K, class... Args>
static cudaError_t launch_coop_kernel(K kern, int grid, int threads, cudaStream_t s, Args... args) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3((unsigned)grid);
  cfg.blockDim = dim3((unsigned)threads);
  cfg.stream = s;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeCooperative;
  attr[0].val.cooperative = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  return cudaLaunchKernelEx(&cfg, kern, args...);
}
template <class K>
static cudaError_t launch_loop_kernel(K kern, int grid, int threads, cudaStream_t s, const Ctx& c, bool pdl) {
  return launch_loop_kernel_ex(kern, grid, threads, s, pdl, 0, c);
}

// the vector kernels of the loop: direct (kernels.cuh) or bulk-copy staged (vec_pipe.cuh), by the handle's vec_kernel
enum { VK_Z = 0, VK_P = 1, VK_XR = 2, VK_XRZ = 3 };
static cudaError_t launch_vec(amp_pcg* h, int which, cudaStream_t s, const Ctx& c, bool pdl) {
  if (h->use_vstage & ((which == VK_Z || which == VK_P) ? 1 : 2)) {
    void (*kern)(const Ctx) = which == VK_Z ? k_z_st : which == VK_P ? k_p_st : which == VK_XR ? k_xr_st : k_xrz_st;
    return launch_loop_kernel_ex(kern, h->num_sms, kVpThreads, s, pdl, (size_t)kVpSmemBytes, c);
  }
  switch (which) {
    case VK_Z: return launch_loop_kernel(k_z, h->grid_z, kVecThreads, s, c, pdl);
    case VK_P: return launch_loop_kernel(k_p, h->grid_p, kVecThreads, s, c, pdl);
    case VK_XR: return launch_loop_kernel(k_xr, h->grid_xr, kVecThreads, s, c, pdl);
    default: return launch_loop_kernel(k_xrz, h->grid_xrz, kVecThreads, s, c, pdl);
  }
}

// step a4 inside the loop (zmode = 0), or the mat-vec q = A z inside the Chebyshev-Jacobi preconditioner (zmode = 1):
// the direct kernel, followed by the bulk-copy pipelined kernel when the matrix is eligible (it takes the u_r = FP32
// phases; whichever kernel's phase it is not returns at once)
// pdl_first: whether the first of the (up to) two kernels may start early (false when the mat-vec opens an iteration)
static cudaError_t launch_spmv_loop(amp_pcg* h, cudaStream_t s, const Ctx& c, bool pdl, int zmode = 0, int pdl_first = -1) {
  const bool p1 = pdl_first < 0 ? pdl : pdl_first != 0;
  const bool sh = c.sh != nullptr;  // attached to a shard group: the twins whose gathers of p are coherent loads (kernels.cuh)
  cudaError_t e = (h->use_uni_kernel && zmode == 0)
                      ? launch_loop_kernel_ex(sh ? k_spmv_uni_sh : k_spmv_uni, h->spmv_grid, kSpmvThreads, s, p1, 0, c)
                      : launch_loop_kernel_ex(sh ? k_spmv_sh : k_spmv, h->spmv_grid, kSpmvThreads, s, p1, 0, c, zmode);
  if (e == cudaSuccess && h->use_pipe)
    e = launch_loop_kernel_ex(sh ? k_spmv_pipe_sh : k_spmv_pipe, h->pipe_grid, kPipeThreads, s, pdl, (size_t)kPipeSmemBytes, c, zmode);
  return e;
}

// ---- optional event bracketing of every loop kernel (policy.profile_kernels, stream loop) ----
static cudaError_t prof_mark(amp_pcg* h, cudaStream_t s, int kernel, int iter) {
  if (h->prof_used == h->prof_events.size()) {
    cudaEvent_t e;
    const cudaError_t r = cudaEventCreate(&e);
    if (r != cudaSuccess) return r;
    h->prof_events.push_back(e);
  }
  h->prof_kernel.push_back((int8_t)kernel);
  h->prof_iter.push_back(iter);
  return cudaEventRecord(h->prof_events[h->prof_used++], s);
}

// the four kernels of one iteration; pdl: the last three are launched as programmatic dependents.
// prof_iter >= 0: an event is recorded before every kernel and after the last one (and pdl is off).
static cudaError_t launch_iteration(amp_pcg* h, const Ctx& c, cudaStream_t s, bool pdl, int prof_iter = -1) {
  const bool prof = prof_iter >= 0;
  if (prof) pdl = false;
  cudaError_t e = cudaSuccess;
  if (h->cheb_s > 0) {  // step a2 with M^-1 = Chebyshev-accelerated Jacobi: first sweep, then (mat-vec, sweep) s - 1 times
    if (prof) e = prof_mark(h, s, AMP_K_CHEB0, prof_iter);
    if (e == cudaSuccess) e = launch_loop_kernel(k_cheb0, h->grid_cheb0, kVecThreads, s, c, false);
    for (int i = 1; i < h->cheb_s && e == cudaSuccess; ++i) {
      if (prof) e = prof_mark(h, s, AMP_K_SPMV, prof_iter);
      if (e == cudaSuccess) e = launch_spmv_loop(h, s, c, pdl, 1);
      if (prof && e == cudaSuccess) e = prof_mark(h, s, AMP_K_CHEBSTEP, prof_iter);
      if (e == cudaSuccess) e = launch_loop_kernel_ex(k_cheb_step, h->grid_cheb_step, kVecThreads, s, pdl, 0, c, i);
    }
  } else {
    if (prof) e = prof_mark(h, s, AMP_K_Z, prof_iter);
    if (e == cudaSuccess) e = launch_vec(h, VK_Z, s, c, false);
  }
  if (prof && e == cudaSuccess) e = prof_mark(h, s, AMP_K_P, prof_iter);
  if (e == cudaSuccess) e = launch_vec(h, VK_P, s, c, pdl);
  if (prof && e == cudaSuccess) e = prof_mark(h, s, AMP_K_SPMV, prof_iter);
  if (e == cudaSuccess) e = launch_spmv_loop(h, s, c, pdl);
  if (prof && e == cudaSuccess) e = prof_mark(h, s, AMP_K_XR, prof_iter);
  if (e == cudaSuccess) e = launch_vec(h, VK_XR, s, c, pdl);
  if (prof && e == cudaSuccess) e = prof_mark(h, s, -1, prof_iter);
  return e;
}

// lagged variant: three kernels per iteration (z_0 comes from one k_z before the loop)
static cudaError_t launch_iteration_lagged(amp_pcg* h, const Ctx& c, cudaStream_t s, bool pdl, int prof_iter = -1) {
  const bool prof = prof_iter >= 0;
  if (prof) pdl = false;
  cudaError_t e = cudaSuccess;
  if (prof) e = prof_mark(h, s, AMP_K_P, prof_iter);
  if (e == cudaSuccess) e = launch_vec(h, VK_P, s, c, false);
  if (prof && e == cudaSuccess) e = prof_mark(h, s, AMP_K_SPMV, prof_iter);
  if (e == cudaSuccess) e = launch_spmv_loop(h, s, c, pdl);
  if (prof && e == cudaSuccess) e = prof_mark(h, s, AMP_K_XRZ, prof_iter);
  if (e == cudaSuccess) e = launch_vec(h, VK_XRZ, s, c, pdl);
  if (prof && e == cudaSuccess) e = prof_mark(h, s, -1, prof_iter);
  return e;
}

// loop body with the fused vector kernel (vec_fused.cuh): the mat-vec of iteration k, then x/r of k and z, p of k + 1 in
// one cooperative kernel (z_0, p_0 come from k_z, k_p before the loop)
static cudaError_t launch_iteration_fused(amp_pcg* h, const Ctx& c0, cudaStream_t s, bool pdl, bool lagged, int prof_iter = -1) {
  const bool prof = prof_iter >= 0;
  if (prof) pdl = false;
  Ctx c = c0;
  c.defer_gamma = 1;  // the mat-vec publishes partial sums, k_vec_fused adds them and computes alpha
  cudaError_t e = cudaSuccess;
  if (prof) e = prof_mark(h, s, AMP_K_SPMV, prof_iter);
  if (e == cudaSuccess) e = launch_spmv_loop(h, s, c, pdl, 0, 0);
  if (prof && e == cudaSuccess) e = prof_mark(h, s, AMP_K_VEC_FUSED, prof_iter);
  if (e == cudaSuccess)
    e = lagged ? launch_coop_kernel(k_vec_fused<true>, h->grid_fused, kFusedThreads, s, c)
               : launch_coop_kernel(k_vec_fused<false>, h->grid_fused, kFusedThreads, s, c);
  if (prof && e == cudaSuccess) e = prof_mark(h, s, -1, prof_iter);
  return e;
}

// One graph = one WHILE conditional node whose body is the four loop kernels; the condition is
// written from the device by epi_delta / epi_gamma, so a whole solve is a single launch.
static cudaError_t launch_iteration_sharded(amp_pcg* h, const Ctx& c, cudaStream_t s, bool pdl, bool lagged);

enum { GK_PLAIN = 0, GK_SHARDED = 1, GK_FUSED = 2 };
static int build_graph_once(amp_pcg* h, bool pdl, bool lagged, int kind) {
  const bool sharded = kind == GK_SHARDED, fused = kind == GK_FUSED;
  cudaGraph_t& graph = fused ? h->graph_fu[lagged] : sharded ? h->graph_sh[lagged] : (lagged ? h->graph_lag : h->graph);
  cudaGraphExec_t& graph_exec =
      fused ? h->graph_fu_exec[lagged] : sharded ? h->graph_sh_exec[lagged] : (lagged ? h->graph_lag_exec : h->graph_exec);
  cudaGraphConditionalHandle& cond = fused ? h->cond_fu[lagged] : sharded ? h->cond_sh[lagged] : (lagged ? h->cond_lag : h->cond);
  CU_TRY(cudaGraphCreate(&graph, 0), return AMP_ERR_CUDA);
  CU_TRY(cudaGraphConditionalHandleCreate(&cond, graph, 1, cudaGraphCondAssignDefault), return AMP_ERR_CUDA);
  cudaGraphNodeParams np = {};
  np.type = cudaGraphNodeTypeConditional;
  np.conditional.handle = cond;
  np.conditional.type = cudaGraphCondTypeWhile;
  np.conditional.size = 1;
  cudaGraphNode_t node;
  CU_TRY(cudaGraphAddNode(&node, graph, nullptr, 0, &np), return AMP_ERR_CUDA);
  cudaGraph_t body = np.conditional.phGraph_out[0];
  cudaStream_t cap;
  CU_TRY(cudaStreamCreateWithFlags(&cap, cudaStreamNonBlocking), return AMP_ERR_CUDA);
  Ctx c = h->ctx;
  c.cond = cond;
  c.use_cond = 1;
  cudaError_t e = cudaStreamBeginCaptureToGraph(cap, body, nullptr, nullptr, 0, cudaStreamCaptureModeRelaxed);
  if (e == cudaSuccess) {
    cudaError_t el = cudaSuccess;
    // the body holds several iterations: the loop kernels return at once when the solve has ended, so the WHILE
    // condition is evaluated (and the body re-launched) once per kGraphUnroll iterations
    for (int u = 0; u < kGraphUnroll && el == cudaSuccess; ++u)
      el = fused     ? launch_iteration_fused(h, c, cap, pdl, lagged)
           : sharded ? launch_iteration_sharded(h, c, cap, pdl, lagged)
                     : (lagged ? launch_iteration_lagged(h, c, cap, pdl) : launch_iteration(h, c, cap, pdl));
    e = cudaStreamEndCapture(cap, nullptr);
    if (e == cudaSuccess) e = el;
  }
  cudaStreamDestroy(cap);
  if (e != cudaSuccess) { set_error("graph capture failed: %s", cudaGetErrorString(e)); cudaGetLastError(); return AMP_ERR_CUDA; }
  CU_TRY(cudaGraphInstantiate(&graph_exec, graph, 0), { cudaGetLastError(); return AMP_ERR_CUDA; });
  return AMP_OK;
}

static int build_graph(amp_pcg* h, bool lagged, int kind = GK_PLAIN) {
  const bool sharded = kind == GK_SHARDED, fused = kind == GK_FUSED;
  cudaGraph_t& graph = fused ? h->graph_fu[lagged] : sharded ? h->graph_sh[lagged] : (lagged ? h->graph_lag : h->graph);
  cudaGraphExec_t& graph_exec =
      fused ? h->graph_fu_exec[lagged] : sharded ? h->graph_sh_exec[lagged] : (lagged ? h->graph_lag_exec : h->graph_exec);
  if (graph_exec) return AMP_OK;
  int rc = build_graph_once(h, h->pdl != 0, lagged, kind);
  if (rc != AMP_OK && h->pdl) {  // programmatic edges not accepted inside the conditional body: plain edges
    if (graph_exec) { cudaGraphExecDestroy(graph_exec); graph_exec = nullptr; }
    if (graph) { cudaGraphDestroy(graph); graph = nullptr; }
    h->pdl = 0;
    rc = build_graph_once(h, false, lagged, kind);
  }
  return rc;
}

// ------------------------------------------------------------------ solve -------------------
// policy with its "0 means default" fields resolved; false = invalid tol / maxit / policy
static bool resolve_policy(const amp_policy_t* policy, double tol, int32_t maxit, amp_policy_t* out) {
  amp_policy_t pol;
  if (policy) pol = *policy; else amp_policy_default(&pol);
  if (pol.eps32 == 0.0) pol.eps32 = std::ldexp(1.0, -24);
  if (pol.eta_safety == 0.0) pol.eta_safety = 1.0;
  if (pol.stop_safety == 0.0) pol.stop_safety = 1.0;
  if (pol.C == 0.0 && !policy) pol.C = 1.0;
  *out = pol;
  return !(!(tol > 0.0) || maxit < 1 || maxit > (1 << 24) || pol.u0 < 0 || pol.u0 > 2 ||
           pol.eta_rule < 0 || pol.eta_rule > 2 || pol.scale_mode < 0 || pol.scale_mode > 4 || pol.d < 1 || pol.d > kMaxWindow ||
           pol.ell < 1 || pol.ell > kMaxWindow || pol.loop_mode < 0 || pol.loop_mode > 3 || !(pol.tau_zs >= 0.0) ||
           !(pol.tau_zh >= 0.0) || !(pol.eps32 > 0.0) || !(pol.eta_safety > 0.0) || !(pol.stop_safety > 0.0) ||
           (pol.profile_kernels != 0 && pol.loop_mode != AMP_LOOP_STREAM));
}

// the host-written part of the device state of one solve
static void fill_state(DevState* hs, const amp_pcg* h, const double* b, double* x, double tol, int32_t maxit, const amp_policy_t& pol) {
  std::memset(hs, 0, sizeof(DevState));
  hs->b = b; hs->x = x; hs->hist = h->hist;
  hs->tol = tol; hs->tau_zs = pol.tau_zs; hs->tau_zh = pol.tau_zh; hs->eps32 = pol.eps32; hs->C = pol.C;
  hs->eta_safety = pol.eta_safety; hs->stop_safety = pol.stop_safety;
  hs->amp = pol.amp ? 1 : 0; hs->u0 = pol.u0; hs->eta_rule = pol.eta_rule; hs->d = pol.d; hs->ell = pol.ell;
  hs->scale_mode = pol.scale_mode; hs->no_stop = pol.no_stop ? 1 : 0; hs->maxit = maxit;
  hs->status = AMP_MAXIT; hs->it_ur32 = hs->it_uz32 = hs->it_uz16 = -1;
  hs->relres_true = -1.0;
}

static int ensure_hist(amp_pcg* h, int32_t maxit) {
  if ((int64_t)maxit + 2 > h->hist_cap) {
    if (h->hist) cudaFree(h->hist);
    h->hist = nullptr;
    h->hist_cap = 0;
    CU_TRY(cudaMalloc(&h->hist, sizeof(double) * ((size_t)maxit + 2)), return AMP_ERR_NOMEM);
    h->hist_cap = (int64_t)maxit + 2;
  }
  return AMP_OK;
}

// precisions in use at iteration k (from the switch iterations)
static void phase_of(const DevState* hs, int k, int& uz, int& ur) {
  ur = (hs->it_ur32 >= 0 && k >= hs->it_ur32) ? AMP_FP32 : AMP_FP64;
  uz = hs->amp ? hs->u0 : AMP_FP64;
  if (hs->it_uz32 >= 0 && k >= hs->it_uz32) uz = std::max(uz, (int)AMP_FP32);
  if (hs->it_uz16 >= 0 && k >= hs->it_uz16) uz = AMP_FP16;
}

static void fill_stats(const amp_pcg* h, const DevState* hs, int mode, bool lagged, float ms, amp_stats_t* stats) {
  const int iters = hs->k;
  std::memset(stats, 0, sizeof(*stats));
  stats->status = hs->status; stats->iters = iters;
  stats->it_ur32 = hs->it_ur32; stats->it_uz32 = hs->it_uz32; stats->it_uz16 = hs->it_uz16;
  stats->loop_mode = mode;
  stats->bnorm = hs->bnorm;
  stats->relres_updated = (hs->bnorm > 0.0) ? hs->delta / hs->bnorm : 0.0;
  stats->relres_true = hs->relres_true;
  stats->solve_ms = ms;
  double bytes = 0.0;
  for (int k = 0; k < iters; ++k) {
    int uz, ur;
    phase_of(hs, k, uz, ur);
    bytes += amp_pcg_iteration_bytes(h, uz, ur);
    if (lagged) bytes -= (double)h->n * ((ur == AMP_FP64) ? 8.0 : 4.0);  // r is not read a second time
  }
  stats->algorithmic_bytes = bytes;
  stats->fp16_subnormal = hs->fp16_subnormal; stats->fp16_flushed = hs->fp16_flushed; stats->fp16_inf = hs->fp16_inf;
}

static int solve_impl(amp_pcg* h, const double* b, double* x, double tol, int32_t maxit, const amp_policy_t* policy,
                      amp_stats_t* stats) {
  g_last_error.clear();
  if (!h || !b || !x) { set_error("amp_pcg_solve: null argument"); return AMP_ERR_INVALID; }
  if (h->halo_lo > 0 || h->halo_hi > 0 || h->shard_world > 0) {
    set_error("amp_pcg_solve: this handle is a block row of a sharded system; use amp_pcg_solve_sharded");
    return AMP_ERR_INVALID;
  }
  amp_policy_t pol;
  if (!resolve_policy(policy, tol, maxit, &pol) || !aligned16(b) || !aligned16(x)) {
    set_error("amp_pcg_solve: invalid tol/maxit/policy or misaligned b/x");
    return AMP_ERR_INVALID;
  }
  CU_TRY(cudaSetDevice(h->device), return AMP_ERR_CUDA);
  cudaStream_t st = h->stream;
  { const int rc = ensure_hist(h, maxit); if (rc != AMP_OK) return rc; }
  int mode = pol.loop_mode;
  // measured on B200 (us per iteration, persistent vs graph): n = 4 K 17 vs 23, 16 K 19.6 vs 24.0, 262 K 20.9 vs 29.0,
  // 512 K 25.0 vs 32.1, 2.1 M (c2) 58 vs 57, 4.1 M (c3) 95 vs 92: the persistent kernel wins while the iteration is
  // latency-bound; from c2 up the graph loop wins because each of its kernels has its own register budget
  const bool lagged = pol.amp && pol.scale_mode == AMP_SCALE_LAGGED;
  if (h->cheb_s > 0 && (lagged || mode == AMP_LOOP_PERSISTENT)) {
    set_error("amp_pcg_solve: the Chebyshev-Jacobi preconditioner is not available with AMP_SCALE_LAGGED or AMP_LOOP_PERSISTENT");
    return AMP_ERR_INVALID;
  }
  if (mode == AMP_LOOP_AUTO)
    mode = (h->persist_ok && h->n <= kPersistAutoMaxRows && h->cheb_s == 0) ? AMP_LOOP_PERSISTENT : AMP_LOOP_GRAPH;
  if (mode == AMP_LOOP_PERSISTENT && !h->persist_ok) {
    set_error("amp_pcg_solve: persistent loop not available for this problem/device");
    return AMP_ERR_INVALID;
  }
  const bool fused = h->use_fused && mode != AMP_LOOP_PERSISTENT;
  if (mode == AMP_LOOP_GRAPH) { const int rc = build_graph(h, lagged, fused ? GK_FUSED : GK_PLAIN); if (rc != AMP_OK) return rc; }

  DevState* hs = h->h_state;
  fill_state(hs, h, b, x, tol, maxit, pol);
  h->launches = 0;
  const bool profile = pol.profile_kernels != 0;
  h->prof_used = 0;
  h->prof_kernel.clear();
  h->prof_iter.clear();
  h->prof_result.clear();

  CU_TRY(cudaEventRecord(h->ev0, st), return AMP_ERR_CUDA);
  CU_TRY(cudaMemcpyAsync(h->ctx.st, hs, sizeof(DevState), cudaMemcpyHostToDevice, st), return AMP_ERR_CUDA);
  // a0: r0 = b - A x0 (FP64), ||b||, delta_0
  if (!pol.x0_zero) { spmv_dispatch(h, AMP_FP64, AMP_FP64, x, h->ctx.q64); }
  k_setup<<<h->vec_grid, kVecThreads, 0, st>>>(h->ctx, pol.x0_zero ? 1 : 0);
  h->launches += 1;

  if ((lagged || fused) && mode != AMP_LOOP_PERSISTENT) {  // z_0, rho_0 for the first pass of a loop that opens with p or A p
    CU_TRY(launch_vec(h, VK_Z, st, h->ctx, false), return AMP_ERR_CUDA);
    h->launches += 1;
  }
  if (fused) {  // p_0 too: the fused loop opens with the mat-vec
    CU_TRY(launch_vec(h, VK_P, st, h->ctx, false), return AMP_ERR_CUDA);
    h->launches += 1;
  }
  if (mode == AMP_LOOP_GRAPH) {
    CU_TRY(cudaGraphLaunch(fused ? h->graph_fu_exec[lagged] : (lagged ? h->graph_lag_exec : h->graph_exec), st), return AMP_ERR_CUDA);
  } else if (mode == AMP_LOOP_PERSISTENT) {
    const int rc = persistent_launch(h->ctx, h->persist_grid, st);
    if (rc != 0) { set_error("persistent kernel launch failed: %s", cudaGetErrorString((cudaError_t)rc)); return AMP_ERR_CUDA; }
  } else {
    const int batch = 32;
    int done_iters = 0;
    while (done_iters < maxit) {
      const int nb = std::min(batch, maxit - done_iters);
      for (int i = 0; i < nb; ++i) {
        const int pit = profile ? done_iters + i : -1;
        const cudaError_t el = fused    ? launch_iteration_fused(h, h->ctx, st, h->pdl != 0, lagged, pit)
                               : lagged ? launch_iteration_lagged(h, h->ctx, st, h->pdl != 0, pit)
                                        : launch_iteration(h, h->ctx, st, h->pdl != 0, pit);
        if (el != cudaSuccess) {
          set_error("amp_pcg_solve: loop kernel launch failed: %s", cudaGetErrorString(el));
          cudaGetLastError();
          cudaStreamSynchronize(st);
          return AMP_ERR_CUDA;
        }
      }
      done_iters += nb;
      CU_TRY(cudaMemcpyAsync(h->h_flag, &h->ctx.st->done, sizeof(int), cudaMemcpyDeviceToHost, st), return AMP_ERR_CUDA);
      CU_TRY(cudaStreamSynchronize(st), return AMP_ERR_CUDA);
      if (*h->h_flag) break;
    }
  }
  CU_TRY(cudaEventRecord(h->ev1, st), return AMP_ERR_CUDA);
  if (pol.true_residual) spmv_dispatch(h, AMP_FP64, AMP_FP64, x, h->ctx.q64);
  k_finalize<<<h->vec_grid, kVecThreads, 0, st>>>(h->ctx, pol.true_residual ? 1 : 0);
  h->launches += 1;
  CU_TRY(cudaMemcpyAsync(hs, h->ctx.st, sizeof(DevState), cudaMemcpyDeviceToHost, st), return AMP_ERR_CUDA);
  CU_TRY(cudaStreamSynchronize(st), return AMP_ERR_CUDA);
  CU_TRY(cudaGetLastError(), return AMP_ERR_CUDA);
  float ms = 0.f;
  cudaEventElapsedTime(&ms, h->ev0, h->ev1);

  const int iters = hs->k;
  h->last_iters = iters;
  if (profile) {  // event-to-event device time of every executed loop kernel, summed per (kernel, u_z, u_r)
    amp_kernel_time_t acc[AMP_K_COUNT][3][2];
    std::memset(acc, 0, sizeof(acc));
    for (size_t i = 0; i + 1 < h->prof_used; ++i) {
      const int kern = h->prof_kernel[i], k = h->prof_iter[i];
      if (kern < 0 || k >= iters) continue;
      float dt = 0.f;
      if (cudaEventElapsedTime(&dt, h->prof_events[i], h->prof_events[i + 1]) != cudaSuccess) { cudaGetLastError(); continue; }
      int uz, ur;
      phase_of(hs, k, uz, ur);
      acc[kern][uz][ur].launches += 1;
      acc[kern][uz][ur].total_ms += dt;
    }
    const double n_ = (double)h->n;
    for (int kern = 0; kern < AMP_K_COUNT; ++kern)
      for (int uz = 0; uz < 3; ++uz)
        for (int ur = 0; ur < 2; ++ur) {
          amp_kernel_time_t& a = acc[kern][uz][ur];
          if (a.launches == 0) continue;
          const double sr = (ur == AMP_FP64) ? 8.0 : 4.0, sz = vec_size(uz), sd = (uz == AMP_FP64) ? 8.0 : 4.0;
          a.kernel = kern; a.uz = uz; a.ur = ur;
          switch (kern) {
            case AMP_K_Z: a.bytes_per_launch = n_ * (sr + sd + sz); break;
            case AMP_K_P: a.bytes_per_launch = n_ * (3.0 * sz + (shadow_phase(uz, ur) ? 4.0 : 0.0)); break;
            case AMP_K_SPMV: a.bytes_per_launch = loop_spmv_bytes(h, uz, ur); break;  // (z-mode launches: within 4 B per row of it)
            case AMP_K_CHEB0: a.bytes_per_launch = n_ * (sr + sd + 2.0 * sz); break;
            case AMP_K_CHEBSTEP: a.bytes_per_launch = n_ * (2.0 * sr + sd + 4.0 * sz); break;
            case AMP_K_XR: a.bytes_per_launch = n_ * (16.0 + sz + 3.0 * sr); break;
            case AMP_K_VEC_FUSED:  // x/r of this iteration, then z and p (of the next one: its phase, but for 1-3 launches, is this one's)
              a.bytes_per_launch = n_ * ((16.0 + sz + 3.0 * sr) + (lagged ? sd + sz : sr + sd + sz) + 3.0 * sz +
                                         (shadow_phase(uz, ur) ? 4.0 : 0.0));
              break;
            default: a.bytes_per_launch = n_ * (16.0 + sz + 3.0 * sr + sd + sz); break;  // AMP_K_XRZ
          }
          h->prof_result.push_back(a);
        }
  }
  {
    const int spmv_k = h->use_pipe ? 2 : 1, sweeps = std::max(h->cheb_s, 1);
    const int per_it = fused ? 1 + spmv_k : (lagged ? 2 : 3) + spmv_k + (sweeps - 1) * (spmv_k + 1);  // vector kernels + a4 + extra sweeps
    // a graph body holds kGraphUnroll iterations: the ones after the last are launched too (and return at once)
    const int64_t its_launched = (mode == AMP_LOOP_GRAPH) ? (int64_t)(iters + kGraphUnroll - 1) / kGraphUnroll * kGraphUnroll : iters;
    h->launches += (mode == AMP_LOOP_PERSISTENT) ? 1 : (int64_t)per_it * its_launched;
  }
  if (stats) fill_stats(h, hs, mode, lagged, ms, stats);
  return hs->status;
}

#include "shard_host.cuh"

extern "C" int amp_pcg_solve(amp_pcg_t* h, const double* b, double* x, double tol, int32_t maxit,
                             const amp_policy_t* policy, amp_stats_t* stats) {
  return solve_impl(h, b, x, tol, maxit, policy, stats);
}

extern "C" int amp_pcg_solve_host(amp_pcg_t* h, const double* b_host, double* x_host, double tol, int32_t maxit,
                                  const amp_policy_t* policy, amp_stats_t* stats) {
  g_last_error.clear();
  if (!h || !b_host || !x_host) { set_error("amp_pcg_solve_host: null argument"); return AMP_ERR_INVALID; }
  CU_TRY(cudaSetDevice(h->device), return AMP_ERR_CUDA);
  const size_t bytes = sizeof(double) * (size_t)h->n;
  CU_TRY(cudaMemcpyAsync(h->d_b_stage, b_host, bytes, cudaMemcpyHostToDevice, h->stream), return AMP_ERR_CUDA);
  if (!(policy && policy->x0_zero))
    CU_TRY(cudaMemcpyAsync(h->d_x_stage, x_host, bytes, cudaMemcpyHostToDevice, h->stream), return AMP_ERR_CUDA);
  const int rc = solve_impl(h, h->d_b_stage, h->d_x_stage, tol, maxit, policy, stats);
  if (rc < 0 && rc != AMP_ERR_BREAKDOWN) return rc;
  CU_TRY(cudaMemcpyAsync(x_host, h->d_x_stage, bytes, cudaMemcpyDeviceToHost, h->stream), return AMP_ERR_CUDA);
  CU_TRY(cudaStreamSynchronize(h->stream), return AMP_ERR_CUDA);
  return rc;
}

extern "C" int32_t amp_pcg_residual_history(amp_pcg_t* h, double* out_host, int32_t count) {
  if (!h || !out_host || count < 0) return AMP_ERR_INVALID;
  if (h->last_iters < 0 || !h->hist) return 0;
  const int32_t m = std::min<int32_t>(count, h->last_iters + 1);
  if (m == 0) return 0;
  CU_TRY(cudaMemcpyAsync(out_host, h->hist, sizeof(double) * (size_t)m, cudaMemcpyDeviceToHost, h->stream), return AMP_ERR_CUDA);
  CU_TRY(cudaStreamSynchronize(h->stream), return AMP_ERR_CUDA);
  return m;
}

// eta_hat_m(k), k = 0..m, of (4.7) from the residual-norm history of the last solve: with
// c_t = (3+C)||r_{t-1}|| + (2+C)||r_t|| (||r_{-1}|| := ||r_0||, reading R2), eta_hat_m(k) = eps64 * (c_0 + .. + c_k) +
// eps32 * (c_k + .. + c_m): one prefix and one suffix sum on the host.  Diagnostic post-processing, not on the hot path.
extern "C" int32_t amp_pcg_eta_posteriori(amp_pcg_t* h, double C, double eps32, double* out_host, int32_t count) {
  g_last_error.clear();
  if (!h || !out_host || count < 0 || !(C >= 0.0) || !(eps32 >= 0.0)) { set_error("amp_pcg_eta_posteriori: invalid argument"); return AMP_ERR_INVALID; }
  if (h->last_iters < 0 || !h->hist) return 0;
  if (eps32 == 0.0) eps32 = std::ldexp(1.0, -24);
  const double eps64 = std::ldexp(1.0, -53);
  const int32_t m = h->last_iters;
  std::vector<double> hist((size_t)m + 1), c((size_t)m + 1), suffix((size_t)m + 2, 0.0);
  CU_TRY(cudaSetDevice(h->device), return AMP_ERR_CUDA);
  CU_TRY(cudaMemcpyAsync(hist.data(), h->hist, sizeof(double) * hist.size(), cudaMemcpyDeviceToHost, h->stream), return AMP_ERR_CUDA);
  CU_TRY(cudaStreamSynchronize(h->stream), return AMP_ERR_CUDA);
  for (int32_t t = 0; t <= m; ++t) c[(size_t)t] = (3.0 + C) * hist[(size_t)(t > 0 ? t - 1 : 0)] + (2.0 + C) * hist[(size_t)t];
  for (int32_t t = m; t >= 0; --t) suffix[(size_t)t] = suffix[(size_t)t + 1] + c[(size_t)t];
  const int32_t nout = std::min<int32_t>(count, m + 1);
  double prefix = 0.0;
  for (int32_t k = 0; k < nout; ++k) {
    prefix += c[(size_t)k];
    out_host[k] = eps64 * prefix + eps32 * suffix[(size_t)k];
  }
  return nout;
}

extern "C" int32_t amp_pcg_kernel_times(amp_pcg_t* h, amp_kernel_time_t* out_host, int32_t cap) {
  if (!h || !out_host || cap < 0) return AMP_ERR_INVALID;
  const int32_t m = std::min<int32_t>(cap, (int32_t)h->prof_result.size());
  for (int32_t i = 0; i < m; ++i) out_host[i] = h->prof_result[(size_t)i];
  return m;
}

// ------------------------------------------------------------------ diagnostic entry points --
static bool debug_vec(amp_pcg* h, int which, int prec, void** ptr, size_t* elem) {
  const Ctx& c = h->ctx;
  *ptr = nullptr;
  *elem = prec == AMP_FP64 ? 8 : (prec == AMP_FP32 ? 4 : 2);
  switch (which) {
    case AMP_VEC_R: *ptr = prec == AMP_FP64 ? (void*)c.r64 : prec == AMP_FP32 ? (void*)c.r32 : nullptr; break;
    case AMP_VEC_Q: *ptr = prec == AMP_FP64 ? (void*)c.q64 : prec == AMP_FP32 ? (void*)c.q32 : nullptr; break;
    case AMP_VEC_Z: *ptr = prec == AMP_FP64 ? (void*)c.z64 : prec == AMP_FP32 ? (void*)c.z32 : prec == AMP_FP16 ? (void*)c.z16 : nullptr; break;
    case AMP_VEC_P: *ptr = prec == AMP_FP64 ? (void*)c.p64 : prec == AMP_FP32 ? (void*)c.p32 : prec == AMP_FP16 ? (void*)c.p16 : nullptr; break;
    case AMP_VEC_DINV: *ptr = prec == AMP_FP64 ? (void*)c.dinv64 : prec == AMP_FP32 ? (void*)c.dinv32 : nullptr; break;
    case AMP_VEC_D: *ptr = prec == AMP_FP64 ? (void*)c.d64 : prec == AMP_FP32 ? (void*)c.d32 : prec == AMP_FP16 ? (void*)c.d16 : nullptr; break;
    default: break;
  }
  return *ptr != nullptr;
}

extern "C" int amp_pcg_debug_set_vector(amp_pcg_t* h, int which, int prec, const void* src) {
  g_last_error.clear();
  void* dst; size_t es;
  if (!h || !src || which == AMP_VEC_DINV || !debug_vec(h, which, prec, &dst, &es)) {
    set_error("amp_pcg_debug_set_vector: invalid handle / vector / precision");
    return AMP_ERR_INVALID;
  }
  CU_TRY(cudaSetDevice(h->device), return AMP_ERR_CUDA);
  CU_TRY(cudaMemsetAsync(dst, 0, es * (size_t)h->npad, h->stream), return AMP_ERR_CUDA);
  CU_TRY(cudaMemcpyAsync(dst, src, es * (size_t)h->n, cudaMemcpyDeviceToDevice, h->stream), return AMP_ERR_CUDA);
  if (which == AMP_VEC_P && prec == AMP_FP64) {  // keep the FP32 copy RN32(p) the (FP64, FP32) phase gathers in step
    const int cgrid = (int)std::min<int64_t>((h->n + 255) / 256, (int64_t)h->num_sms * 16);
    k_to_fp32<<<cgrid, 256, 0, h->stream>>>(h->n, h->ctx.p64, h->ctx.p32);
  }
  return AMP_OK;
}

extern "C" int amp_pcg_debug_get_vector(amp_pcg_t* h, int which, int prec, void* dst) {
  g_last_error.clear();
  void* src; size_t es;
  if (!h || !dst || !debug_vec(h, which, prec, &src, &es)) {
    set_error("amp_pcg_debug_get_vector: invalid handle / vector / precision");
    return AMP_ERR_INVALID;
  }
  CU_TRY(cudaSetDevice(h->device), return AMP_ERR_CUDA);
  CU_TRY(cudaMemcpyAsync(dst, src, es * (size_t)h->n, cudaMemcpyDeviceToDevice, h->stream), return AMP_ERR_CUDA);
  return AMP_OK;
}

extern "C" int amp_pcg_debug_step(amp_pcg_t* h, amp_debug_step_t* io, double* x) {
  g_last_error.clear();
  auto prec_ok = [](int p, int lo) { return p >= 0 && p <= lo; };
  if (!h || !io || io->step < AMP_STEP_Z || io->step > AMP_STEP_CHEBSTEP || !prec_ok(io->rs, 1) || !prec_ok(io->ur, 1) ||
      !prec_ok(io->uz, 2) || !prec_ok(io->ps, 2) || !prec_ok(io->ur_n, 1) || !prec_ok(io->uz_n, 2) || io->rs > io->ur ||
      io->ps > io->uz || io->ur > io->ur_n || io->uz > io->uz_n ||
      ((io->step == AMP_STEP_XR || io->step == AMP_STEP_XRZ) && (!x || !aligned16(x))) ||
      (io->step >= AMP_STEP_CHEB0 && h->cheb_s == 0) ||
      (io->step == AMP_STEP_CHEBSTEP && (io->first < 1 || io->first >= h->cheb_s))) {
    set_error("amp_pcg_debug_step: invalid step / precision combination (precisions only step down) or x missing");
    return AMP_ERR_INVALID;
  }
  CU_TRY(cudaSetDevice(h->device), return AMP_ERR_CUDA);
  cudaStream_t st = h->stream;
  if (h->hist_cap < 64) {
    if (h->hist) cudaFree(h->hist);
    h->hist = nullptr; h->hist_cap = 0;
    CU_TRY(cudaMalloc(&h->hist, sizeof(double) * 64), return AMP_ERR_NOMEM);
    h->hist_cap = 64;
  }
  CU_TRY(cudaMemsetAsync(h->hist, 0, sizeof(double) * 64, st), return AMP_ERR_CUDA);
  CU_TRY(staging_ready(h), return AMP_ERR_CUDA);
  DevState* hs = h->h_state;
  std::memset(hs, 0, sizeof(DevState));
  hs->x = x; hs->hist = h->hist;
  hs->tol = 1.0; hs->eps32 = std::ldexp(1.0, -24); hs->C = 1.0; hs->eta_safety = 1.0; hs->stop_safety = 1.0;
  hs->amp = 0; hs->eta_rule = AMP_ETA_NEVER; hs->d = 10; hs->ell = 5; hs->no_stop = 1; hs->maxit = 1 << 20;
  hs->bnorm = 1.0; hs->rho = 1.0; hs->rho_prev = 1.0;
  hs->status = AMP_MAXIT; hs->it_ur32 = hs->it_uz32 = hs->it_uz16 = -1;
  hs->k = (io->first && io->step == AMP_STEP_P) ? 0 : 1;
  hs->r_store = io->rs; hs->ur = io->ur; hs->uz = io->uz; hs->p_store = io->ps;
  hs->ur_n = io->ur_n; hs->uz_n = io->uz_n;
  hs->omega = io->omega; hs->beta = io->beta; hs->alpha = io->alpha; hs->omega_n = io->omega_n;
  CU_TRY(cudaMemcpyAsync(h->ctx.st, hs, sizeof(DevState), cudaMemcpyHostToDevice, st), return AMP_ERR_CUDA);
  cudaError_t e = cudaSuccess;
  switch (io->step) {  // the very kernels, grids and block sizes the stream / graph loop launches
    case AMP_STEP_Z: e = launch_vec(h, VK_Z, st, h->ctx, false); break;
    case AMP_STEP_P: e = launch_vec(h, VK_P, st, h->ctx, false); break;
    case AMP_STEP_SPMV: e = launch_spmv_loop(h, st, h->ctx, false); break;
    case AMP_STEP_XR: e = launch_vec(h, VK_XR, st, h->ctx, false); break;
    case AMP_STEP_XRZ: e = launch_vec(h, VK_XRZ, st, h->ctx, false); break;
    case AMP_STEP_CHEB0: e = launch_loop_kernel(k_cheb0, h->grid_cheb0, kVecThreads, st, h->ctx, false); break;
    case AMP_STEP_SPMV_Z: e = launch_spmv_loop(h, st, h->ctx, false, 1); break;
    default: e = launch_loop_kernel_ex(k_cheb_step, h->grid_cheb_step, kVecThreads, st, false, 0, h->ctx, (int)io->first); break;
  }
  if (e != cudaSuccess) { set_error("amp_pcg_debug_step: launch failed: %s", cudaGetErrorString(e)); cudaGetLastError(); return AMP_ERR_CUDA; }
  CU_TRY(cudaMemcpyAsync(hs, h->ctx.st, sizeof(DevState), cudaMemcpyDeviceToHost, st), return AMP_ERR_CUDA);
  CU_TRY(cudaStreamSynchronize(st), return AMP_ERR_CUDA);
  CU_TRY(cudaGetLastError(), return AMP_ERR_CUDA);
  io->sum0 = io->sum1 = 0.0;
  switch (io->step) {
    case AMP_STEP_Z: case AMP_STEP_CHEB0: case AMP_STEP_CHEBSTEP: io->sum0 = hs->rho; break;
    case AMP_STEP_SPMV: io->sum0 = hs->gamma; break;
    case AMP_STEP_XR: io->sum0 = hs->delta; break;
    case AMP_STEP_XRZ: io->sum0 = hs->delta; io->sum1 = hs->rho; break;
    default: break;
  }
  return AMP_OK;
}
