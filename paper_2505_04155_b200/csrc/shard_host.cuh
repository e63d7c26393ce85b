// shard_host.cuh — host side of the row-sharded solve (include/amp_pcg.h "row-sharded solve"; SURVEY.md section 8(e),
// 8(f) NEXT-3): the block-row partition, the peer wiring (in-process or CUDA IPC) and the driver that launches the
// loop kernels of every local rank.  Included by amp_pcg.cu (uses its handle struct and launch helpers).
// All arithmetic and both exchanges (halo of p, partial sums) run in the kernels (shard.cuh, kernels.cuh).
#pragma once

// ------------------------------------------------------------------ partition (host only, no CUDA) ----
extern "C" int amp_shard_plan(int64_t n, const int32_t* rowptr, const int32_t* colidx, int32_t world, amp_shard_t* out) {
  g_last_error.clear();
  if (n <= 0 || !rowptr || !out || world < 1 || world > AMP_SHARD_MAX_WORLD || rowptr[0] != 0 || (rowptr[n] > 0 && !colidx)) {
    set_error("amp_shard_plan: invalid argument (1 <= world <= %d)", AMP_SHARD_MAX_WORLD);
    return AMP_ERR_INVALID;
  }
  const int64_t nnz = rowptr[n];
  const int64_t nslices = (n + 31) / 32;
  if (nslices < world) { set_error("amp_shard_plan: fewer than 32 rows per rank"); return AMP_ERR_INVALID; }
  // boundaries on whole SELL-32 slices, balanced by cost = stored entries + 4 per row (the vector kernels' share)
  const double total = (double)nnz + 4.0 * (double)n;
  int64_t row = 0;
  for (int32_t r = 0; r < world; ++r) {
    out[r].row0 = row;
    int64_t end;
    if (r == world - 1) {
      end = n;
    } else {
      const double target = total * (double)(r + 1) / (double)world;
      int64_t lo = row / 32 + 1, hi = nslices - (world - 1 - r);  // at least one slice for this rank and for each later one
      while (lo < hi) {  // first slice boundary whose cumulative cost reaches the target
        const int64_t mid = (lo + hi) / 2, e = std::min<int64_t>(mid * 32, n);
        if ((double)rowptr[e] + 4.0 * (double)e >= target) hi = mid; else lo = mid + 1;
      }
      end = std::min<int64_t>(lo * 32, n);
    }
    out[r].row1 = end;
    out[r].nnz = (int64_t)rowptr[end] - (int64_t)rowptr[row];
    int64_t cmin = row, cmax = end - 1;
    for (int64_t e = rowptr[row]; e < rowptr[end]; ++e) {
      const int64_t j = colidx[e];
      if (j < 0 || j >= n) { set_error("amp_shard_plan: column index out of range"); return AMP_ERR_INVALID; }
      cmin = std::min(cmin, j);
      cmax = std::max(cmax, j);
    }
    out[r].halo_lo = ((row - cmin) + 7) / 8 * 8;
    out[r].halo_hi = ((cmax - (end - 1)) + 7) / 8 * 8;
    row = end;
  }
  // a halo must lie inside the adjacent rank.  The widths are rounded up to 8 and a rank's p is zero-padded to a multiple of 8
  // (the pushed chunks may cover the padding), so the bound is the neighbour's PADDED row count: only the last rank's can
  // differ from its row count (the other boundaries are multiples of 32)
  for (int32_t r = 0; r < world; ++r) {
    const int64_t below = r > 0 ? out[r - 1].row1 - out[r - 1].row0 : 0;
    const int64_t above = r + 1 < world ? (out[r + 1].row1 - out[r + 1].row0 + 7) / 8 * 8 : 0;
    if (r == 0) out[r].halo_lo = 0;
    if (r == world - 1) out[r].halo_hi = 0;
    if (out[r].halo_lo > below || out[r].halo_hi > above) {
      set_error("amp_shard_plan: the halo of rank %d (%lld below, %lld above) reaches past its neighbour ranks (%lld, %lld rows): "
                "the coupling is not banded enough for %d ranks", r, (long long)out[r].halo_lo, (long long)out[r].halo_hi,
                (long long)below, (long long)above, world);
      return AMP_ERR_INVALID;
    }
  }
  return AMP_OK;
}

extern "C" int amp_shard_extract(int64_t n, const int32_t* rowptr, const int32_t* colidx, const double* vals, const amp_shard_t* s,
                                 int32_t* rowptr_out, int32_t* colidx_out, double* vals_out) {
  g_last_error.clear();
  if (n <= 0 || !rowptr || !s || !rowptr_out || s->row0 < 0 || s->row1 > n || s->row0 >= s->row1 ||
      (s->nnz > 0 && (!colidx || !vals || !colidx_out || !vals_out))) {
    set_error("amp_shard_extract: invalid argument");
    return AMP_ERR_INVALID;
  }
  const int64_t e0 = rowptr[s->row0], shift = s->halo_lo - s->row0, ncols = s->halo_lo + (s->row1 - s->row0) + s->halo_hi;
  if ((int64_t)rowptr[s->row1] - e0 != s->nnz) { set_error("amp_shard_extract: the plan does not belong to this matrix"); return AMP_ERR_INVALID; }
  for (int64_t i = s->row0; i <= s->row1; ++i) rowptr_out[i - s->row0] = (int32_t)(rowptr[i] - e0);
  for (int64_t e = 0; e < s->nnz; ++e) {
    const int64_t j = (int64_t)colidx[e0 + e] + shift;
    if (j < 0 || j >= ncols) { set_error("amp_shard_extract: an entry lies outside the planned halo"); return AMP_ERR_INVALID; }
    colidx_out[e] = (int32_t)j;
    vals_out[e] = vals[e0 + e];
  }
  return AMP_OK;
}

// ------------------------------------------------------------------ wiring ------------------------
static int ensure_xchg(amp_pcg* h) {
  if (h->xchg) return AMP_OK;
  CU_TRY(cudaSetDevice(h->device), return AMP_ERR_CUDA);
  void* p = nullptr;
  CU_TRY(cudaMalloc(&p, kXchgBytes), return AMP_ERR_NOMEM);
  h->owned.push_back(p);
  CU_TRY(cudaMemset(p, 0, kXchgBytes), return AMP_ERR_CUDA);
  h->xchg = static_cast<char*>(p);
  return AMP_OK;
}
static Mail* xchg_mbox(char* x) { return reinterpret_cast<Mail*>(x); }
static unsigned long long* xchg_flags(char* x) { return reinterpret_cast<unsigned long long*>(x + sizeof(Mail) * kMailEntries); }

struct ShardPeer {  // what a rank needs to know about another rank
  int64_t n, halo_lo, halo_hi, guard;
  char* xchg;       // its exchange block, mapped here
  char* p[3];       // its p64 / p32 / p16 (first OWNED entry), mapped here; nullptr if not a neighbour
};

// build and upload this rank's peer table
static int shard_wire(amp_pcg* h, int rank, int world, const ShardPeer* peers, bool concurrent) {
  const ShardPeer& me = peers[rank];
  if (me.n != h->n || me.halo_lo != h->halo_lo || me.halo_hi != h->halo_hi) { set_error("shard attach: inconsistent geometry of rank %d", rank); return AMP_ERR_INVALID; }
  ShardCtx sc;
  std::memset(&sc, 0, sizeof(sc));
  sc.rank = rank; sc.world = world;
  sc.inline_epi = concurrent ? 1 : 0;
  sc.mbox = xchg_mbox(h->xchg);
  sc.flags = xchg_flags(h->xchg);
  for (int r = 0; r < world; ++r) sc.peer_mbox[r] = xchg_mbox(peers[r].xchg);
  const size_t es[3] = {8, 4, 2};
  if (rank == 0 && h->halo_lo != 0) { set_error("shard attach: rank 0 must have halo_lo = 0"); return AMP_ERR_INVALID; }
  if (rank == world - 1 && h->halo_hi != 0) { set_error("shard attach: the last rank must have halo_hi = 0"); return AMP_ERR_INVALID; }
  if (rank > 0) {  // rank-1 needs my first halo_hi(rank-1) entries in its upper band
    const ShardPeer& nb = peers[rank - 1];
    if (nb.halo_hi > h->npad || h->halo_lo > nb.n || nb.halo_hi > nb.guard || (nb.n & 31)) {  // npad: see amp_shard_plan
      set_error("shard attach: halo of rank %d / %d does not fit its neighbour (or %d's rows are not a multiple of 32)", rank - 1, rank, rank - 1);
      return AMP_ERR_INVALID;
    }
    sc.send_lo = (int32_t)nb.halo_hi;
    if (sc.send_lo > 0)
      for (int k = 0; k < 3; ++k) sc.peer_lo_band[k] = nb.p[k] + (size_t)nb.n * es[k];
    sc.peer_flag_lo = xchg_flags(nb.xchg) + 1;  // raised even when nothing is pushed: the neighbour waits for it
  }
  if (rank + 1 < world) {  // rank+1 needs my last halo_lo(rank+1) entries in its lower band
    const ShardPeer& nb = peers[rank + 1];
    if (nb.halo_lo > h->n || h->halo_hi > (nb.n + 7) / 8 * 8 || nb.halo_lo > nb.guard || (h->n & 31)) {
      set_error("shard attach: halo of rank %d / %d does not fit its neighbour (or %d's rows are not a multiple of 32)", rank, rank + 1, rank);
      return AMP_ERR_INVALID;
    }
    sc.send_hi = (int32_t)nb.halo_lo;
    if (sc.send_hi > 0)
      for (int k = 0; k < 3; ++k) sc.peer_hi_band[k] = nb.p[k] - (size_t)sc.send_hi * es[k];
    sc.peer_flag_hi = xchg_flags(nb.xchg) + 0;
  }
  CU_TRY(cudaSetDevice(h->device), return AMP_ERR_CUDA);
  if (!h->d_shard) {
    void* p = nullptr;
    CU_TRY(cudaMalloc(&p, sizeof(ShardCtx)), return AMP_ERR_NOMEM);
    h->owned.push_back(p);
    h->d_shard = static_cast<ShardCtx*>(p);
  }
  CU_TRY(cudaMemcpy(h->d_shard, &sc, sizeof(sc), cudaMemcpyHostToDevice), return AMP_ERR_CUDA);
  h->ctx.sh = h->d_shard;
  h->ctx.n_scale = 0;
  for (int r = 0; r < world; ++r) h->ctx.n_scale += peers[r].n;  // the n of omega = sqrt(n)/||r|| is the whole system's
  h->shard_rank = rank; h->shard_world = world; h->shard_epoch = 0;
  h->shard_inline = concurrent ? 1 : 0;
  for (int i = 0; i < 2; ++i) {  // graphs captured with another wiring are stale
    if (h->graph_sh_exec[i]) { cudaGraphExecDestroy(h->graph_sh_exec[i]); h->graph_sh_exec[i] = nullptr; }
    if (h->graph_sh[i]) { cudaGraphDestroy(h->graph_sh[i]); h->graph_sh[i] = nullptr; }
  }
  return AMP_OK;
}

static bool shard_capable(const amp_pcg* h) { return h && h->cheb_s == 0; }

extern "C" int amp_pcg_shard_attach_local(amp_pcg_t* const* handles, int32_t world) {
  g_last_error.clear();
  if (!handles || world < 1 || world > kMaxWorld) { set_error("amp_pcg_shard_attach_local: invalid argument"); return AMP_ERR_INVALID; }
  ShardPeer peers[kMaxWorld];
  for (int r = 0; r < world; ++r) {
    amp_pcg* h = handles[r];
    if (!shard_capable(h) || h->precond != handles[0]->precond) {
      set_error("amp_pcg_shard_attach_local: null handle, Chebyshev-Jacobi handle, or preconditioners differ");
      return AMP_ERR_INVALID;
    }
    const int rc = ensure_xchg(h);
    if (rc != AMP_OK) return rc;
    peers[r] = ShardPeer{h->n, h->halo_lo, h->halo_hi, h->guard, h->xchg,
                         {reinterpret_cast<char*>(h->ctx.p64), reinterpret_cast<char*>(h->ctx.p32), reinterpret_cast<char*>(h->ctx.p16)}};
  }
  for (int r = 0; r < world; ++r)  // ranks on different devices of this process: direct peer access
    for (int q = 0; q < world; ++q)
      if (handles[r]->device != handles[q]->device) {
        CU_TRY(cudaSetDevice(handles[r]->device), return AMP_ERR_CUDA);
        const cudaError_t e = cudaDeviceEnablePeerAccess(handles[q]->device, 0);
        if (e != cudaSuccess && e != cudaErrorPeerAccessAlreadyEnabled) { set_error("cudaDeviceEnablePeerAccess failed: %s", cudaGetErrorString(e)); return AMP_ERR_CUDA; }
        cudaGetLastError();
      }
  // ranks that share a device run one after the other: the scalar steps then need kernels of their own (k_epi), launched
  // after the reducing kernels of ALL ranks; ranks on distinct devices (and a single rank) run concurrently
  bool concurrent = true;
  for (int r = 0; r < world; ++r)
    for (int q = 0; q < r; ++q) concurrent = concurrent && handles[r]->device != handles[q]->device;
  for (int r = 0; r < world; ++r) {
    const int rc = shard_wire(handles[r], r, world, peers, concurrent);
    if (rc != AMP_OK) return rc;
  }
  return AMP_OK;
}

extern "C" int amp_pcg_shard_export(amp_pcg_t* h, amp_shard_export_t* out) {
  g_last_error.clear();
  if (!shard_capable(h) || !out) { set_error("amp_pcg_shard_export: invalid argument"); return AMP_ERR_INVALID; }
  static_assert(sizeof(cudaIpcMemHandle_t) <= 64, "IPC handle size");
  const int rc = ensure_xchg(h);
  if (rc != AMP_OK) return rc;
  std::memset(out, 0, sizeof(*out));
  out->n = h->n; out->halo_lo = h->halo_lo; out->halo_hi = h->halo_hi; out->guard = h->guard;
  void* objs[4] = {h->xchg, h->p_base[0], h->p_base[1], h->p_base[2]};
  const size_t es[4] = {1, 8, 4, 2};
  for (int k = 0; k < 4; ++k) {
    cudaIpcMemHandle_t mh;
    CU_TRY(cudaIpcGetMemHandle(&mh, objs[k]), return AMP_ERR_CUDA);
    std::memcpy(out->mem[k], &mh, sizeof(mh));
    out->off[k] = k == 0 ? 0 : (int64_t)((size_t)h->guard * es[k]);  // first owned entry of p inside its allocation
  }
  return AMP_OK;
}

extern "C" int amp_pcg_shard_attach(amp_pcg_t* h, int32_t rank, int32_t world, const amp_shard_export_t* all) {
  g_last_error.clear();
  if (!shard_capable(h) || !all || world < 1 || world > kMaxWorld || rank < 0 || rank >= world) {
    set_error("amp_pcg_shard_attach: invalid argument");
    return AMP_ERR_INVALID;
  }
  const int rc = ensure_xchg(h);
  if (rc != AMP_OK) return rc;
  CU_TRY(cudaSetDevice(h->device), return AMP_ERR_CUDA);
  for (void* p : h->ipc_opened) cudaIpcCloseMemHandle(p);
  h->ipc_opened.clear();
  ShardPeer peers[kMaxWorld];
  auto open = [&](const unsigned char* blob, char** out) -> int {
    cudaIpcMemHandle_t mh;
    std::memcpy(&mh, blob, sizeof(mh));
    void* p = nullptr;
    CU_TRY(cudaIpcOpenMemHandle(&p, mh, cudaIpcMemLazyEnablePeerAccess), return AMP_ERR_CUDA);
    h->ipc_opened.push_back(p);
    *out = static_cast<char*>(p);
    return AMP_OK;
  };
  for (int r = 0; r < world; ++r) {
    const amp_shard_export_t& e = all[r];
    peers[r] = ShardPeer{e.n, e.halo_lo, e.halo_hi, e.guard, nullptr, {nullptr, nullptr, nullptr}};
    if (r == rank) {
      peers[r].xchg = h->xchg;
      peers[r].p[0] = reinterpret_cast<char*>(h->ctx.p64); peers[r].p[1] = reinterpret_cast<char*>(h->ctx.p32);
      peers[r].p[2] = reinterpret_cast<char*>(h->ctx.p16);
      continue;
    }
    char* base = nullptr;
    int rc2 = open(e.mem[0], &base);  // every rank's mailbox
    if (rc2 != AMP_OK) return rc2;
    peers[r].xchg = base + e.off[0];
    if (r == rank - 1 || r == rank + 1) {  // the neighbours' p vectors
      for (int k = 0; k < 3; ++k) {
        rc2 = open(e.mem[1 + k], &base);
        if (rc2 != AMP_OK) return rc2;
        peers[r].p[k] = base + e.off[1 + k];
      }
    }
  }
  return shard_wire(h, rank, world, peers, true);  // one process per GPU: all ranks run concurrently
}

// ------------------------------------------------------------------ driver ------------------------
enum ShardStep { SS_Z, SS_EPI_RHO, SS_P, SS_SPMV, SS_EPI_GAMMA, SS_XR, SS_EPI_DELTA, SS_XRZ, SS_EPI_DELTA_LAGGED };
static const int kShardStepsPlain[] = {SS_Z, SS_EPI_RHO, SS_P, SS_SPMV, SS_EPI_GAMMA, SS_XR, SS_EPI_DELTA};
static const int kShardStepsLagged[] = {SS_P, SS_SPMV, SS_EPI_GAMMA, SS_XRZ, SS_EPI_DELTA_LAGGED};

static bool shard_step_is_epi(int step) {
  return step == SS_EPI_RHO || step == SS_EPI_GAMMA || step == SS_EPI_DELTA || step == SS_EPI_DELTA_LAGGED;
}

static cudaError_t launch_shard_step(amp_pcg* h, const Ctx& c, cudaStream_t s, bool pdl, int step) {
  if (h->shard_inline && shard_step_is_epi(step)) return cudaSuccess;  // done by the reducing kernel itself
  switch (step) {
    case SS_Z: return launch_vec(h, VK_Z, s, c, pdl);
    case SS_EPI_RHO: return launch_loop_kernel_ex(k_epi, 1, 32, s, pdl, 0, c, (int)kEpiRho);
    case SS_P: return launch_loop_kernel(k_p_sh, h->grid_p_sh, kVecThreads, s, c, pdl);
    case SS_SPMV: return launch_spmv_loop(h, s, c, pdl);
    case SS_EPI_GAMMA: return launch_loop_kernel_ex(k_epi, 1, 32, s, pdl, 0, c, (int)kEpiGamma);
    case SS_XR: return launch_vec(h, VK_XR, s, c, pdl);
    case SS_EPI_DELTA: return launch_loop_kernel_ex(k_epi, 1, 32, s, pdl, 0, c, (int)kEpiDelta);
    case SS_XRZ: return launch_vec(h, VK_XRZ, s, c, pdl);
    default: return launch_loop_kernel_ex(k_epi, 1, 32, s, pdl, 0, c, (int)kEpiDeltaLagged);
  }
}

// one iteration of ONE rank (graph body of the one-process-per-GPU mode): the first kernel with a plain dependency
static cudaError_t launch_iteration_sharded(amp_pcg* h, const Ctx& c, cudaStream_t s, bool pdl, bool lagged) {
  const int* steps = lagged ? kShardStepsLagged : kShardStepsPlain;
  const int nsteps = lagged ? 5 : 7;
  cudaError_t e = cudaSuccess;
  for (int i = 0; i < nsteps && e == cudaSuccess; ++i) e = launch_shard_step(h, c, s, pdl && i > 0, steps[i]);
  return e;
}

static int shard_group_check(amp_pcg_t* const* handles, int32_t nlocal, const char* who) {
  if (!handles || nlocal < 1 || nlocal > kMaxWorld || !handles[0]) { set_error("%s: invalid handle list", who); return AMP_ERR_INVALID; }
  const int world = handles[0]->shard_world;
  if (world < 1 || (nlocal != 1 && nlocal != world)) {
    set_error("%s: handles are not attached (amp_pcg_shard_attach*) or nlocal is neither 1 nor the group size", who);
    return AMP_ERR_INVALID;
  }
  for (int i = 0; i < nlocal; ++i) {
    const amp_pcg* h = handles[i];
    if (!h || h->shard_world != world || (nlocal > 1 && h->shard_rank != i) || h->shard_epoch != handles[0]->shard_epoch ||
        h->shard_inline != handles[0]->shard_inline) {
      set_error("%s: handle %d does not belong to the group (rank order, group size or solve count differ)", who, i);
      return AMP_ERR_INVALID;
    }
    for (int j = 0; j < i; ++j)
      if (handles[j]->device == h->device && handles[j]->stream != h->stream) {
        set_error("%s: ranks that share a device must share a stream (their kernels wait for one another)", who);
        return AMP_ERR_INVALID;
      }
  }
  return AMP_OK;
}

extern "C" int amp_pcg_solve_sharded(amp_pcg_t* const* handles, int32_t nlocal, const double* const* b, double* const* x, double tol,
                                     int32_t maxit, const amp_policy_t* policy, amp_stats_t* stats) {
  g_last_error.clear();
  int rc = shard_group_check(handles, nlocal, "amp_pcg_solve_sharded");
  if (rc != AMP_OK) return rc;
  amp_policy_t pol;
  bool ok = b && x && resolve_policy(policy, tol, maxit, &pol);
  for (int i = 0; ok && i < nlocal; ++i) ok = b[i] && x[i] && aligned16(b[i]) && aligned16(x[i]);
  if (!ok || pol.profile_kernels || pol.loop_mode == AMP_LOOP_PERSISTENT || (pol.loop_mode == AMP_LOOP_GRAPH && nlocal > 1)) {
    set_error("amp_pcg_solve_sharded: invalid tol/maxit/policy/b/x (no persistent loop, no kernel profile; graph loop only with nlocal = 1)");
    return AMP_ERR_INVALID;
  }
  const bool lagged = pol.amp && pol.scale_mode == AMP_SCALE_LAGGED;
  const int mode = (pol.loop_mode == AMP_LOOP_AUTO) ? (nlocal == 1 ? AMP_LOOP_GRAPH : AMP_LOOP_STREAM) : pol.loop_mode;
  for (int i = 0; i < nlocal; ++i) {
    amp_pcg* h = handles[i];
    CU_TRY(cudaSetDevice(h->device), return AMP_ERR_CUDA);
    rc = ensure_hist(h, maxit);
    if (rc != AMP_OK) return rc;
    if (mode == AMP_LOOP_GRAPH) { rc = build_graph(h, lagged, true); if (rc != AMP_OK) return rc; }
    CU_TRY(staging_ready(h), return AMP_ERR_CUDA);
    h->shard_epoch += 1;
    fill_state(h->h_state, h, b[i], x[i], tol, maxit, pol);
    h->h_state->epoch = h->shard_epoch;
    h->launches = 0;
    CU_TRY(cudaEventRecord(h->ev0, h->stream), return AMP_ERR_CUDA);
    CU_TRY(cudaMemcpyAsync(h->ctx.st, h->h_state, sizeof(DevState), cudaMemcpyHostToDevice, h->stream), return AMP_ERR_CUDA);
  }
  // every kernel of a step is launched for all local ranks before the next step (ranks on one device run one after the
  // other: a kernel that waits for a peer must find that the peer has already run)
#define FOR_RANKS(...)                                                \
  for (int i_ = 0; i_ < nlocal; ++i_) {                               \
    amp_pcg* h = handles[i_];                                         \
    CU_TRY(cudaSetDevice(h->device), return AMP_ERR_CUDA);            \
    __VA_ARGS__;                                                      \
  }
  // a0: r0 = b - A x0 in FP64 (x0 and its halo go through the p vector), ||b||, delta_0
  if (!pol.x0_zero) {
    FOR_RANKS(k_shard_load_p<<<h->vec_grid, kVecThreads, 0, h->stream>>>(h->ctx, h->h_state->x, (int)P64, kHaloTagSetup));
    FOR_RANKS(spmv_dispatch(h, AMP_FP64, AMP_FP64, h->ctx.p64, h->ctx.q64, kHaloTagSetup));
  }
  FOR_RANKS(k_setup<<<h->vec_grid, kVecThreads, 0, h->stream>>>(h->ctx, pol.x0_zero ? 1 : 0));
  const bool split_epi = handles[0]->shard_inline == 0;
  if (split_epi) { FOR_RANKS(k_epi<<<1, 32, 0, h->stream>>>(h->ctx, (int)kEpiSetup)); }
  if (lagged) {
    FOR_RANKS(CU_TRY(launch_vec(h, VK_Z, h->stream, h->ctx, false), return AMP_ERR_CUDA));
    if (split_epi) { FOR_RANKS(k_epi<<<1, 32, 0, h->stream>>>(h->ctx, (int)kEpiRho)); }
  }
  if (mode == AMP_LOOP_GRAPH) {
    FOR_RANKS(CU_TRY(cudaGraphLaunch(h->graph_sh_exec[lagged], h->stream), return AMP_ERR_CUDA));
  } else {
    const int* steps = lagged ? kShardStepsLagged : kShardStepsPlain;
    const int nsteps = lagged ? 5 : 7, batch = 32;
    int done_iters = 0;
    while (done_iters < maxit) {
      const int nbatch = std::min(batch, maxit - done_iters);
      for (int it = 0; it < nbatch; ++it)
        for (int sidx = 0; sidx < nsteps; ++sidx) {
          FOR_RANKS({
            const cudaError_t el = launch_shard_step(h, h->ctx, h->stream, h->pdl != 0 && sidx > 0 && nlocal == 1, steps[sidx]);
            if (el != cudaSuccess) {
              set_error("amp_pcg_solve_sharded: loop kernel launch failed: %s", cudaGetErrorString(el));
              cudaGetLastError();
              return AMP_ERR_CUDA;
            }
          });
        }
      done_iters += nbatch;
      FOR_RANKS(CU_TRY(cudaMemcpyAsync(h->h_flag, &h->ctx.st->done, sizeof(int), cudaMemcpyDeviceToHost, h->stream), return AMP_ERR_CUDA));
      bool all_done = true;
      FOR_RANKS({
        CU_TRY(cudaStreamSynchronize(h->stream), return AMP_ERR_CUDA);
        all_done = all_done && *h->h_flag != 0;
      });
      if (all_done) break;
    }
  }
  FOR_RANKS(CU_TRY(cudaEventRecord(h->ev1, h->stream), return AMP_ERR_CUDA));
  if (pol.true_residual) {  // ||b - A x|| / ||b|| in FP64: x and its halo through the p vector once more
    FOR_RANKS(k_shard_load_p<<<h->vec_grid, kVecThreads, 0, h->stream>>>(h->ctx, h->h_state->x, (int)P64, kHaloTagFinal));
    FOR_RANKS(spmv_dispatch(h, AMP_FP64, AMP_FP64, h->ctx.p64, h->ctx.q64, kHaloTagFinal));
  }
  FOR_RANKS(k_finalize<<<h->vec_grid, kVecThreads, 0, h->stream>>>(h->ctx, pol.true_residual ? 1 : 0));
  if (pol.true_residual && split_epi) { FOR_RANKS(k_epi<<<1, 32, 0, h->stream>>>(h->ctx, (int)kEpiFinal)); }
  FOR_RANKS(CU_TRY(cudaMemcpyAsync(h->h_state, h->ctx.st, sizeof(DevState), cudaMemcpyDeviceToHost, h->stream), return AMP_ERR_CUDA));
  int status = AMP_OK;
  for (int i = 0; i < nlocal; ++i) {
    amp_pcg* h = handles[i];
    CU_TRY(cudaSetDevice(h->device), return AMP_ERR_CUDA);
    CU_TRY(cudaStreamSynchronize(h->stream), return AMP_ERR_CUDA);
    CU_TRY(cudaGetLastError(), return AMP_ERR_CUDA);
    float ms = 0.f;
    cudaEventElapsedTime(&ms, h->ev0, h->ev1);
    const DevState* hs = h->h_state;
    h->last_iters = hs->k;
    const int spmv_k = h->use_pipe ? 2 : 1;
    const int epi = split_epi ? 1 : 0;  // k_epi launches per reduction point
    const int64_t its = (mode == AMP_LOOP_GRAPH) ? (int64_t)(hs->k + kGraphUnroll - 1) / kGraphUnroll * kGraphUnroll : hs->k;
    h->launches = 1 + epi + (pol.x0_zero ? 0 : 2) + (lagged ? 1 + epi : 0) + (pol.true_residual ? 3 + epi : 1) +
                  its * ((lagged ? 2 : 3) + spmv_k + (lagged ? 2 : 3) * epi);
    if (stats) fill_stats(h, hs, mode, lagged, ms, stats + i);
    if (i == 0) status = hs->status;
    else if (hs->status != status || hs->k != handles[0]->h_state->k) {
      set_error("amp_pcg_solve_sharded: ranks disagree (status %d vs %d, iterations %d vs %d)", hs->status, status, hs->k,
                handles[0]->h_state->k);
      return AMP_ERR_CUDA;
    }
  }
  if (status == AMP_ERR_CUDA) set_error("amp_pcg_solve_sharded: a rank waited longer than 10 s for a peer");
  return status;
}

extern "C" int amp_spmv_sharded(amp_pcg_t* const* handles, int32_t nlocal, int mat_prec, int vec_prec, const void* const* p,
                                void* const* q) {
  g_last_error.clear();
  int rc = shard_group_check(handles, nlocal, "amp_spmv_sharded");
  if (rc != AMP_OK) return rc;
  if (!p || !q || mat_prec < AMP_FP64 || mat_prec > AMP_FP32 || vec_prec < AMP_FP64 || vec_prec > AMP_FP16) {
    set_error("amp_spmv_sharded: mat_prec must be FP64/FP32 and vec_prec FP64/FP32/FP16");
    return AMP_ERR_INVALID;
  }
  for (int i = 0; i < nlocal; ++i) {  // the halo tags carry the group's call counter
    amp_pcg* h = handles[i];
    if (!p[i] || !q[i]) { set_error("amp_spmv_sharded: null vector"); return AMP_ERR_INVALID; }
    CU_TRY(cudaSetDevice(h->device), return AMP_ERR_CUDA);
    CU_TRY(staging_ready(h), return AMP_ERR_CUDA);
    h->shard_epoch += 1;
    std::memset(h->h_state, 0, sizeof(DevState));
    h->h_state->epoch = h->shard_epoch;
    CU_TRY(cudaMemcpyAsync(h->ctx.st, h->h_state, sizeof(DevState), cudaMemcpyHostToDevice, h->stream), return AMP_ERR_CUDA);
    h->h_state_upload_queued = true;  // this call returns without synchronising
    h->launches = 2;
  }
  FOR_RANKS(k_shard_load_p<<<h->vec_grid, kVecThreads, 0, h->stream>>>(h->ctx, p[i_], vec_prec, kHaloTagSpmv));
  FOR_RANKS({
    const void* pin = vec_prec == AMP_FP64 ? (const void*)h->ctx.p64 : vec_prec == AMP_FP32 ? (const void*)h->ctx.p32 : (const void*)h->ctx.p16;
    spmv_dispatch(h, mat_prec, vec_prec, pin, q[i_], kHaloTagSpmv);
  });
  FOR_RANKS(CU_TRY(cudaGetLastError(), return AMP_ERR_CUDA));
  return AMP_OK;
}
#undef FOR_RANKS
