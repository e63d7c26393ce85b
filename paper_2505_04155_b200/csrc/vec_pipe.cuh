// vec_pipe.cuh — the vector steps of the loop (a2 z/rho, a3 p, a5 x/r/delta, lagged a5+a2; Alg 4.1 lines 4-6, 10, 15-17,
// PAPER.md:274-301) as persistent, bulk-copy staged kernels.
//
// Why.  The direct vector kernels (kernels.cuh) are not limited by HBM: every warp loads its chunks, waits, then runs
// its FP64 arithmetic and the storage-format conversions (2-5 per element on the XU pipe, 16 lanes per clock and SM), so
// memory and arithmetic alternate instead of overlapping, and a third of the elapsed time is ramp and tail
// (ncu, profiles/r02a.md: k_z 0.45, k_p 0.45 of the copy rate on c4).  Here, as in the pipelined SpMV (spmv_pipe.cuh):
//   * one block per SM, resident for the whole pass, owns a contiguous range of elements;
//   * ONE producer thread streams the input vectors of that range with cp.async.bulk into a ring of shared-memory
//     stages (one stage = one chunk of E elements for each of the 512 consumer threads), completion on an mbarrier per
//     stage: the loads run ahead of the arithmetic whatever the consumers do;
//   * 16 consumer warps take one chunk per thread and stage, run the SAME chunk body as the direct kernel (phases.cuh:
//     z_chunk, p_chunk, xr_chunk, xrz_chunk — same operations, same single rounding, so results are bit-identical) and
//     store their outputs straight to global memory with 128-bit stores.
// The last, partial group of 8 elements (x is caller-owned and exactly n long) is done by direct loads.
#pragma once
#include "async_copy.cuh"
#include "phases.cuh"
#include "shard.cuh"

namespace amp {

constexpr int kVpConsumers = 512;                 // consumer threads: 16 warps
constexpr int kVpThreads = kVpConsumers + 32;     // + one producer warp
constexpr int kVpDataBytes = 160 * 1024;          // ring of stages
constexpr int kVpMaxStages = 8;
constexpr int kVpSmemBytes = kVpDataBytes + 2 * kVpMaxStages * 8;

struct VpBars {
  uint64_t* full;
  uint64_t* empty;
};
__device__ __forceinline__ VpBars vp_bars(unsigned char* smem) {
  uint64_t* b = reinterpret_cast<uint64_t*>(smem + kVpDataBytes);
  return VpBars{b, b + kVpMaxStages};
}
// once per kernel, before any role split
__device__ __forceinline__ void vp_init(unsigned char* smem) {
  if (threadIdx.x == 0) {
    const VpBars bars = vp_bars(smem);
#pragma unroll
    for (int s = 0; s < kVpMaxStages; ++s) { mbar_init(bars.full + s, 1); mbar_init(bars.empty + s, kVpConsumers / 32); }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
}

// One staged pass over the elements [0, 8 * (n / 8)).  in[i] / es[i]: base pointer and element size of input stream i
// (use[i] = false: not read, e.g. p at k = 0); stage layout: stream i at byte offset stage_elems * (es[0] + .. + es[i-1]).
// body(sp, t, chunk): sp[i] = stream i of the current stage in shared memory, t = this thread's chunk inside the
// stage, chunk = its global chunk index.  tail(chunk): the chunks of the last partial group of 8 elements, direct loads.
template <int E, int NIN, class Body, class Tail>
__device__ __forceinline__ void vp_run(const Ctx& c, const char* const (&in)[NIN], const int (&es)[NIN], const bool (&use)[NIN],
                                       unsigned char* smem, Body&& body, Tail&& tail) {
  int bpe = 0;
#pragma unroll
  for (int i = 0; i < NIN; ++i) bpe += es[i];
  constexpr int stage_elems = kVpConsumers * E;
  const int stage_bytes = stage_elems * bpe;
  const int nst = min(kVpMaxStages, kVpDataBytes / stage_bytes);
  const VpBars bars = vp_bars(smem);
  const int64_t omain = c.n >> 3;  // full groups of 8 elements
  const int64_t o0 = omain * blockIdx.x / gridDim.x, o1 = omain * (blockIdx.x + 1) / gridDim.x;
  const int64_t e_begin = o0 * 8, e_end = o1 * 8;
  const int nstages = (int)((e_end - e_begin + stage_elems - 1) / stage_elems);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  if (warp == kVpConsumers / 32) {
    if (lane == 0) {  // ---- producer ----
      for (int si = 0; si < nstages; ++si) {
        const int st = si % nst, round = si / nst;
        if (round > 0) mbar_wait(bars.empty + st, (uint32_t)((round - 1) & 1));
        const int64_t e0 = e_begin + (int64_t)si * stage_elems;
        const uint32_t cnt = (uint32_t)min((int64_t)stage_elems, e_end - e0);
        uint32_t bytes = 0;
#pragma unroll
        for (int i = 0; i < NIN; ++i) bytes += use[i] ? cnt * (uint32_t)es[i] : 0u;
        mbar_arrive_expect_tx(bars.full + st, bytes);
        unsigned char* dst = smem + (size_t)st * stage_bytes;
#pragma unroll
        for (int i = 0; i < NIN; ++i) {
          if (use[i]) bulk_g2s(dst, in[i] + e0 * es[i], cnt * (uint32_t)es[i], bars.full + st);
          dst += stage_elems * es[i];
        }
      }
    }
  } else {  // ---- consumers ----
    const int t = threadIdx.x;
    for (int si = 0; si < nstages; ++si) {
      const int st = si % nst, round = si / nst;
      const int64_t e0 = e_begin + (int64_t)si * stage_elems;
      const int cnt = (int)min((int64_t)stage_elems, e_end - e0);
      mbar_wait(bars.full + st, (uint32_t)(round & 1));
      if (t * E < cnt) {
        const unsigned char* sp[NIN];
        const unsigned char* p = smem + (size_t)st * stage_bytes;
#pragma unroll
        for (int i = 0; i < NIN; ++i) { sp[i] = p; p += stage_elems * es[i]; }
        body(sp, t, e0 / E + t);
      }
      __syncwarp();
      if (lane == 0) mbar_arrive(bars.empty + st);
    }
    // the last partial group of 8 elements (vectors are padded to 8 with zeros; x is exactly n long)
    if (blockIdx.x == gridDim.x - 1) {
      const int64_t ctail0 = omain * 8 / E, ctail1 = c.npad / E;
      if (ctail0 + t < ctail1) tail(ctail0 + t);
    }
  }
}

// ------------------------------------------------------------------ a2 ----------------------
template <int RS, int UR, int UZ>
__device__ __forceinline__ double phase_z_staged(const Ctx& c, const double omega, unsigned char* smem) {
  using T = ZT<RS, UR, UZ>;
  using TR = typename T::TR;
  using TD = typename T::TD;
  constexpr int E = T::E;
  const TR* rin = rvec<RS>(c);
  const TD* dinv = T::dinv(c);
  const char* in[2] = {reinterpret_cast<const char*>(rin), reinterpret_cast<const char*>(dinv)};
  const int es[2] = {(int)sizeof(TR), (int)sizeof(TD)};
  const bool use[2] = {true, true};
  double sum = 0.0;
  vp_run<E, 2>(c, in, es, use, smem,
               [&](const unsigned char* const (&sp)[2], int t, int64_t i) {
                 Chunk<TR, E> rr;
                 Chunk<TD, E> dd;
                 chunk_load(rr, reinterpret_cast<const TR*>(sp[0]), t);
                 chunk_load(dd, reinterpret_cast<const TD*>(sp[1]), t);
                 z_chunk<RS, UR, UZ>(c, omega, rr, dd, i, sum);
               },
               [&](int64_t i) {
                 Chunk<TR, E> rr;
                 Chunk<TD, E> dd;
                 chunk_load(rr, rin, i);
                 chunk_load(dd, dinv, i);
                 z_chunk<RS, UR, UZ>(c, omega, rr, dd, i, sum);
               });
  return sum;
}

// ------------------------------------------------------------------ a3 ----------------------
template <int PS, int UZ>
__device__ __forceinline__ void phase_p_staged(const Ctx& c, const double beta, const bool first, const bool shadow32, unsigned char* smem) {
  using T = PT_<PS, UZ>;
  using TP = typename T::TP;
  using TZ = typename T::TZ;
  constexpr int E = T::E;
  const TP* pin = pvec<PS>(c);
  const TZ* z = zvec<UZ>(c);
  const char* in[2] = {reinterpret_cast<const char*>(z), reinterpret_cast<const char*>(pin)};
  const int es[2] = {(int)sizeof(TZ), (int)sizeof(TP)};
  const bool use[2] = {true, !first};
  const PPush<UZ> ph;
  vp_run<E, 2>(c, in, es, use, smem,
               [&](const unsigned char* const (&sp)[2], int t, int64_t i) {
                 Chunk<TZ, E> zz;
                 Chunk<TP, E> pp;
                 chunk_load(zz, reinterpret_cast<const TZ*>(sp[0]), t);
                 if (!first) chunk_load(pp, reinterpret_cast<const TP*>(sp[1]), t);
                 p_chunk<PS, UZ, false>(c, beta, first, shadow32, ph, zz, pp, i);
               },
               [&](int64_t i) {
                 Chunk<TZ, E> zz;
                 Chunk<TP, E> pp;
                 chunk_load(zz, z, i);
                 if (!first) chunk_load(pp, pin, i);
                 p_chunk<PS, UZ, false>(c, beta, first, shadow32, ph, zz, pp, i);
               });
}

// ------------------------------------------------------------------ a5 ----------------------
template <int UR, int UZ>
__device__ __forceinline__ double phase_xr_staged(const Ctx& c, const double alpha, double* x, unsigned char* smem) {
  using T = XRT<UR, UZ>;
  using TZ = typename T::TZ;
  using TR = typename T::TR;
  constexpr int E = T::E;
  const TZ* p = pvec<UZ>(c);
  const TR* q = qvec<UR>(c);
  const TR* r = rvec<UR>(c);
  const char* in[4] = {reinterpret_cast<const char*>(x), reinterpret_cast<const char*>(p), reinterpret_cast<const char*>(q),
                       reinterpret_cast<const char*>(r)};
  const int es[4] = {8, (int)sizeof(TZ), (int)sizeof(TR), (int)sizeof(TR)};
  const bool use[4] = {true, true, true, true};
  double sum = 0.0;
  vp_run<E, 4>(c, in, es, use, smem,
               [&](const unsigned char* const (&sp)[4], int t, int64_t i) {
                 Chunk<double, E> xx;
                 Chunk<TZ, E> pp;
                 Chunk<TR, E> qq, rr;
                 chunk_load(xx, reinterpret_cast<const double*>(sp[0]), t);
                 chunk_load(pp, reinterpret_cast<const TZ*>(sp[1]), t);
                 chunk_load(qq, reinterpret_cast<const TR*>(sp[2]), t);
                 chunk_load(rr, reinterpret_cast<const TR*>(sp[3]), t);
                 xr_chunk<UR, UZ>(c, alpha, x, xx, pp, qq, rr, i, sum);
               },
               [&](int64_t i) {
                 Chunk<double, E> xx;
                 Chunk<TZ, E> pp;
                 Chunk<TR, E> qq, rr;
                 x_chunk_load<E>(xx, x, i, c.n);
                 chunk_load(pp, p, i);
                 chunk_load(qq, q, i);
                 chunk_load(rr, r, i);
                 xr_chunk<UR, UZ>(c, alpha, x, xx, pp, qq, rr, i, sum);
               });
  return sum;
}

// ------------------------------------------------------------------ lagged a5 + a2 ----------
template <int UR, int URN, int UZ, int UZN>
__device__ __forceinline__ void phase_xrz_staged(const Ctx& c, const double alpha, const double omega_n, double* x, unsigned char* smem,
                                                 double& sum_rr, double& sum_rz) {
  using T = XRZT<UR, URN, UZ, UZN>;
  using TP = typename T::TP;
  using TR = typename T::TR;
  using TD = typename T::TD;
  constexpr int E = T::E;
  const TP* p = pvec<UZ>(c);
  const TR* q = qvec<UR>(c);
  const TR* rin = rvec<UR>(c);
  const TD* dinv = T::dinv(c);
  const char* in[5] = {reinterpret_cast<const char*>(x), reinterpret_cast<const char*>(p), reinterpret_cast<const char*>(q),
                       reinterpret_cast<const char*>(rin), reinterpret_cast<const char*>(dinv)};
  const int es[5] = {8, (int)sizeof(TP), (int)sizeof(TR), (int)sizeof(TR), (int)sizeof(TD)};
  const bool use[5] = {true, true, true, true, true};
  double srr = 0.0, srz = 0.0;
  vp_run<E, 5>(c, in, es, use, smem,
               [&](const unsigned char* const (&sp)[5], int t, int64_t i) {
                 Chunk<double, E> xx;
                 Chunk<TP, E> pp;
                 Chunk<TR, E> qq, rr;
                 Chunk<TD, E> dd;
                 chunk_load(xx, reinterpret_cast<const double*>(sp[0]), t);
                 chunk_load(pp, reinterpret_cast<const TP*>(sp[1]), t);
                 chunk_load(qq, reinterpret_cast<const TR*>(sp[2]), t);
                 chunk_load(rr, reinterpret_cast<const TR*>(sp[3]), t);
                 chunk_load(dd, reinterpret_cast<const TD*>(sp[4]), t);
                 xrz_chunk<UR, URN, UZ, UZN>(c, alpha, omega_n, x, xx, pp, qq, rr, dd, i, srr, srz);
               },
               [&](int64_t i) {
                 Chunk<double, E> xx;
                 Chunk<TP, E> pp;
                 Chunk<TR, E> qq, rr;
                 Chunk<TD, E> dd;
                 x_chunk_load<E>(xx, x, i, c.n);
                 chunk_load(pp, p, i);
                 chunk_load(qq, q, i);
                 chunk_load(rr, rin, i);
                 chunk_load(dd, dinv, i);
                 xrz_chunk<UR, URN, UZ, UZN>(c, alpha, omega_n, x, xx, pp, qq, rr, dd, i, srr, srz);
               });
  sum_rr = srr;
  sum_rz = srz;
}

// ------------------------------------------------------------------ precision dispatch ------
__device__ __forceinline__ double dispatch_z_staged(const Ctx& c, int rs, int ur, int uz, double omega, unsigned char* smem) {
  if (rs == P64 && ur == P64) {
    if (uz == P64) return phase_z_staged<P64, P64, P64>(c, omega, smem);
    if (uz == P32) return phase_z_staged<P64, P64, P32>(c, omega, smem);
    return phase_z_staged<P64, P64, P16>(c, omega, smem);
  }
  if (rs == P64 && ur == P32) {
    if (uz == P64) return phase_z_staged<P64, P32, P64>(c, omega, smem);
    if (uz == P32) return phase_z_staged<P64, P32, P32>(c, omega, smem);
    return phase_z_staged<P64, P32, P16>(c, omega, smem);
  }
  if (uz == P64) return phase_z_staged<P32, P32, P64>(c, omega, smem);
  if (uz == P32) return phase_z_staged<P32, P32, P32>(c, omega, smem);
  return phase_z_staged<P32, P32, P16>(c, omega, smem);
}
__device__ __forceinline__ void dispatch_p_staged(const Ctx& c, int ps, int uz, int ur, double beta, bool first, unsigned char* smem) {
  if (uz == P64) phase_p_staged<P64, P64>(c, beta, first, ur == P32, smem);
  else if (uz == P32) {
    if (ps == P64) phase_p_staged<P64, P32>(c, beta, first, false, smem);
    else phase_p_staged<P32, P32>(c, beta, first, false, smem);
  } else {
    if (ps == P64) phase_p_staged<P64, P16>(c, beta, first, false, smem);
    else if (ps == P32) phase_p_staged<P32, P16>(c, beta, first, false, smem);
    else phase_p_staged<P16, P16>(c, beta, first, false, smem);
  }
}
__device__ __forceinline__ double dispatch_xr_staged(const Ctx& c, int ur, int uz, double alpha, double* x, unsigned char* smem) {
  if (ur == P64) {
    if (uz == P64) return phase_xr_staged<P64, P64>(c, alpha, x, smem);
    if (uz == P32) return phase_xr_staged<P64, P32>(c, alpha, x, smem);
    return phase_xr_staged<P64, P16>(c, alpha, x, smem);
  }
  if (uz == P64) return phase_xr_staged<P32, P64>(c, alpha, x, smem);
  if (uz == P32) return phase_xr_staged<P32, P32>(c, alpha, x, smem);
  return phase_xr_staged<P32, P16>(c, alpha, x, smem);
}
template <int UR, int URN>
__device__ __forceinline__ void dispatch_xrz_z_staged(const Ctx& c, int uz, int uzn, double alpha, double omega_n, double* x,
                                                      unsigned char* smem, double& rr, double& rz) {
  if (uz == P64) {
    if (uzn == P64) phase_xrz_staged<UR, URN, P64, P64>(c, alpha, omega_n, x, smem, rr, rz);
    else if (uzn == P32) phase_xrz_staged<UR, URN, P64, P32>(c, alpha, omega_n, x, smem, rr, rz);
    else phase_xrz_staged<UR, URN, P64, P16>(c, alpha, omega_n, x, smem, rr, rz);
  } else if (uz == P32) {
    if (uzn == P32) phase_xrz_staged<UR, URN, P32, P32>(c, alpha, omega_n, x, smem, rr, rz);
    else phase_xrz_staged<UR, URN, P32, P16>(c, alpha, omega_n, x, smem, rr, rz);
  } else {
    phase_xrz_staged<UR, URN, P16, P16>(c, alpha, omega_n, x, smem, rr, rz);
  }
}
__device__ __forceinline__ void dispatch_xrz_staged(const Ctx& c, int ur, int urn, int uz, int uzn, double alpha, double omega_n,
                                                    double* x, unsigned char* smem, double& rr, double& rz) {
  if (ur == P64 && urn == P64) dispatch_xrz_z_staged<P64, P64>(c, uz, uzn, alpha, omega_n, x, smem, rr, rz);
  else if (ur == P64) dispatch_xrz_z_staged<P64, P32>(c, uz, uzn, alpha, omega_n, x, smem, rr, rz);
  else dispatch_xrz_z_staged<P32, P32>(c, uz, uzn, alpha, omega_n, x, smem, rr, rz);
}

// ------------------------------------------------------------------ loop kernels (staged) ---
// Same contracts as k_z / k_p / k_xr / k_xrz of kernels.cuh (which they replace in the loop when the handle's
// vec_kernel is STAGED); grid = one block per SM, dynamic shared memory kVpSmemBytes.
__global__ void __launch_bounds__(kVpThreads, 1) k_z_st(const Ctx c) {
  extern __shared__ __align__(128) unsigned char vp_smem[];
  __shared__ double red[32];
  DevState* s = c.st;
  pdl_launch_dependents();
  vp_init(vp_smem);
  pdl_wait();
  if (s->done) return;
  const double v = dispatch_z_staged(c, s->r_store, s->ur, s->uz, s->omega, vp_smem);
  grid_reduce<kVpThreads>(v, c.partials + 0 * kMaxGrid, &s->counter[0], blockIdx.x, gridDim.x, red,
                          [&](double tot) { if (c.sh != nullptr) shard_reduce_point(c, kEpiRho, tot, 0.0); else epi_rho(epi_ctx(c), tot); });
}

__global__ void __launch_bounds__(kVpThreads, 1) k_p_st(const Ctx c) {
  extern __shared__ __align__(128) unsigned char vp_smem[];
  const DevState* s = c.st;
  pdl_launch_dependents();
  vp_init(vp_smem);
  pdl_wait();
  if (s->done) return;
  dispatch_p_staged(c, s->p_store, s->uz, s->ur, s->beta, s->k == 0, vp_smem);
}

__global__ void __launch_bounds__(kVpThreads, 1) k_xr_st(const Ctx c) {
  extern __shared__ __align__(128) unsigned char vp_smem[];
  __shared__ double red[32];
  DevState* s = c.st;
  pdl_launch_dependents();
  vp_init(vp_smem);
  pdl_wait();
  if (s->done) {
    if (blockIdx.x == 0 && threadIdx.x == 0) set_loop_cond(epi_ctx(c), 0);
    return;
  }
  const double v = dispatch_xr_staged(c, s->ur, s->uz, s->alpha, s->x, vp_smem);
  grid_reduce<kVpThreads>(v, c.partials + 2 * kMaxGrid, &s->counter[2], blockIdx.x, gridDim.x, red,
                          [&](double tot) { if (c.sh != nullptr) shard_reduce_point(c, kEpiDelta, tot, 0.0); else epi_delta(epi_ctx(c), tot); });
}

__global__ void __launch_bounds__(kVpThreads, 1) k_xrz_st(const Ctx c) {
  extern __shared__ __align__(128) unsigned char vp_smem[];
  __shared__ double red[32];
  DevState* s = c.st;
  pdl_launch_dependents();
  vp_init(vp_smem);
  pdl_wait();
  if (s->done) {
    if (blockIdx.x == 0 && threadIdx.x == 0) set_loop_cond(epi_ctx(c), 0);
    return;
  }
  double rr = 0.0, rz = 0.0;
  dispatch_xrz_staged(c, s->ur, s->ur_n, s->uz, s->uz_n, s->alpha, s->omega_n, s->x, vp_smem, rr, rz);
  grid_reduce2<kVpThreads>(rr, rz, c.partials + 2 * kMaxGrid, &s->counter[2], blockIdx.x, gridDim.x, red, [&](double t0, double t1) {
    if (c.sh != nullptr) shard_reduce_point(c, kEpiDeltaLagged, t0, t1); else epi_delta_lagged(epi_ctx(c), t0, t1);
  });
}

}  // namespace amp
