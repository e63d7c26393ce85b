// spmv.cuh — step a4 of the loop: q = A p in u_r and gamma = q^T p (Alg 4.1 lines 11-13,
// PAPER.md:288-291; the paper also fuses the inner product into its Ax kernel, :537).
//
// CSR, "warp-private bulk pipeline, lanes-per-row" design for sm_100a:
//  * Rows are statically partitioned over all warps of the grid in contiguous ranges of equal
//    cost (stored entries + rows); each range is cut into tiles of <= tile_cap entries and
//    <= kTileRows rows, a whole number of warp passes each (warp_tile / tile_desc, built in
//    amp_pcg_create).
//  * Every warp runs its own ring of kStages shared-memory stages, each guarded by its own
//    mbarrier.  Per tile, lane 0 issues three cp.async.bulk (TMA, 1-D) copies — values, column
//    indices, row pointers — so the HBM stream is fully coalesced whatever the row lengths are,
//    costs no registers, and runs ahead of the arithmetic.  Warps never meet at a block barrier.
//  * L = lanes_per_row lanes own a row: they read their entries from shared memory, gather p_j
//    (adjacent lanes hold adjacent rows, so for banded matrices one gather instruction touches
//    few sectors), accumulate an fma chain in the working precision in registers (L = 1: in CSR
//    order), combine over the L lanes by shuffles, write q_i and add p_i q_i (stored q_i, FP64)
//    to the lane's gamma partial.
//  * A row longer than the tile capacity is a tile of its own, streamed straight from global.
// UR = P64: FP64 values, FP64 products and sums.  UR = P32: FP32 value copy, p_j converted to
// FP32 (exact from FP16/FP32 storage), FP32 products and sums (q computed and
// stored in u_r).
#pragma once
#include "common.cuh"

namespace amp {

constexpr int kStageValsBytes = (kTileNnz + 8) * 8;
constexpr int kStageColsBytes = (kTileNnz + 8) * 4;
constexpr int kStageRpBytes = (kTileRows + 8) * 4;
constexpr int kStageBytes = ((kStageValsBytes + kStageColsBytes + kStageRpBytes + 127) / 128) * 128;
constexpr int kSpmvRingBytes = kSpmvWarps * kStages * kStageBytes;
constexpr int kSpmvSmemBytes = kSpmvRingBytes + kSpmvWarps * kStages * 8;  // + mbarriers
#ifndef AMP_GATHER_BATCH
#define AMP_GATHER_BATCH 8
#endif
constexpr int kGatherBatch = AMP_GATHER_BATCH;  // independent gathers in flight per lane
static_assert(kSpmvSmemBytes <= 227 * 1024, "SpMV ring does not fit in shared memory");

template <int UR> struct SpmvT;
template <> struct SpmvT<P64> { using A = double; };
template <> struct SpmvT<P32> { using A = float; };

// ------------------------------------------------------------------ mbarrier / bulk copy ----
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_inval(uint64_t* bar) {
  asm volatile("mbarrier.inval.shared::cta.b64 [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t* bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
  uint32_t ok;
  do {
    asm volatile("{\n .reg .pred p;\n mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n selp.u32 %0, 1, 0, p;\n}"
                 : "=r"(ok) : "r"(smem_u32(bar)), "r"(parity) : "memory");
  } while (!ok);
}
// 1-D bulk copy global -> shared (16-byte aligned addresses, size a multiple of 16), completion on bar
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, uint32_t bytes, uint64_t* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
               ::"r"(smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}
// order this thread's generic-proxy accesses to shared memory before later async-proxy (bulk copy) writes
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

template <int UR> __device__ __forceinline__ const typename SpmvT<UR>::A* mat_vals(const Ctx& c);
template <> __device__ __forceinline__ const double* mat_vals<P64>(const Ctx& c) { return c.vals64; }
template <> __device__ __forceinline__ const float* mat_vals<P32>(const Ctx& c) { return c.vals32; }

template <bool COH> __device__ __forceinline__ double gatherA(double, const double* p, int j) { return gather64<COH>(p, j); }
template <bool COH> __device__ __forceinline__ double gatherA(double, const float* p, int j) { return gather64<COH>(p, j); }
template <bool COH> __device__ __forceinline__ double gatherA(double, const __half* p, int j) { return gather64<COH>(p, j); }
template <bool COH> __device__ __forceinline__ float gatherA(float, const double* p, int j) { return gather32<COH>(p, j); }
template <bool COH> __device__ __forceinline__ float gatherA(float, const float* p, int j) { return gather32<COH>(p, j); }
template <bool COH> __device__ __forceinline__ float gatherA(float, const __half* p, int j) { return gather32<COH>(p, j); }

// Issue the three bulk copies of tile [r0,r1) x [e0,e1) into one stage (one lane).  Element
// ranges are widened to multiples of 4 entries / rows so every address and size is 16-byte
// aligned; the (at most 3) entries past the last multiple of 4 of the whole arrays are fetched
// with plain loads because the borrowed CSR arrays are not padded.  A long row (more entries
// than a stage holds) only completes the barrier phase: it is streamed from global memory.
template <int UR>
__device__ __forceinline__ void spmv_issue_tile(const Ctx& c, int t, unsigned char* stage, uint64_t* bar) {
  using A = typename SpmvT<UR>::A;
  const int2 d0 = c.tile_desc[t], d1 = c.tile_desc[t + 1];
  const int r0 = d0.x, e0 = d0.y, r1 = d1.x, e1 = d1.y;
  if (e1 - e0 > kTileNnz) {
    mbar_arrive_expect_tx(bar, 0u);
    return;
  }
  const int ea = e0 & ~3;
  const int nbody = (int)(c.nnz & ~(int64_t)3);
  int eb = (e1 + 3) & ~3;
  if (eb > nbody) eb = nbody;
  A* vs = reinterpret_cast<A*>(stage);
  int* cs = reinterpret_cast<int*>(stage + kStageValsBytes);
  int* rs = reinterpret_cast<int*>(stage + kStageValsBytes + kStageColsBytes);
  const A* gv = mat_vals<UR>(c);
  bool tail = false;
  for (int e = (eb > ea ? eb : ea); e < e1; ++e) {  // array tail (last tile of the matrix only)
    vs[e - ea] = gv[e];
    cs[e - ea] = c.colidx[e];
    tail = true;
  }
  if (tail) fence_proxy_async();
  const int r0a = r0 & ~3;
  const int nr = ((r1 + 1 - r0a) + 3) & ~3;  // rowptr_pad is padded, so this never overruns
  const uint32_t cnt = eb > ea ? (uint32_t)(eb - ea) : 0u;
  mbar_arrive_expect_tx(bar, cnt * (uint32_t)(sizeof(A) + 4) + (uint32_t)nr * 4u);
  if (cnt) {
    bulk_g2s(vs, gv + ea, cnt * (uint32_t)sizeof(A), bar);
    bulk_g2s(cs, c.colidx + ea, cnt * 4u, bar);
  }
  bulk_g2s(rs, c.rowptr_pad + r0a, (uint32_t)nr * 4u, bar);
}

// COH = true: p is written earlier in the same (persistent) kernel, so it is gathered with
// plain coherent loads after the grid barrier instead of the read-only (ld.global.nc) path.
// Returns this thread's part of gamma = sum_i p_i q_i.
template <int UR, bool COH, int L, class PT>
__device__ __forceinline__ double phase_spmv(const Ctx& c, const PT* p, typename Store<UR>::T* q, int bid, int nb,
                                             unsigned char* smem_raw) {
  using A = typename SpmvT<UR>::A;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int gw = bid * kSpmvWarps + warp;  // global warp id: owns tiles [t_begin, t_end)
  unsigned char* ring = smem_raw + warp * (kStages * kStageBytes);
  uint64_t* bars = reinterpret_cast<uint64_t*>(smem_raw + kSpmvRingBytes) + warp * kStages;
  constexpr int rows_per_pass = 32 / L;
  const int sub = lane % L, rl = lane / L;
  const int t_begin = c.warp_tile[gw], t_end = c.warp_tile[gw + 1];
  double gsum = 0.0;
  if (t_begin >= t_end) return gsum;

  if (lane == 0) {
#pragma unroll
    for (int s = 0; s < kStages; ++s) mbar_init(bars + s, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
#pragma unroll
    for (int s = 0; s < kStages; ++s)
      if (t_begin + s < t_end) spmv_issue_tile<UR>(c, t_begin + s, ring + s * kStageBytes, bars + s);
  }
  __syncwarp();

  for (int t = t_begin; t < t_end; ++t) {
    const int it = t - t_begin;
    const int slot = it % kStages;
    const int2 d0 = c.tile_desc[t], d1 = c.tile_desc[t + 1];
    const int r0 = d0.x, e0 = d0.y, nrows = d1.x - d0.x, e1 = d1.y;
    unsigned char* stage = ring + slot * kStageBytes;
    mbar_wait(bars + slot, (uint32_t)((it / kStages) & 1));

    if (e1 - e0 > kTileNnz) {  // one long row: warp-strided accumulation straight from global
      const A* gv = mat_vals<UR>(c);
      A acc = 0;
      for (int e = e0 + lane; e < e1; e += 32) acc = fma(gv[e], gatherA<COH>(A(0), p, c.colidx[e]), acc);
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
      if (lane == 0) {
        q[r0] = acc;
        gsum = fma(gather64<COH>(p, r0), (double)acc, gsum);
      }
    } else {
      const A* vs = reinterpret_cast<const A*>(stage);
      const int* cs = reinterpret_cast<const int*>(stage + kStageValsBytes);
      const int* rs = reinterpret_cast<const int*>(stage + kStageValsBytes + kStageColsBytes) + (r0 - (r0 & ~3));
      const int ea = e0 & ~3;
      // L lanes per row: each lane reads its entries from shared memory, gathers p_j (the
      // rows of a warp are adjacent, so for banded matrices the gathers of one instruction fall
      // into few sectors), and accumulates an fma chain in the working precision (L = 1: in
      // CSR order); the L partial sums are combined by shuffles.
      for (int rb = 0; rb < nrows; rb += rows_per_pass) {
        const int row = rb + rl;
        A acc = 0;
        double pi = 0.0;
        if (row < nrows) {
          const int jb = rs[row] - ea, je = rs[row + 1] - ea;
          if (sub == 0) pi = gather64<COH>(p, r0 + row);
          for (int j0 = jb + sub; j0 < je; j0 += kGatherBatch * L) {
            A a[kGatherBatch], xg[kGatherBatch];
            int cj[kGatherBatch];
#pragma unroll
            for (int u = 0; u < kGatherBatch; ++u) {
              const int jj = j0 + u * L;
              const bool ok = jj < je;
              cj[u] = ok ? cs[jj] : (r0 + row);
              a[u] = ok ? vs[jj] : A(0);
            }
#pragma unroll
            for (int u = 0; u < kGatherBatch; ++u) xg[u] = gatherA<COH>(A(0), p, cj[u]);
#pragma unroll
            for (int u = 0; u < kGatherBatch; ++u) acc = fma(a[u], xg[u], acc);
          }
        }
#pragma unroll
        for (int o = L >> 1; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
        if (row < nrows && sub == 0) {
          q[r0 + row] = acc;
          gsum = fma(pi, (double)acc, gsum);
        }
      }
    }

    // every lane is done reading the stage: hand it back to the producer
    __syncwarp();
    if (lane == 0 && t + kStages < t_end) spmv_issue_tile<UR>(c, t + kStages, stage, bars + slot);
    __syncwarp();
  }

  if (lane == 0) {
#pragma unroll
    for (int s = 0; s < kStages; ++s) mbar_inval(bars + s);
  }
  return gsum;
}

}  // namespace amp
