// spmv.cuh — step a4 of the loop: q = A p in u_r and gamma = q^T p (Alg 4.1 lines 11-13,
// PAPER.md:288-291; the paper also fuses the inner product into its Ax kernel, :537).
//
// CSR, "bulk-staged, lanes-per-row" design for sm_100a:
//  * Rows are statically partitioned over the grid in contiguous ranges of equal cost
//    (stored entries + rows) and each range is cut into tiles of <= kTileNnz entries and
//    <= kTileRows rows (block_tile / tile_row, built in amp_pcg_create).
//  * Per tile one elected thread issues three cp.async.bulk (TMA, 1-D) copies — values, column
//    indices, row pointers — into a shared-memory stage and all threads wait on the stage's
//    mbarrier.  kStages stages form a ring, so the HBM stream of tile i+1.. runs under the
//    arithmetic of tile i: streaming is fully coalesced and independent of the row lengths,
//    and costs no registers.
//  * L = lanes_per_row lanes own a row: they read their entries from shared memory, gather p_j
//    (coalesced across the rows of a warp for banded matrices), accumulate an fma chain in the
//    working precision in registers, combine over the L lanes by shuffles, write q_i and add
//    p_i q_i (stored q_i, FP64) to the block's gamma partial.
//  * A row longer than kTileNnz is a tile of its own and is streamed directly from global memory.
// UR = P64: FP64 values, FP64 fma chain.  UR = P32: FP32 value copy, p_j converted to FP32
// (exact from FP16/FP32 storage), FP32 fma chain (q computed and stored in u_r).
#pragma once
#include "common.cuh"

namespace amp {

constexpr int kStageValsBytes = (kTileNnz + 8) * 8;
constexpr int kStageColsBytes = (kTileNnz + 8) * 4;
constexpr int kStageRpBytes = (kTileRows + 8) * 4;
constexpr int kStageBytes = ((kStageValsBytes + kStageColsBytes + kStageRpBytes + 127) / 128) * 128;
constexpr int kStages = 2;
constexpr int kSpmvSmemBytes = kStages * kStageBytes + 64;  // + mbarriers
constexpr int kGatherBatch = 8;                             // independent gathers in flight per lane

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

template <int UR> __device__ __forceinline__ const typename SpmvT<UR>::A* mat_vals(const Ctx& c);
template <> __device__ __forceinline__ const double* mat_vals<P64>(const Ctx& c) { return c.vals64; }
template <> __device__ __forceinline__ const float* mat_vals<P32>(const Ctx& c) { return c.vals32; }

template <bool COH> __device__ __forceinline__ double gatherA(double, const double* p, int j) { return gather64<COH>(p, j); }
template <bool COH> __device__ __forceinline__ double gatherA(double, const float* p, int j) { return gather64<COH>(p, j); }
template <bool COH> __device__ __forceinline__ double gatherA(double, const __half* p, int j) { return gather64<COH>(p, j); }
template <bool COH> __device__ __forceinline__ float gatherA(float, const double* p, int j) { return gather32<COH>(p, j); }
template <bool COH> __device__ __forceinline__ float gatherA(float, const float* p, int j) { return gather32<COH>(p, j); }
template <bool COH> __device__ __forceinline__ float gatherA(float, const __half* p, int j) { return gather32<COH>(p, j); }

// Issue the three bulk copies of tile t into stage memory (one thread).  Element ranges are
// widened to multiples of 4 entries / rows so every address and size is 16-byte aligned; the
// (at most 3) entries past the last multiple of 4 of the whole arrays are fetched with plain
// loads because the borrowed CSR arrays are not padded.
template <int UR>
__device__ __forceinline__ void spmv_issue_tile(const Ctx& c, int t, unsigned char* stage, uint64_t* bar) {
  using A = typename SpmvT<UR>::A;
  const int r0 = c.tile_row[t], r1 = c.tile_row[t + 1];
  const int e0 = c.rowptr[r0], e1 = c.rowptr[r1];
  const int ea = e0 & ~3;
  const int nbody = (int)(c.nnz & ~(int64_t)3);
  int eb = (e1 + 3) & ~3;
  if (eb > nbody) eb = nbody;
  A* vs = reinterpret_cast<A*>(stage);
  int* cs = reinterpret_cast<int*>(stage + kStageValsBytes);
  int* rs = reinterpret_cast<int*>(stage + kStageValsBytes + kStageColsBytes);
  const A* gv = mat_vals<UR>(c);
  for (int e = (eb > ea ? eb : ea); e < e1; ++e) {  // array tail (last tile only)
    vs[e - ea] = gv[e];
    cs[e - ea] = c.colidx[e];
  }
  const int r0a = r0 & ~3;
  const int nr = ((r1 + 1 - r0a) + 3) & ~3;  // rowptr_pad is padded, so this never overruns
  const uint32_t bytes_e = eb > ea ? (uint32_t)(eb - ea) : 0u;
  const uint32_t tx = bytes_e * (uint32_t)(sizeof(A) + 4) + (uint32_t)nr * 4u;
  mbar_arrive_expect_tx(bar, tx);
  if (bytes_e) {
    bulk_g2s(vs, gv + ea, bytes_e * (uint32_t)sizeof(A), bar);
    bulk_g2s(cs, c.colidx + ea, bytes_e * 4u, bar);
  }
  bulk_g2s(rs, c.rowptr_pad + r0a, (uint32_t)nr * 4u, bar);
}

// COH = true: p is written earlier in the same (persistent) kernel, so it is gathered with
// plain coherent loads after the grid barrier instead of the read-only (ld.global.nc) path.
template <int UR, bool COH, class PT>
__device__ __forceinline__ double phase_spmv(const Ctx& c, const PT* p, typename Store<UR>::T* q, int bid, int nb,
                                             unsigned char* smem_raw, double* red_sm) {
  using A = typename SpmvT<UR>::A;
  uint64_t* bars = reinterpret_cast<uint64_t*>(smem_raw + kStages * kStageBytes);
  const int tid = threadIdx.x;
  const int L = c.lanes_per_row;
  const int sub = tid % L, rl = tid / L, rows_per_pass = kSpmvThreads / L;
  const int t_begin = c.block_tile[bid], t_end = c.block_tile[bid + 1];
  double gsum = 0.0;

  if (tid == 0) {
#pragma unroll
    for (int s = 0; s < kStages; ++s) mbar_init(bars + s, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();

  // producer cursor (meaningful in thread 0 only): next tile to look at, staged tiles issued so far
  int ti = t_begin, n_issued = 0;
  auto is_long = [&](int t) { return c.rowptr[c.tile_row[t + 1]] - c.rowptr[c.tile_row[t]] > kTileNnz; };
  auto issue_next = [&]() {
    while (ti < t_end && is_long(ti)) ++ti;
    if (ti < t_end) {
      const int slot = n_issued % kStages;
      spmv_issue_tile<UR>(c, ti, smem_raw + slot * kStageBytes, bars + slot);
      ++n_issued;
      ++ti;
    }
  };
  if (tid == 0) {
    for (int s = 0; s < kStages; ++s) issue_next();
  }

  int n_consumed = 0;
  for (int t = t_begin; t < t_end; ++t) {
    const int r0 = c.tile_row[t], r1 = c.tile_row[t + 1];
    const int nrows = r1 - r0;
    const int e0 = c.rowptr[r0], e1 = c.rowptr[r1];

    if (e1 - e0 > kTileNnz) {  // one long row: block-wide strided accumulation straight from global
      const A* gv = mat_vals<UR>(c);
      A acc = 0;
      for (int e = e0 + tid; e < e1; e += kSpmvThreads) acc = fma(gv[e], gatherA<COH>(A(0), p, c.colidx[e]), acc);
      const double tot = block_sum<kSpmvThreads>((double)acc, red_sm);
      if (tid == 0) {
        const A qs = (A)tot;
        q[r0] = qs;
        gsum = fma(gather64<COH>(p, r0), (double)qs, gsum);
      }
      __syncthreads();
      continue;
    }

    const int slot = n_consumed % kStages;
    unsigned char* stage = smem_raw + slot * kStageBytes;
    mbar_wait(bars + slot, (uint32_t)((n_consumed / kStages) & 1));
    const A* vs = reinterpret_cast<const A*>(stage);
    const int* cs = reinterpret_cast<const int*>(stage + kStageValsBytes);
    const int* rs = reinterpret_cast<const int*>(stage + kStageValsBytes + kStageColsBytes) + (r0 - (r0 & ~3));
    const int ea = e0 & ~3;

    for (int rb = 0; rb < nrows; rb += rows_per_pass) {
      const int row = rb + rl;
      A acc = 0;
      if (row < nrows) {
        const int jb = rs[row] - ea, je = rs[row + 1] - ea;
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
      for (int o = L >> 1; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
      if (row < nrows && sub == 0) {
        q[r0 + row] = acc;
        gsum = fma(gather64<COH>(p, r0 + row), (double)acc, gsum);
      }
    }
    __syncthreads();  // every thread is done reading this stage
    ++n_consumed;
    if (tid == 0) issue_next();
  }

  __syncthreads();
  if (tid == 0) {
#pragma unroll
    for (int s = 0; s < kStages; ++s) mbar_inval(bars + s);
  }
  return gsum;
}

}  // namespace amp
