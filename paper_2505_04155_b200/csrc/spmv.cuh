// spmv.cuh — step a4 of the loop: q = A p in u_r and gamma = q^T p (Alg 4.1 lines 11-13,
// PAPER.md:288-291; the paper also fuses the inner product into its Ax kernel, :537).
//
// Matrix format: SELL-32 ("sliced ELLPACK", slice height = warp width), repacked once from the
// caller's CSR in amp_pcg_create and owned by the handle (indices, FP64 values and the FP32-rounded
// value copy of the u_r = FP32 phase).
//  * A slice is 32 consecutive rows (of the row order `perm`: identity, or rows sorted by length
//    inside windows of 1024 when the lengths vary enough for padding to cost > 3 %); lane l of a
//    warp owns row l of the slice.
//  * The slice width w = longest row of the slice; shorter rows are padded with value 0 and a valid
//    column.  w is cut as 4a + 2b + c and stored as a blocks of [lane][4] entries, then b block of
//    [lane][2], then c block of [lane][1], so a lane reads its row with 128-bit loads (64-/32-bit
//    for the remainder) and every warp-wide load is one contiguous, fully used 512-byte (256-,
//    128-byte) run: no padding beyond the slice maximum, 4 B per SLICE of table (the cumulative
//    widths) instead of CSR's 4 B per ROW of row pointer.  FP64 values use [lane][2] blocks
//    throughout (a quad = two consecutive pair blocks).
//  * Column indices come in three forms (ColSrc below): diagonal-aligned slices need none at all
//    (col = row + one offset per entry position), banded matrices get 16-bit offsets, the rest
//    32-bit indices.
//  * Entries keep their CSR order within the row (aligned slices interleave explicit zeros, which
//    leave an fma chain unchanged) and each lane accumulates ONE fma chain in the working
//    precision, so q_i is bit-identical to a sequential CSR-order fma loop.
//  * Matrix data is streamed with ld.global.cs (evict-first) so that it does not displace the
//    vectors from L2 (measured: 57 vs 65 us per iteration on c2 against default caching); the value
//    stream of wide slices is prefetched into L2 two passes ahead; p is gathered through the
//    read-only path (L1-cached) — adjacent lanes hold adjacent rows, so for banded matrices one
//    gather instruction touches one or two lines.
//  * Rows longer than max(256, 8 nnz/n) are left out of the slices (length 0 there) and summed
//    straight from the borrowed CSR arrays by a whole block each.
// UR = P64: FP64 values, FP64 products and sums.  UR = P32: FP32 value copy, p_j converted to
// FP32 (exact from FP16/FP32 storage), FP32 products and sums (q computed and
// stored in u_r).
#pragma once
#include "common.cuh"

namespace amp {

template <int UR> struct SpmvT;
template <> struct SpmvT<P64> { using A = double; };
template <> struct SpmvT<P32> { using A = float; };

// ------------------------------------------------------------------ SELL-32 addressing ------
// position (in elements, relative to the slice start) of entry k of lane `lane` in a slice of
// width w.  pos32: column indices and FP32 values; pos64: FP64 values.
__host__ __device__ __forceinline__ int64_t sell_pos32(int k, int lane, int w) {
  const int a = w >> 2;
  if (k < 4 * a) return (int64_t)(k >> 2) * 128 + lane * 4 + (k & 3);
  if ((w & 2) && k < 4 * a + 2) return (int64_t)a * 128 + lane * 2 + (k - 4 * a);
  return (int64_t)a * 128 + ((w & 2) ? 64 : 0) + lane;
}
__host__ __device__ __forceinline__ int64_t sell_pos64(int k, int lane, int w) {
  const int a = w >> 2;
  if (k < 4 * a) return (int64_t)(k >> 2) * 128 + ((k >> 1) & 1) * 64 + lane * 2 + (k & 1);
  if ((w & 2) && k < 4 * a + 2) return (int64_t)a * 128 + lane * 2 + (k - 4 * a);
  return (int64_t)a * 128 + ((w & 2) ? 64 : 0) + lane;
}

// streaming (evict-first) loads of matrix data
#ifndef AMP_SPMV_MATRIX_LOAD
#define AMP_SPMV_MATRIX_LOAD __ldcs
#endif
__device__ __forceinline__ int4 lds_i4(const int32_t* p) { return AMP_SPMV_MATRIX_LOAD(reinterpret_cast<const int4*>(p)); }
__device__ __forceinline__ int2 lds_i2(const int32_t* p) { return AMP_SPMV_MATRIX_LOAD(reinterpret_cast<const int2*>(p)); }
__device__ __forceinline__ int lds_i1(const int32_t* p) { return AMP_SPMV_MATRIX_LOAD(p); }
__device__ __forceinline__ void lds_quad(const float* v, float (&a)[4]) {
  const float4 t = AMP_SPMV_MATRIX_LOAD(reinterpret_cast<const float4*>(v));
  a[0] = t.x; a[1] = t.y; a[2] = t.z; a[3] = t.w;
}
__device__ __forceinline__ void lds_quad(const double* v, double (&a)[4]) {  // v -> first pair block, lane offset applied
  const double2 t0 = AMP_SPMV_MATRIX_LOAD(reinterpret_cast<const double2*>(v));
  const double2 t1 = AMP_SPMV_MATRIX_LOAD(reinterpret_cast<const double2*>(v + 64));
  a[0] = t0.x; a[1] = t0.y; a[2] = t1.x; a[3] = t1.y;
}
__device__ __forceinline__ void lds_pair(const float* v, float (&a)[2]) {
  const float2 t = AMP_SPMV_MATRIX_LOAD(reinterpret_cast<const float2*>(v));
  a[0] = t.x; a[1] = t.y;
}
__device__ __forceinline__ void lds_pair(const double* v, double (&a)[2]) {
  const double2 t = AMP_SPMV_MATRIX_LOAD(reinterpret_cast<const double2*>(v));
  a[0] = t.x; a[1] = t.y;
}

template <int UR> __device__ __forceinline__ const typename SpmvT<UR>::A* sell_vals(const Ctx& c);
template <> __device__ __forceinline__ const double* sell_vals<P64>(const Ctx& c) { return c.sell_vals64; }
template <> __device__ __forceinline__ const float* sell_vals<P32>(const Ctx& c) { return c.sell_vals32; }
template <int UR> __device__ __forceinline__ const typename SpmvT<UR>::A* csr_vals(const Ctx& c);
template <> __device__ __forceinline__ const double* csr_vals<P64>(const Ctx& c) { return c.vals64; }
template <> __device__ __forceinline__ const float* csr_vals<P32>(const Ctx& c) { return c.vals32; }

template <bool COH> __device__ __forceinline__ double gatherA(double, const double* p, int j) { return gather64<COH>(p, j); }
template <bool COH> __device__ __forceinline__ double gatherA(double, const float* p, int j) { return gather64<COH>(p, j); }
template <bool COH> __device__ __forceinline__ double gatherA(double, const __half* p, int j) { return gather64<COH>(p, j); }
template <bool COH> __device__ __forceinline__ float gatherA(float, const double* p, int j) { return gather32<COH>(p, j); }
template <bool COH> __device__ __forceinline__ float gatherA(float, const float* p, int j) { return gather32<COH>(p, j); }
template <bool COH> __device__ __forceinline__ float gatherA(float, const __half* p, int j) { return gather32<COH>(p, j); }

template <class A> struct LaneQ;  // elements a lane owns per 128-bit load of a value block
template <> struct LaneQ<float> { static constexpr int v = 4; };
template <> struct LaneQ<double> { static constexpr int v = 2; };
__device__ __forceinline__ float lds_one(const float* v) { return AMP_SPMV_MATRIX_LOAD(v); }
__device__ __forceinline__ double lds_one(const double* v) { return AMP_SPMV_MATRIX_LOAD(v); }

// ------------------------------------------------------------------ column index sources ----
// CM = 0: 32-bit column indices.
// CM = 1: 16-bit offsets from a per-(slice, entry) base (the smallest column of entry k over the 32
//         rows of the slice, sell_base[w0 + k]); chosen for the whole matrix in create() when every
//         offset fits, which holds for banded matrices: 2 B per entry + 4 B per 32 entries.
// CM = 2: "aligned" slice (chosen per slice in create()): the entries of the 32 rows were placed so
//         that entry k of every row lies on the same diagonal, col = row + sell_base[w0 + k]
//         (rows that lack a diagonal hold an explicit zero there).  No per-entry index is read at
//         all: 4 B per 32 entries.  Typical for stencil / structured-grid matrices.
// The base of entry k is held by lane k % 32 and broadcast by a shuffle.
constexpr int kPrefetchMinWidth = 16;  // groups narrower than this many entries per row are not prefetched
constexpr int kAlignedFlag = (int)0x80000000u;  // bit 31 of sell_wptr[s]: slice s is aligned
constexpr int kUniformFlag = 0x40000000;        // bit 30: slice s is aligned, Ctx::uni_w wide, with the diagonal offsets Ctx::uni_base
constexpr int kWptrFlags = kAlignedFlag | kUniformFlag;
template <int CM> struct ColSrc;
template <> struct ColSrc<0> {
  using RawQ = int4; using RawP = int2; using RawS = int;
  const int32_t* cp;
  __device__ __forceinline__ ColSrc() {}
  __device__ __forceinline__ ColSrc(const Ctx& c, int w0, int, int, int) : cp(c.sell_cols + (int64_t)w0 * 32) {}
  __device__ __forceinline__ void refresh(int, int) {}
  __device__ __forceinline__ RawQ quad(int off, int lane) const { return lds_i4(cp + off + lane * 4); }
  __device__ __forceinline__ RawP pair(int off, int lane) const { return lds_i2(cp + off + lane * 2); }
  __device__ __forceinline__ RawS single(int off, int lane) const { return lds_i1(cp + off + lane); }
  __device__ __forceinline__ void dq(RawQ r, int, int (&j)[4]) const { j[0] = r.x; j[1] = r.y; j[2] = r.z; j[3] = r.w; }
  __device__ __forceinline__ void dp(RawP r, int, int (&j)[2]) const { j[0] = r.x; j[1] = r.y; }
  __device__ __forceinline__ int ds(RawS r, int) const { return r; }
  static __device__ __forceinline__ RawQ zq() { return make_int4(0, 0, 0, 0); }
  static __device__ __forceinline__ RawP zp() { return make_int2(0, 0); }
};
struct ColBase {  // bases of the entries of one slice, 32 at a time, one per lane
  const int32_t* bp;
  int w, blk, bl;
  __device__ __forceinline__ void init(const Ctx& c, int w0, int w_, int lane) {
    bp = c.sell_base + w0; w = w_; blk = 0;
    bl = (lane < w) ? __ldg(bp + lane) : 0;
  }
  // make the bases of entries [32*(k/32), +32) current (slices wider than 32 entries only)
  __device__ __forceinline__ void refresh(int k, int lane) {
    if ((k >> 5) != blk) {
      blk = k >> 5;
      bl = (blk * 32 + lane < w) ? __ldg(bp + blk * 32 + lane) : 0;
    }
  }
  __device__ __forceinline__ int base(int k) const { return __shfl_sync(0xffffffffu, bl, k & 31); }
};
template <> struct ColSrc<1> : ColBase {
  using RawQ = uint2; using RawP = uint32_t; using RawS = uint32_t;
  const uint16_t* cp;
  __device__ __forceinline__ ColSrc() {}
  __device__ __forceinline__ ColSrc(const Ctx& c, int w0, int w_, int lane, int) : cp(c.sell_cols16 + (int64_t)w0 * 32) {
    init(c, w0, w_, lane);
  }
  __device__ __forceinline__ RawQ quad(int off, int lane) const { return __ldcs(reinterpret_cast<const uint2*>(cp + off + lane * 4)); }
  __device__ __forceinline__ RawP pair(int off, int lane) const { return __ldcs(reinterpret_cast<const uint32_t*>(cp + off + lane * 2)); }
  __device__ __forceinline__ RawS single(int off, int lane) const { return (uint32_t)__ldcs(cp + off + lane); }
  __device__ __forceinline__ void dq(RawQ r, int k, int (&j)[4]) const {
    j[0] = base(k) + (int)(r.x & 0xffffu); j[1] = base(k + 1) + (int)(r.x >> 16);
    j[2] = base(k + 2) + (int)(r.y & 0xffffu); j[3] = base(k + 3) + (int)(r.y >> 16);
  }
  __device__ __forceinline__ void dp(RawP r, int k, int (&j)[2]) const {
    j[0] = base(k) + (int)(r & 0xffffu); j[1] = base(k + 1) + (int)(r >> 16);
  }
  __device__ __forceinline__ int ds(RawS r, int k) const { return base(k) + (int)r; }
  static __device__ __forceinline__ RawQ zq() { return make_uint2(0u, 0u); }
  static __device__ __forceinline__ RawP zp() { return 0u; }
};
template <> struct ColSrc<2> : ColBase {
  using RawQ = int; using RawP = int; using RawS = int;  // nothing is loaded per entry
  int row, cmin_, cmax_;
  __device__ __forceinline__ ColSrc() {}
  __device__ __forceinline__ ColSrc(const Ctx& c, int w0, int w_, int lane, int row_)
      : row(row_ < 0 ? 0 : row_), cmin_(c.col_min), cmax_(c.col_max) {
    init(c, w0, w_, lane);
  }
  __device__ __forceinline__ RawQ quad(int, int) const { return 0; }
  __device__ __forceinline__ RawP pair(int, int) const { return 0; }
  __device__ __forceinline__ RawS single(int, int) const { return 0; }
  // explicit zeros of rows that lack diagonal k may point outside the vector (owned entries, halo bands, zero guard):
  // clamp (their value is 0)
  __device__ __forceinline__ int col(int k) const { return min(max(row + base(k), cmin_), cmax_); }
  __device__ __forceinline__ void dq(RawQ, int k, int (&j)[4]) const { j[0] = col(k); j[1] = col(k + 1); j[2] = col(k + 2); j[3] = col(k + 3); }
  __device__ __forceinline__ void dp(RawP, int k, int (&j)[2]) const { j[0] = col(k); j[1] = col(k + 1); }
  __device__ __forceinline__ int ds(RawS, int k) const { return col(k); }
  static __device__ __forceinline__ RawQ zq() { return 0; }
  static __device__ __forceinline__ RawP zp() { return 0; }
};

// One slice of any width: this lane's row sum (one fma chain in stored order = CSR order).
// Full trips of QT quads (all wide loads and all 4 QT gathers of a trip issued before its first fma),
// then ONE tail step for the remaining < QT quads, the pair and the single: branch-free, absent parts
// keep value 0 and a valid column, so the tail also waits for memory once.
template <class A> struct SpmvTrip;  // quads per trip
template <> struct SpmvTrip<float> { static constexpr int QT = 4; };
template <> struct SpmvTrip<double> { static constexpr int QT = 2; };

template <int UR, bool COH, int CM, class PT>
__device__ __forceinline__ typename SpmvT<UR>::A slice_sum(const Ctx& c, const PT* p, int w0, int w, int lane, int row) {
  using A = typename SpmvT<UR>::A;
  using CS = ColSrc<CM>;
  constexpr int LQ = LaneQ<A>::v;
  constexpr int QT = SpmvTrip<A>::QT;
  CS cs(c, w0, w, lane, row);
  const A* vp = sell_vals<UR>(c) + (int64_t)w0 * 32;
  const int a = w >> 2;
  A acc = 0;
  int cq = 0;
  for (; cq + QT <= a; cq += QT) {
    cs.refresh(4 * cq, lane);  // QT divides 8: a trip never straddles a block of 32 bases
    typename CS::RawQ r[QT];
    A v[QT][4];
#pragma unroll
    for (int t = 0; t < QT; ++t) {
      r[t] = cs.quad((cq + t) * 128, lane);
      lds_quad(vp + (cq + t) * 128 + lane * LQ, v[t]);
    }
    A x[QT][4];
#pragma unroll
    for (int t = 0; t < QT; ++t) {
      int j[4];
      cs.dq(r[t], 4 * (cq + t), j);
#pragma unroll
      for (int u = 0; u < 4; ++u) x[t][u] = gatherA<COH>(A(0), p, j[u]);
    }
#pragma unroll
    for (int t = 0; t < QT; ++t) {
#pragma unroll
      for (int u = 0; u < 4; ++u) acc = fma(v[t][u], x[t][u], acc);
    }
  }
  if (cq * 4 == w) return acc;
  {  // tail: up to QT-1 quads, one pair, one single
    cs.refresh(4 * cq, lane);
    const int rem = a - cq;
    const bool hp = (w & 2) != 0, hs = (w & 1) != 0;
    const int tail = a * 128, tail1 = tail + (hp ? 64 : 0);
    typename CS::RawQ rq[QT - 1];
    typename CS::RawP rp = CS::zp();
    typename CS::RawS rs = 0;
    A vq[QT - 1][4], vpair[2] = {A(0), A(0)}, vs = A(0);
#pragma unroll
    for (int t = 0; t < QT - 1; ++t) {
      rq[t] = CS::zq();
      vq[t][0] = vq[t][1] = vq[t][2] = vq[t][3] = A(0);
      if (t < rem) { rq[t] = cs.quad((cq + t) * 128, lane); lds_quad(vp + (cq + t) * 128 + lane * LQ, vq[t]); }
    }
    if (hp) { rp = cs.pair(tail, lane); lds_pair(vp + tail + lane * 2, vpair); }
    if (hs) { rs = cs.single(tail1, lane); vs = lds_one(vp + tail1 + lane); }
    // entries past the real ones decode with k clamped into this block of bases: a valid column
    const int klast = w - 1;
    A xq[QT - 1][4], xp[2], xs;
#pragma unroll
    for (int t = 0; t < QT - 1; ++t) {
      int j[4];
      cs.dq(rq[t], min(4 * (cq + t), klast & ~3), j);
#pragma unroll
      for (int u = 0; u < 4; ++u) xq[t][u] = gatherA<COH>(A(0), p, j[u]);
    }
    {
      int j[2];
      cs.dp(rp, min(4 * a, klast & ~1), j);
      xp[0] = gatherA<COH>(A(0), p, j[0]);
      xp[1] = gatherA<COH>(A(0), p, j[1]);
      xs = gatherA<COH>(A(0), p, cs.ds(rs, klast));
    }
#pragma unroll
    for (int t = 0; t < QT - 1; ++t) {
#pragma unroll
      for (int u = 0; u < 4; ++u) acc = fma(vq[t][u], xq[t][u], acc);
    }
    acc = fma(vpair[0], xp[0], acc);
    acc = fma(vpair[1], xp[1], acc);
    acc = fma(vs, xs, acc);
  }
  return acc;
}

// G consecutive narrow slices (every width <= 7: one quad, one pair, one single at most) at once.
// Branch-free: absent parts keep offset 0 and value 0, so all matrix loads of the group are issued
// (predicated) before the first gather and all 7 G gathers before the first fma — a warp keeps G times
// the bytes of one short-row slice in flight and waits for memory three times per group, not per part.
template <int UR, bool COH, int CM, int G, class PT>
__device__ __forceinline__ void narrow_group_sum(const Ctx& c, const PT* p, const int (&wp)[G + 1], int lane,
                                                 const int (&rows)[G], typename SpmvT<UR>::A (&acc)[G]) {
  using A = typename SpmvT<UR>::A;
  using CS = ColSrc<CM>;
  constexpr int LQ = LaneQ<A>::v;
  const A* vals = sell_vals<UR>(c);
  CS cs[G];
  typename CS::RawQ rq[G];
  typename CS::RawP rp[G];
  typename CS::RawS rs[G];
  A v[G][7];
#pragma unroll
  for (int g = 0; g < G; ++g) {
    const int w = wp[g + 1] - wp[g];
    cs[g] = CS(c, wp[g], w, lane, rows[g]);
    const A* vp = vals + (int64_t)wp[g] * 32;
    const bool hq = (w & 4) != 0, hp = (w & 2) != 0, hs = (w & 1) != 0;
    const int tail = hq ? 128 : 0, tail1 = tail + (hp ? 64 : 0);
    rq[g] = CS::zq(); rp[g] = CS::zp(); rs[g] = 0;
    A vq[4] = {A(0), A(0), A(0), A(0)}, vpair[2] = {A(0), A(0)}, vs = A(0);
    if (hq) { rq[g] = cs[g].quad(0, lane); lds_quad(vp + lane * LQ, vq); }
    if (hp) { rp[g] = cs[g].pair(tail, lane); lds_pair(vp + tail + lane * 2, vpair); }
    if (hs) { rs[g] = cs[g].single(tail1, lane); vs = lds_one(vp + tail1 + lane); }
    v[g][0] = vq[0]; v[g][1] = vq[1]; v[g][2] = vq[2]; v[g][3] = vq[3]; v[g][4] = vpair[0]; v[g][5] = vpair[1]; v[g][6] = vs;
  }
  A x[G][7];
#pragma unroll
  for (int g = 0; g < G; ++g) {
    const int w = wp[g + 1] - wp[g];
    const int kp = w & 4, ks = kp + (w & 2);  // entry index of the pair and of the single
    int jq[4], jp[2];
    cs[g].dq(rq[g], 0, jq);
    cs[g].dp(rp[g], kp, jp);
    const int js = cs[g].ds(rs[g], ks);
#pragma unroll
    for (int u = 0; u < 4; ++u) x[g][u] = gatherA<COH>(A(0), p, jq[u]);
    x[g][4] = gatherA<COH>(A(0), p, jp[0]);
    x[g][5] = gatherA<COH>(A(0), p, jp[1]);
    x[g][6] = gatherA<COH>(A(0), p, js);
  }
#pragma unroll
  for (int g = 0; g < G; ++g) {
    A t = 0;
#pragma unroll
    for (int u = 0; u < 7; ++u) t = fma(v[g][u], x[g][u], t);
    acc[g] = t;
  }
}

// G consecutive slices of the handle's UNIFORM STENCIL (structured-grid matrices: every such slice is diagonal-aligned,
// Ctx::uni_w <= 7 wide and has the diagonal offsets Ctx::uni_base, flagged in create()).  The columns are row + a
// constant held in the kernel's parameter block: no base load, no shuffle, and — CLAMP = false: the operand has a guard
// band — no clamp per entry.  The narrow slices were instruction-bound, not memory-bound (c2, FP32 phase: 130
// instructions per slice); this path issues about half of them.  Same entries in the same order: same bits.
template <int UR, bool COH, int G, bool CLAMP, class PT>
__device__ __forceinline__ void narrow_uniform_sum(const Ctx& c, const PT* p, const int (&wp)[G + 1], int lane, const int (&rows)[G],
                                                   typename SpmvT<UR>::A (&acc)[G]) {
  using A = typename SpmvT<UR>::A;
  constexpr int LQ = LaneQ<A>::v;
  const A* vals = sell_vals<UR>(c);
  const int w = c.uni_w;
  const bool hq = (w & 4) != 0, hp = (w & 2) != 0, hs = (w & 1) != 0;
  const int tail = hq ? 128 : 0, tail1 = tail + (hp ? 64 : 0);
  const int kp = w & 4, ks = kp + (w & 2);  // entry index of the pair and of the single
  // offsets of the 7 value slots (quad 0-3, pair 4-5, single 6); absent parts keep value 0 and take offset 0 of entry 0
  int off[7];
#pragma unroll
  for (int u = 0; u < 4; ++u) off[u] = hq ? c.uni_base[u] : c.uni_base[0];
  off[4] = hp ? c.uni_base[kp] : c.uni_base[0];
  off[5] = hp ? c.uni_base[kp + 1] : c.uni_base[0];
  off[6] = hs ? c.uni_base[ks] : c.uni_base[0];
  A v[G][7];
#pragma unroll
  for (int g = 0; g < G; ++g) {
    const A* vp = vals + (int64_t)wp[g] * 32;
    A vq[4] = {A(0), A(0), A(0), A(0)}, vpair[2] = {A(0), A(0)}, vs = A(0);
    if (hq) lds_quad(vp + lane * LQ, vq);
    if (hp) lds_pair(vp + tail + lane * 2, vpair);
    if (hs) vs = lds_one(vp + tail1 + lane);
    v[g][0] = vq[0]; v[g][1] = vq[1]; v[g][2] = vq[2]; v[g][3] = vq[3]; v[g][4] = vpair[0]; v[g][5] = vpair[1]; v[g][6] = vs;
  }
  A x[G][7];
#pragma unroll
  for (int g = 0; g < G; ++g) {
    const int r = rows[g] < 0 ? 0 : rows[g];
#pragma unroll
    for (int u = 0; u < 7; ++u) {
      int j = r + off[u];
      if (CLAMP) j = min(max(j, c.col_min), c.col_max);
      x[g][u] = gatherA<COH>(A(0), p, j);
    }
  }
#pragma unroll
  for (int g = 0; g < G; ++g) {
    A t = 0;
#pragma unroll
    for (int u = 0; u < 7; ++u) t = fma(v[g][u], x[g][u], t);
    acc[g] = t;
  }
}

template <int UR> struct SpmvGroup;  // slices a warp takes per pass
#ifndef AMP_SPMV_G32
#define AMP_SPMV_G32 2
#endif
#ifndef AMP_SPMV_G64
#define AMP_SPMV_G64 1
#endif
template <> struct SpmvGroup<P32> { static constexpr int G = AMP_SPMV_G32; };
template <> struct SpmvGroup<P64> { static constexpr int G = AMP_SPMV_G64; };
constexpr int kSpmvGroupMax = AMP_SPMV_G32 > AMP_SPMV_G64 ? AMP_SPMV_G32 : AMP_SPMV_G64;

// q = A p over the slice groups first, first + stride, ... of this warp (a group = G consecutive
// slices), then the long rows of this block.  COH = true: p was written earlier in the same
// (persistent) kernel, so it is gathered with plain coherent loads instead of the read-only path.
// NT = threads per block.
// Returns this thread's part of gamma = sum_i p_i q_i (stored q_i, FP64 products and sums).
// pg: the STORED p (u_z precision) for gamma = q^T p; it differs from the gathered operand p only in phase
// (u_z = FP64, u_r = FP32), where p is the FP32 copy RN32(p) written by the p update.
// G: slices a warp takes per pass (SpmvGroup<UR>::G)
template <int UR, bool COH, int CMG, int NT, int G, class PT, class PG>
__device__ __forceinline__ double phase_spmv_fmt(const Ctx& c, const PT* p, const PG* pg, typename Store<UR>::T* q, int bid, int nb,
                                                 double* red) {
  using A = typename SpmvT<UR>::A;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  constexpr int wpb = NT / 32;
  const int32_t* __restrict__ wptr = c.sell_wptr;
  const int nslices = c.nslices;
  const int n = (int)c.n;
  const int ngroups = (nslices + G - 1) / G;
  double gsum = 0.0;

  int gi = bid * wpb + warp;
  int wnext[G + 1];
#pragma unroll
  for (int g = 0; g <= G; ++g) wnext[g] = (gi < ngroups) ? __ldg(wptr + min(gi * G + g, nslices)) : 0;
  for (; gi < ngroups; gi += nb * wpb) {
    const int s0 = gi * G;
    int wp[G + 1], rows[G];
    int wmax = 0;
    bool all_al = true, any_al = false, all_uni = true, al_g[G];
#pragma unroll
    for (int g = 0; g <= G; ++g) wp[g] = wnext[g];
    {  // slice table entries of this warp's next group: off the critical path of the next pass
      const int gn = gi + nb * wpb;
      if (gn < ngroups) {
#pragma unroll
        for (int g = 0; g <= G; ++g) wnext[g] = __ldg(wptr + min(gn * G + g, nslices));
      }
    }
#ifndef AMP_SPMV_NO_PREFETCH
    // extent of the group two passes ahead: its value stream is prefetched into L2 at the end of this pass
    int pf0 = 0, pf1 = 0;
    {
      const int g2 = gi + 2 * nb * wpb;
      if (g2 < ngroups) {
        pf0 = __ldg(wptr + min(g2 * G, nslices)) & ~kWptrFlags;
        pf1 = __ldg(wptr + min(g2 * G + G, nslices)) & ~kWptrFlags;
      }
    }
#endif
#pragma unroll
    for (int g = 0; g < G; ++g) {
      al_g[g] = wp[g] < 0;  // kAlignedFlag
      all_uni = all_uni && (wp[g] & kUniformFlag) != 0;
      all_al = all_al && al_g[g];
      any_al = any_al || al_g[g];
    }
#pragma unroll
    for (int g = 0; g <= G; ++g) wp[g] &= ~kWptrFlags;
    double pi[G];
#pragma unroll
    for (int g = 0; g < G; ++g) {
      wmax = max(wmax, wp[g + 1] - wp[g]);
      int row = (s0 + g) * 32 + lane;
      if (s0 + g >= nslices) row = -1;
      else if (c.sell_perm != nullptr) row = __ldg(c.sell_perm + row);  // -1: padding slot
      if (row >= n) row = -1;
      rows[g] = row;
      pi[g] = gather64<COH>(pg, row < 0 ? 0 : row);  // p_i for gamma, issued with the other gathers
    }
    A acc[G];
    if (all_uni) {  // uniform stencil: columns are row + a constant of the handle
      if (c.uni_noclamp) narrow_uniform_sum<UR, COH, G, false>(c, p, wp, lane, rows, acc);
      else narrow_uniform_sum<UR, COH, G, true>(c, p, wp, lane, rows, acc);
    } else if (wmax <= 7 && (all_al || !any_al)) {
      if constexpr (G <= 2) {
        if (all_al) narrow_group_sum<UR, COH, 2, G>(c, p, wp, lane, rows, acc);
        else narrow_group_sum<UR, COH, CMG, G>(c, p, wp, lane, rows, acc);
      } else {  // bases / per-entry indices need registers too: two slices at a time
        static_assert(G % 2 == 0, "group size");
#pragma unroll
        for (int h = 0; h < G; h += 2) {
          const int wp2[3] = {wp[h], wp[h + 1], wp[h + 2]};
          const int rows2[2] = {rows[h], rows[h + 1]};
          A acc2[2];
          if (all_al) narrow_group_sum<UR, COH, 2, 2>(c, p, wp2, lane, rows2, acc2);
          else narrow_group_sum<UR, COH, CMG, 2>(c, p, wp2, lane, rows2, acc2);
          acc[h] = acc2[0]; acc[h + 1] = acc2[1];
        }
      }
    } else {
#pragma unroll
      for (int g = 0; g < G; ++g) {
        if (al_g[g]) acc[g] = slice_sum<UR, COH, 2>(c, p, wp[g], wp[g + 1] - wp[g], lane, rows[g]);
        else acc[g] = slice_sum<UR, COH, CMG>(c, p, wp[g], wp[g + 1] - wp[g], lane, rows[g]);
      }
    }
#pragma unroll
    for (int g = 0; g < G; ++g) {
      bool mine = rows[g] >= 0;
      // a long row has length 0 in its slice; the block that sums it from the CSR arrays (below) is the ONLY writer of
      // its q (nothing orders a store from here against that one)
      if (c.nlong > 0 && mine) mine = (c.rowptr[rows[g] + 1] - c.rowptr[rows[g]]) <= c.long_min;
      if (mine) {
        q[rows[g]] = acc[g];
        gsum = fma(pi[g], (double)acc[g], gsum);
      }
    }
#ifndef AMP_SPMV_NO_PREFETCH
    if (pf1 - pf0 > kPrefetchMinWidth) {  // one 128-byte line per lane and trip
      const char* src = reinterpret_cast<const char*>(sell_vals<UR>(c) + (int64_t)pf0 * 32);
      const int nbytes = (pf1 - pf0) * 32 * (int)sizeof(A);
      for (int off = lane * 128; off < nbytes; off += 32 * 128) asm volatile("prefetch.global.L2 [%0];" ::"l"(src + off));
    }
#endif
  }

  // rows too long for the slices: one block per row, straight from the CSR arrays
  for (int lr = bid; lr < c.nlong; lr += nb) {
    const int row = c.long_rows[lr];
    const int e0 = c.rowptr[row], e1 = c.rowptr[row + 1];
    const A* gv = csr_vals<UR>(c);
    A acc = 0;
    for (int e = e0 + (int)threadIdx.x; e < e1; e += NT) acc = fma(gv[e], gatherA<COH>(A(0), p, c.colidx[e] - c.col_shift), acc);
    const double tot = block_sum<NT>((double)acc, red);
    if (threadIdx.x == 0) {
      const A qi = (A)tot;
      q[row] = qi;
      gsum = fma(gather64<COH>(pg, row), (double)qi, gsum);
    }
  }
  return gsum;
}

// The mat-vec of a UNIFORM-STENCIL matrix as a lean loop of its own (k_spmv_uni): every slice diagonal-aligned, natural
// row order, no long rows (create() checks).  The general loop above carries the row order, the long-row test, the L2
// prefetch and three index formats through every pass: at 7 entries per row that bookkeeping was more than half of the
// 267 instructions of a pass and spilled loop-carried values at the 64-register budget (ncu source page, c2).
// Slices that are not flagged uniform (grid boundaries) take the aligned slice_sum.  Same fma chains: same bits.
// COH: as in phase_spmv (true: p holds entries a peer GPU stored while this kernel was already running — the halo bands of a
// sharded solve — so every gather is a plain coherent load, never ld.global.nc)
template <int UR, int NT, bool COH = false, class PT, class PG>
__device__ __forceinline__ double phase_spmv_uni(const Ctx& c, const PT* p, const PG* pg, typename Store<UR>::T* q, int bid, int nb) {
  using A = typename SpmvT<UR>::A;
  constexpr int G = SpmvGroup<UR>::G;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  constexpr int wpb = NT / 32;
  const int32_t* __restrict__ wptr = c.sell_wptr;
  const int nslices = c.nslices;
  const int n = (int)c.n;
  const int ngroups = (nslices + G - 1) / G;
  const int stride = nb * wpb;
  double gsum = 0.0;
  int gi = bid * wpb + warp;
  int wnext[G + 1];
#pragma unroll
  for (int g = 0; g <= G; ++g) wnext[g] = (gi < ngroups) ? __ldg(wptr + min(gi * G + g, nslices)) : 0;
  for (; gi < ngroups; gi += stride) {
    int wp[G + 1];
#pragma unroll
    for (int g = 0; g <= G; ++g) wp[g] = wnext[g];
    if (gi + stride < ngroups) {  // slice table of the next pass: off the critical path
#pragma unroll
      for (int g = 0; g <= G; ++g) wnext[g] = __ldg(wptr + min((gi + stride) * G + g, nslices));
    }
    bool all_uni = true;
#pragma unroll
    for (int g = 0; g < G; ++g) all_uni = all_uni && (wp[g] & kUniformFlag) != 0;
#pragma unroll
    for (int g = 0; g <= G; ++g) wp[g] &= ~kWptrFlags;
    int rows[G];
    double pi[G];
#pragma unroll
    for (int g = 0; g < G; ++g) {
      const int row = (gi * G + g) * 32 + lane;
      rows[g] = (gi * G + g < nslices && row < n) ? row : -1;
      pi[g] = gather64<COH>(pg, rows[g] < 0 ? 0 : rows[g]);  // the stored p_i for gamma
    }
    A acc[G];
    if (all_uni) {
      if (c.uni_noclamp) narrow_uniform_sum<UR, COH, G, false>(c, p, wp, lane, rows, acc);
      else narrow_uniform_sum<UR, COH, G, true>(c, p, wp, lane, rows, acc);
    } else {
#pragma unroll
      for (int g = 0; g < G; ++g) acc[g] = slice_sum<UR, COH, 2>(c, p, wp[g], wp[g + 1] - wp[g], lane, rows[g]);
    }
#pragma unroll
    for (int g = 0; g < G; ++g) {
      if (rows[g] >= 0) {
        q[rows[g]] = acc[g];
        gsum = fma(pi[g], (double)acc[g], gsum);
      }
    }
  }
  return gsum;
}

template <int UR, bool COH, int NT, class PT, class PG>
__device__ __forceinline__ double phase_spmv(const Ctx& c, const PT* p, const PG* pg, typename Store<UR>::T* q, int bid, int nb,
                                             double* red) {
  // (measured, profiles/r02.md: groups of 4 slices in the FP32 phase of uniform-stencil matrices spill at the 64-register
  // budget and are slower: c2 32.1 vs 25.0 us, c3 52.4 vs 40.7 us)
  constexpr int G = SpmvGroup<UR>::G;
  if (c.sell_cols16 != nullptr) return phase_spmv_fmt<UR, COH, 1, NT, G>(c, p, pg, q, bid, nb, red);
  return phase_spmv_fmt<UR, COH, 0, NT, G>(c, p, pg, q, bid, nb, red);
}

// ------------------------------------------------------------------ create(): CSR -> SELL-32 --
__device__ __forceinline__ int warp_min_i(int v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v = min(v, __shfl_xor_sync(0xffffffffu, v, o));
  return v;
}
__device__ __forceinline__ int warp_max_i(int v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v = max(v, __shfl_xor_sync(0xffffffffu, v, o));
  return v;
}

// Diagonal alignment of one slice (whole warp): the distinct offsets col - row of its 32 rows are
// enumerated in increasing order; position k of every row holds its entry on the k-th diagonal or
// an explicit zero.  place(k, offset, mine, e) is called for every position; returns the number of
// positions, or -1 if some row is not strictly increasing in column or more than kcap diagonals
// exist (the slice then keeps the general format).
template <class F>
__device__ __forceinline__ int sell_align(int row, int e0, int len, const int32_t* __restrict__ colidx, int kcap, F place) {
  const int kInf = 0x7fffffff;
  int ptr = 0, k = 0;
  bool bad = false;
  int cur = (ptr < len) ? colidx[e0 + ptr] - row : kInf;
  while (true) {
    const int m = warp_min_i(cur);
    if (m == kInf) break;
    if (k >= kcap) { bad = true; break; }
    const bool mine = (cur == m);
    place(k, m, mine, e0 + ptr);
    if (mine) {
      ++ptr;
      const int nxt = (ptr < len) ? colidx[e0 + ptr] - row : kInf;
      if (nxt <= m) bad = true;
      cur = nxt;
    }
    ++k;
  }
  return __any_sync(0xffffffffu, bad) ? -1 : k;
}

__device__ __forceinline__ void sell_slot(int n, int s, int lane, int long_min, const int32_t* __restrict__ rowptr,
                                          const int32_t* __restrict__ perm, int& row, int& e0, int& len) {
  row = s * 32 + lane;
  if (perm != nullptr) row = perm[row];
  e0 = 0; len = 0;
  if (row >= 0 && row < n) {
    e0 = rowptr[row];
    len = rowptr[row + 1] - e0;
    if (len > long_min) len = 0;
  } else {
    row = -1;
  }
}

// pass 1: width of every slice; bit 31 set = the slice is stored diagonal-aligned
// shift (= halo_lo of a block row of a sharded system, else 0) is subtracted from every column index: stored columns are
// relative to the first OWNED entry of p
__global__ void k_sell_scan(int n, int nslices, int long_min, int allow_aligned, int shift, const int32_t* __restrict__ rowptr,
                            const int32_t* __restrict__ colidx, const int32_t* __restrict__ perm, int32_t* __restrict__ width) {
  const int lane = threadIdx.x & 31;
  const int s = (int)(((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5);
  if (s >= nslices) return;
  int row, e0, len;
  sell_slot(n, s, lane, long_min, rowptr, perm, row, e0, len);
  const int wnat = warp_max_i(len);
  int w = wnat;
  if (allow_aligned && wnat > 0) {
    const int d = sell_align((row < 0 ? 0 : row) + shift, e0, len, colidx, wnat + (wnat >> 2), [](int, int, bool, int) {});
    if (d >= 0) w = d | kAlignedFlag;
  }
  if (lane == 0) width[s] = w;
}

// after pass 2: flag (bit 30 of wptr) every diagonal-aligned slice that is ref_w wide and has the diagonal offsets of the
// reference slice (bases[ref_w0 .. ref_w0 + ref_w)); counts the flagged slices
__global__ void k_mark_uniform(int nslices, int32_t* __restrict__ wptr, const int32_t* __restrict__ bases, int ref_w0, int ref_w,
                               int* __restrict__ count) {
  const int s = blockIdx.x * blockDim.x + threadIdx.x;
  if (s >= nslices) return;
  const int a = wptr[s], b = wptr[s + 1];
  if (a >= 0) return;  // not aligned
  const int w0 = a & ~kWptrFlags, w = (b & ~kWptrFlags) - w0;
  if (w != ref_w) return;
  for (int k = 0; k < w; ++k)
    if (bases[w0 + k] != bases[ref_w0 + k]) return;
  atomicOr(wptr + s, kUniformFlag);
  atomicAdd(count, 1);
}

// pass 2: one warp per slice; lane = row slot.  Long rows and padding slots get length 0.
// General slices: padding entries take the smallest real column of their entry index k (the base of
// the 16-bit format) and value 0; flag16 is set when some offset from the base does not fit 16 bits.
__global__ void k_sell_pack(int n, int nslices, int long_min, int shift, const int32_t* __restrict__ rowptr,
                            const int32_t* __restrict__ colidx, const double* __restrict__ vals,
                            const int32_t* __restrict__ wptr, const int32_t* __restrict__ perm, int32_t* __restrict__ cols,
                            uint16_t* __restrict__ cols16, int32_t* __restrict__ bases, double* __restrict__ v64,
                            float* __restrict__ v32, int* __restrict__ flag16) {
  const int lane = threadIdx.x & 31;
  const int s = (int)(((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5);
  if (s >= nslices) return;
  const bool aligned = wptr[s] < 0;
  const int w0 = wptr[s] & ~kWptrFlags, w = (wptr[s + 1] & ~kWptrFlags) - w0;
  const int64_t base = (int64_t)w0 * 32;
  int row, e0, len;
  sell_slot(n, s, lane, long_min, rowptr, perm, row, e0, len);
  if (aligned) {
    sell_align((row < 0 ? 0 : row) + shift, e0, len, colidx, w, [&](int k, int off, bool mine, int e) {
      const double v = mine ? vals[e] : 0.0;
      v32[base + sell_pos32(k, lane, w)] = __double2float_rn(v);
      v64[base + sell_pos64(k, lane, w)] = v;
      if (lane == 0) bases[w0 + k] = off;
    });
    return;
  }
  bool wide = false;
  for (int k = 0; k < w; ++k) {
    const bool ok = k < len;
    int j = ok ? colidx[e0 + k] - shift : 0x7fffffff;
    const int mn = warp_min_i(j), mx = warp_max_i(ok ? j : (int)0x80000000);
    if (!ok) j = mn;
    if (mx >= mn && mx - mn > 65535) wide = true;
    const double v = ok ? vals[e0 + k] : 0.0;
    const int64_t p32 = base + sell_pos32(k, lane, w);
    cols[p32] = j;
    cols16[p32] = (uint16_t)min(j - mn, 65535);
    v32[p32] = __double2float_rn(v);
    v64[base + sell_pos64(k, lane, w)] = v;
    if (lane == 0) bases[w0 + k] = mn;
  }
  if (wide && lane == 0) atomicOr(flag16, 1);
}

}  // namespace amp
