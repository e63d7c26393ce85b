// spmv.cuh — step a4 of the loop: q = A p in u_r and gamma = q^T p (Alg 4.1 lines 11-13,
// PAPER.md:288-291; the paper also fuses the inner product into its Ax kernel, :537).
//
// Matrix format: SELL-32 ("sliced ELLPACK", slice height = warp width), repacked once from the
// caller's CSR in amp_pcg_create and owned by the handle (column indices, FP64 values and the
// FP32-rounded value copy of the u_r = FP32 phase).
//  * A slice is 32 consecutive rows (of the row order `perm`, identity unless the row lengths
//    vary enough for a windowed sort to pay); lane l of a warp owns row l of the slice.
//  * The slice width w = longest row of the slice; shorter rows are padded with (value 0,
//    column = own row).  w is cut as 4a + 2b + c and stored as a blocks of [lane][4] entries,
//    then b block of [lane][2], then c block of [lane][1], so a lane reads its row with 128-bit
//    loads (64-/32-bit for the remainder) and every warp-wide load is one contiguous, fully used
//    512-byte (256-, 128-byte) run: no padding beyond the slice maximum, 0.125 B/row of index
//    overhead (the cumulative widths) instead of CSR's 4 B/row row pointer.
//    FP64 values use [lane][2] blocks throughout (a quad = two consecutive pair blocks).
//  * Entries keep their CSR order within the row and each lane accumulates ONE fma chain in the
//    working precision, so q_i is bit-identical to a sequential CSR-order fma loop.
//  * Matrix data is streamed with ld.global.cs (evict-first) so that it does not displace the
//    vectors from L2; p is gathered through the read-only path (L1-cached) — adjacent lanes hold
//    adjacent rows, so for banded matrices one gather instruction touches one or two lines.
//  * Rows longer than the cap `long_row_min` are left out of the slices (length 0 there) and
//    summed straight from the borrowed CSR arrays by a whole block each.
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
__device__ __forceinline__ int4 lds_i4(const int32_t* p) { return __ldcs(reinterpret_cast<const int4*>(p)); }
__device__ __forceinline__ int2 lds_i2(const int32_t* p) { return __ldcs(reinterpret_cast<const int2*>(p)); }
__device__ __forceinline__ int lds_i1(const int32_t* p) { return __ldcs(p); }
__device__ __forceinline__ void lds_quad(const float* v, float (&a)[4]) {
  const float4 t = __ldcs(reinterpret_cast<const float4*>(v));
  a[0] = t.x; a[1] = t.y; a[2] = t.z; a[3] = t.w;
}
__device__ __forceinline__ void lds_quad(const double* v, double (&a)[4]) {  // v -> first pair block, lane offset applied
  const double2 t0 = __ldcs(reinterpret_cast<const double2*>(v));
  const double2 t1 = __ldcs(reinterpret_cast<const double2*>(v + 64));
  a[0] = t0.x; a[1] = t0.y; a[2] = t1.x; a[3] = t1.y;
}
__device__ __forceinline__ void lds_pair(const float* v, float (&a)[2]) {
  const float2 t = __ldcs(reinterpret_cast<const float2*>(v));
  a[0] = t.x; a[1] = t.y;
}
__device__ __forceinline__ void lds_pair(const double* v, double (&a)[2]) {
  const double2 t = __ldcs(reinterpret_cast<const double2*>(v));
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
__device__ __forceinline__ float lds_one(const float* v) { return __ldcs(v); }
__device__ __forceinline__ double lds_one(const double* v) { return __ldcs(v); }

// ------------------------------------------------------------------ column index sources ----
// I16 = false: 32-bit column indices.  I16 = true: 16-bit offsets from a per-(slice, entry) base
// (the smallest column of entry k over the 32 rows of the slice, sell_base[w0 + k]); chosen in
// create() when every offset fits, which holds for banded / stencil matrices.  The base of entry
// k is held by lane k % 32 and broadcast by a shuffle, so the index stream is 2 B per entry plus
// 4 B per 32 entries.
template <bool I16> struct ColSrc;
template <> struct ColSrc<false> {
  using RawQ = int4; using RawP = int2; using RawS = int;
  const int32_t* cp;
  __device__ __forceinline__ ColSrc(const Ctx& c, int w0, int, int) : cp(c.sell_cols + (int64_t)w0 * 32) {}
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
template <> struct ColSrc<true> {
  using RawQ = uint2; using RawP = uint32_t; using RawS = uint32_t;
  const uint16_t* cp;
  const int32_t* bp;  // bases of this slice
  int w, blk, bl;
  __device__ __forceinline__ ColSrc(const Ctx& c, int w0, int w_, int lane)
      : cp(c.sell_cols16 + (int64_t)w0 * 32), bp(c.sell_base + w0), w(w_), blk(0) {
    bl = (lane < w) ? __ldg(bp + lane) : 0;
  }
  // make the bases of entries [32*(k/32), +32) current (slices wider than 32 entries only)
  __device__ __forceinline__ void refresh(int k, int lane) {
    if ((k >> 5) != blk) {
      blk = k >> 5;
      bl = (blk * 32 + lane < w) ? __ldg(bp + blk * 32 + lane) : 0;
    }
  }
  __device__ __forceinline__ RawQ quad(int off, int lane) const { return __ldcs(reinterpret_cast<const uint2*>(cp + off + lane * 4)); }
  __device__ __forceinline__ RawP pair(int off, int lane) const { return __ldcs(reinterpret_cast<const uint32_t*>(cp + off + lane * 2)); }
  __device__ __forceinline__ RawS single(int off, int lane) const { return (uint32_t)__ldcs(cp + off + lane); }
  __device__ __forceinline__ int base(int k) const { return __shfl_sync(0xffffffffu, bl, k & 31); }
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

// One slice of any width: this lane's row sum (one fma chain in CSR order).
template <int UR, bool COH, bool I16, class PT>
__device__ __forceinline__ typename SpmvT<UR>::A slice_sum(const Ctx& c, const PT* p, int w0, int w, int lane) {
  using A = typename SpmvT<UR>::A;
  using CS = ColSrc<I16>;
  constexpr int LQ = LaneQ<A>::v;
  CS cs(c, w0, w, lane);
  const A* vp = sell_vals<UR>(c) + (int64_t)w0 * 32;
  const int a = w >> 2;
  A acc = 0;
  int cq = 0;
  for (; cq + 2 <= a; cq += 2) {  // two quads per trip: 4 (FP32) / 6 (FP64) wide loads in flight
    cs.refresh(4 * cq, lane);
    const typename CS::RawQ r0 = cs.quad(cq * 128, lane), r1 = cs.quad((cq + 1) * 128, lane);
    A v0[4], v1[4];
    lds_quad(vp + cq * 128 + lane * LQ, v0);
    lds_quad(vp + (cq + 1) * 128 + lane * LQ, v1);
    int j0[4], j1[4];
    cs.dq(r0, 4 * cq, j0);
    cs.dq(r1, 4 * cq + 4, j1);
    const A x0 = gatherA<COH>(A(0), p, j0[0]), x1 = gatherA<COH>(A(0), p, j0[1]);
    const A x2 = gatherA<COH>(A(0), p, j0[2]), x3 = gatherA<COH>(A(0), p, j0[3]);
    const A x4 = gatherA<COH>(A(0), p, j1[0]), x5 = gatherA<COH>(A(0), p, j1[1]);
    const A x6 = gatherA<COH>(A(0), p, j1[2]), x7 = gatherA<COH>(A(0), p, j1[3]);
    acc = fma(v0[0], x0, acc); acc = fma(v0[1], x1, acc); acc = fma(v0[2], x2, acc); acc = fma(v0[3], x3, acc);
    acc = fma(v1[0], x4, acc); acc = fma(v1[1], x5, acc); acc = fma(v1[2], x6, acc); acc = fma(v1[3], x7, acc);
  }
  // remainder: at most one quad, one pair, one single
  const bool hq = cq < a, hp = (w & 2) != 0, hs = (w & 1) != 0;
  const int tail = a * 128, tail1 = tail + (hp ? 64 : 0);
  if (hq) {
    cs.refresh(4 * cq, lane);
    const typename CS::RawQ r = cs.quad(cq * 128, lane);
    A v[4];
    lds_quad(vp + cq * 128 + lane * LQ, v);
    int j[4];
    cs.dq(r, 4 * cq, j);
    const A x0 = gatherA<COH>(A(0), p, j[0]), x1 = gatherA<COH>(A(0), p, j[1]);
    const A x2 = gatherA<COH>(A(0), p, j[2]), x3 = gatherA<COH>(A(0), p, j[3]);
    acc = fma(v[0], x0, acc); acc = fma(v[1], x1, acc); acc = fma(v[2], x2, acc); acc = fma(v[3], x3, acc);
  }
  if (hp) {
    cs.refresh(4 * a, lane);
    const typename CS::RawP r = cs.pair(tail, lane);
    A v[2];
    lds_pair(vp + tail + lane * 2, v);
    int j[2];
    cs.dp(r, 4 * a, j);
    const A x0 = gatherA<COH>(A(0), p, j[0]), x1 = gatherA<COH>(A(0), p, j[1]);
    acc = fma(v[0], x0, acc); acc = fma(v[1], x1, acc);
  }
  if (hs) {
    cs.refresh(w - 1, lane);
    const typename CS::RawS r = cs.single(tail1, lane);
    const A v = lds_one(vp + tail1 + lane);
    acc = fma(v, gatherA<COH>(A(0), p, cs.ds(r, w - 1)), acc);
  }
  return acc;
}

// G consecutive narrow slices (every width <= 7: one quad, one pair, one single at most) at once.
// Branch-free: absent parts keep offset 0 and value 0, so all matrix loads of the group are issued
// (predicated) before the first gather and all 7 G gathers before the first fma — a warp keeps G times
// the bytes of one short-row slice in flight and waits for memory three times per group, not per part.
template <int UR, bool COH, bool I16, int G, class PT>
__device__ __forceinline__ void narrow_group_sum(const Ctx& c, const PT* p, const int (&wp)[G + 1], int lane,
                                                 typename SpmvT<UR>::A (&acc)[G]) {
  using A = typename SpmvT<UR>::A;
  using CS = ColSrc<I16>;
  constexpr int LQ = LaneQ<A>::v;
  const A* vals = sell_vals<UR>(c);
  typename CS::RawQ rq[G];
  typename CS::RawP rp[G];
  typename CS::RawS rs[G];
  int bl[G];
  A v[G][7];
#pragma unroll
  for (int g = 0; g < G; ++g) {
    const int w = wp[g + 1] - wp[g];
    CS cs(c, wp[g], w, lane);
    if constexpr (I16) bl[g] = cs.bl; else bl[g] = 0;
    const A* vp = vals + (int64_t)wp[g] * 32;
    const bool hq = (w & 4) != 0, hp = (w & 2) != 0, hs = (w & 1) != 0;
    const int tail = hq ? 128 : 0, tail1 = tail + (hp ? 64 : 0);
    rq[g] = CS::zq(); rp[g] = CS::zp(); rs[g] = 0;
    A vq[4] = {A(0), A(0), A(0), A(0)}, vpair[2] = {A(0), A(0)}, vs = A(0);
    if (hq) { rq[g] = cs.quad(0, lane); lds_quad(vp + lane * LQ, vq); }
    if (hp) { rp[g] = cs.pair(tail, lane); lds_pair(vp + tail + lane * 2, vpair); }
    if (hs) { rs[g] = cs.single(tail1, lane); vs = lds_one(vp + tail1 + lane); }
    v[g][0] = vq[0]; v[g][1] = vq[1]; v[g][2] = vq[2]; v[g][3] = vq[3]; v[g][4] = vpair[0]; v[g][5] = vpair[1]; v[g][6] = vs;
  }
  A x[G][7];
#pragma unroll
  for (int g = 0; g < G; ++g) {
    const int w = wp[g + 1] - wp[g];
    CS cs(c, wp[g], 0, 32);  // addressing only; the bases were loaded above
    if constexpr (I16) cs.bl = bl[g];
    const int kp = w & 4, ks = kp + (w & 2);  // entry index of the pair and of the single
    int jq[4], jp[2];
    cs.dq(rq[g], 0, jq);
    cs.dp(rp[g], kp, jp);
    const int js = cs.ds(rs[g], ks);
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
template <int UR, bool COH, bool I16, int NT, class PT>
__device__ __forceinline__ double phase_spmv_fmt(const Ctx& c, const PT* p, typename Store<UR>::T* q, int bid, int nb,
                                                 double* red) {
  using A = typename SpmvT<UR>::A;
  constexpr int G = SpmvGroup<UR>::G;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  constexpr int wpb = NT / 32;
  const int32_t* __restrict__ wptr = c.sell_wptr;
  const int nslices = c.nslices;
  const int n = (int)c.n;
  const int ngroups = (nslices + G - 1) / G;
  double gsum = 0.0;

  for (int gi = bid * wpb + warp; gi < ngroups; gi += nb * wpb) {
    const int s0 = gi * G;
    int wp[G + 1];
    int wmax = 0;
#pragma unroll
    for (int g = 0; g <= G; ++g) wp[g] = __ldg(wptr + min(s0 + g, nslices));
#pragma unroll
    for (int g = 0; g < G; ++g) wmax = max(wmax, wp[g + 1] - wp[g]);
    A acc[G];
    if (wmax <= 7) {
      narrow_group_sum<UR, COH, I16, G>(c, p, wp, lane, acc);
    } else {
#pragma unroll
      for (int g = 0; g < G; ++g)
        acc[g] = slice_sum<UR, COH, I16>(c, p, wp[g], wp[g + 1] - wp[g], lane);
    }
#pragma unroll
    for (int g = 0; g < G; ++g) {
      if (s0 + g < nslices) {
        int row = (s0 + g) * 32 + lane;
        if (c.sell_perm != nullptr) row = __ldg(c.sell_perm + row);  // -1: padding slot
        if (row >= 0 && row < n) {
          q[row] = acc[g];
          gsum = fma(gather64<COH>(p, row), (double)acc[g], gsum);
        }
      }
    }
  }

  // rows too long for the slices: one block per row, straight from the CSR arrays
  for (int lr = bid; lr < c.nlong; lr += nb) {
    const int row = c.long_rows[lr];
    const int e0 = c.rowptr[row], e1 = c.rowptr[row + 1];
    const A* gv = csr_vals<UR>(c);
    A acc = 0;
    for (int e = e0 + (int)threadIdx.x; e < e1; e += NT) acc = fma(gv[e], gatherA<COH>(A(0), p, c.colidx[e]), acc);
    const double tot = block_sum<NT>((double)acc, red);
    if (threadIdx.x == 0) {
      const A qi = (A)tot;
      q[row] = qi;
      gsum = fma(gather64<COH>(p, row), (double)qi, gsum);
    }
  }
  return gsum;
}

template <int UR, bool COH, int NT, class PT>
__device__ __forceinline__ double phase_spmv(const Ctx& c, const PT* p, typename Store<UR>::T* q, int bid, int nb,
                                             double* red) {
  if (c.sell_cols16 != nullptr) return phase_spmv_fmt<UR, COH, true, NT>(c, p, q, bid, nb, red);
  return phase_spmv_fmt<UR, COH, false, NT>(c, p, q, bid, nb, red);
}

// ------------------------------------------------------------------ create(): CSR -> SELL-32 --
// one warp per slice; lane = row slot.  Long rows and padding slots get length 0.  Padding entries
// take the smallest real column of their entry index k (the base of the 16-bit format) and value 0.
// flag16 is set when some offset from the base does not fit 16 bits.
__global__ void k_sell_pack(int n, int nslices, int long_min, const int32_t* __restrict__ rowptr,
                            const int32_t* __restrict__ colidx, const double* __restrict__ vals,
                            const int32_t* __restrict__ wptr, const int32_t* __restrict__ perm, int32_t* __restrict__ cols,
                            uint16_t* __restrict__ cols16, int32_t* __restrict__ bases, double* __restrict__ v64,
                            float* __restrict__ v32, int* __restrict__ flag16) {
  const int lane = threadIdx.x & 31;
  const int s = (int)(((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5);
  if (s >= nslices) return;
  const int w0 = wptr[s], w = wptr[s + 1] - w0;
  const int64_t base = (int64_t)w0 * 32;
  int row = s * 32 + lane;
  if (perm != nullptr) row = perm[row];
  int e0 = 0, len = 0;
  if (row >= 0 && row < n) {
    e0 = rowptr[row];
    len = rowptr[row + 1] - e0;
    if (len > long_min) len = 0;
  }
  bool wide = false;
  for (int k = 0; k < w; ++k) {
    const bool ok = k < len;
    int j = ok ? colidx[e0 + k] : 0x7fffffff;
    int mn = j, mx = ok ? j : -1;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      mn = min(mn, __shfl_xor_sync(0xffffffffu, mn, o));
      mx = max(mx, __shfl_xor_sync(0xffffffffu, mx, o));
    }
    if (!ok) j = mn;
    if (mx - mn > 65535) wide = true;
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
