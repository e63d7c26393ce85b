// common.cuh — device state, kernel context and small device helpers of the AMP-PCG loop.
//
// Notation follows Algorithm 4.1 of arXiv 2505.04155: r, z, p, q, x,
// rho = r^T z, beta, gamma = q^T p, alpha, delta = ||r||, omega = scaling factor,
// u_r = precision of r, q and of the matrix copy, u_z = precision of z, p.
#pragma once
#include <cuda_fp16.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace amp {

constexpr int P64 = 0, P32 = 1, P16 = 2;       // precision codes (= AMP_FP64/32/16 of the C ABI)
constexpr int kVecThreads = 256;               // block size of the vector kernels
constexpr int kSpmvThreads = 256;              // block size of the SpMV kernel: 8 warps, one SELL slice per warp and pass
constexpr int kSpmvWarps = kSpmvThreads / 32;
#ifndef AMP_SPMV_MINBLOCKS
#define AMP_SPMV_MINBLOCKS 4
#endif
constexpr int kSpmvMinBlocks = AMP_SPMV_MINBLOCKS;  // resident SpMV blocks per SM the register budget is set for
#ifndef AMP_PERSIST_THREADS
#define AMP_PERSIST_THREADS 512
#endif
constexpr int kPersistThreads = AMP_PERSIST_THREADS;  // block size of the persistent (whole-loop) kernel: one block per SM; 512 threads
                                                      // = 128 registers each (measured, us per iteration, 512 vs 1024 threads: c1 13.9 vs 18.8,
                                                      // 262 K rows 17.6 vs 20.6, 1 M rows 34.7 vs 35.8; profiles/r02.md)
constexpr int kPersistAutoMaxRows = 1 << 20;   // AMP_LOOP_AUTO takes the persistent kernel up to this many rows
constexpr int kPersistMinBlocks = 1;           // resident blocks per SM its register budget is set for
constexpr int kMaxGrid = 8192;                 // capacity of each partial-sum array
constexpr int kMaxWindow = 64;                 // max d / ell of the indicators
constexpr int kMaxChebDegree = 16;             // max sweeps of the Chebyshev-Jacobi preconditioner
constexpr int kMaxWorld = 16;                  // max ranks of a row-sharded solve (= AMP_SHARD_MAX_WORLD)

// Scalars of one solve, resident in device memory.  The host writes the policy part before the
// loop and reads the whole block once after it; inside the loop only kernels touch it.
struct DevState {
  // ---- per-solve inputs (host-written) ----
  const double* b;
  double* x;
  double* hist;            // ||r_t||, t = 0..maxit
  double tol, tau_zs, tau_zh, eps32, C, eta_safety, stop_safety;
  int32_t amp, u0, eta_rule, d, ell, scale_mode, no_stop, maxit;
  // ---- loop scalars (device-written) ----
  double bnorm, delta, omega, rho, rho_prev, beta, gamma, alpha, relres_true;
  int32_t k, done, status, zero_x;
  int32_t ur, uz;          // precisions selected for iteration k by (4.1)
  int32_t r_store, p_store;  // precisions r and p are currently stored in
  int32_t it_ur32, it_uz32, it_uz16, pad0;
  // lagged variant (AMP_SCALE_LAGGED): decisions already taken for the NEXT iteration
  int32_t ur_n, uz_n;
  double omega_n;
  // row-sharded solve: number of cross-rank reductions completed in this solve (written by k_epi only) and the solve
  // counter of the group (host-written); together they tag every mailbox entry and halo flag
  unsigned int xseq, epoch;
  unsigned int counter[4];  // last-block tickets of the three reductions (+ setup; + the halo push of the p update)
  unsigned long long fp16_subnormal, fp16_flushed, fp16_inf;
  // ---- grid barrier of the persistent kernel: arrivals since the start of the solve (host-zeroed); never
  //      written back from a block's replica ----
  unsigned int bar_count, bar_pad;
};

// Row-sharded solve (shard.cuh): what a rank needs to reach its peers.  One entry of a mailbox = one rank's partial sums
// of one reduction point; 2 halves (solve parity) x 4 slots (reduction sequence number mod 4) x kMaxWorld senders.
struct Mail { double v0, v1; unsigned long long tag, pad; };
constexpr int kMailSlots = 4;
constexpr int kMailEntries = 2 * kMailSlots * kMaxWorld;
struct ShardCtx {
  int32_t rank, world;
  int32_t inline_epi, pad0;            // 1: the block that completes a reduction also collects the other ranks' partial sums
                                       //    and runs the scalar step (ranks run concurrently: one per GPU); 0: k_epi does
                                       //    (ranks share a device and run one after the other)
  int32_t send_lo, send_hi;            // entries of p pushed to rank-1 (its upper halo) / rank+1 (its lower halo); multiples of 8
  Mail* mbox;                          // this rank's mailbox [kMailEntries]
  Mail* peer_mbox[kMaxWorld];          // every rank's mailbox (own included), peer-mapped
  unsigned long long* flags;           // this rank's halo flags: [0] set by rank-1 (lower band complete), [1] by rank+1
  unsigned long long* peer_flag_lo;    // flags[1] of rank-1, or nullptr
  unsigned long long* peer_flag_hi;    // flags[0] of rank+1, or nullptr
  char* peer_lo_band[3];               // [precision] where this rank's entry 0 goes in rank-1's p vector (its p + its n)
  char* peer_hi_band[3];               // [precision] where this rank's entry n - send_hi goes in rank+1's p vector (its p - send_hi)
};

// Handle-lifetime constants, passed to every kernel by value.
struct Ctx {
  DevState* st;
  int64_t n;       // rows
  int64_t npad;    // n rounded up to a multiple of 8: length of the library-owned vectors (zero padded)
  int64_t nnz;
  const int32_t* rowptr;
  const int32_t* colidx;
  const double* vals64;   // borrowed FP64 values
  const float* vals32;    // owned FP32-rounded copy (u_r = FP32 phase)
  const double* dinv64;   // 1/a_ii in FP64 (1 for M = I), used while u_z = FP64
  const float* dinv32;    // RN32(1/a_ii), used when u_z < FP64 (reading R6)
  double* r64; float* r32;
  double* q64; float* q32;
  double* z64; float* z32; __half* z16;
  double* p64; float* p32; __half* p16;
  double* d64; float* d32; __half* d16;   // Chebyshev direction d (AMP_PRECOND_CHEBJACOBI only), stored like z
  double* partials;       // [4][kMaxGrid] per-block partial sums
  // SELL-32 repack of A (spmv.cuh), owned by the handle
  const int32_t* sell_wptr;   // [nslices+1] cumulative slice widths; slice s starts at element 32*sell_wptr[s]
  const int32_t* sell_cols;   // 32-bit column indices (nullptr when the 16-bit format is in use)
  const uint16_t* sell_cols16;  // 16-bit column offsets from sell_base, or nullptr
  const int32_t* sell_base;   // [sum of widths] smallest column of entry k of each slice
  const double* sell_vals64;  // FP64 values
  const float* sell_vals32;   // FP32-rounded values (u_r = FP32 phase)
  const int32_t* sell_perm;   // [32*nslices] row of each slot (-1 = padding), or nullptr = identity
  const int32_t* long_rows;   // [nlong] rows kept out of the slices (longer than the cap), summed from CSR
  int32_t nslices;
  int32_t nlong;
  int32_t long_min;           // rows with more stored entries than this are "long": kept out of the slices
  // bulk-copy pipelined SpMV (spmv_pipe.cuh), only when the matrix is eligible (use_pipe)
  const int32_t* pipe_chunks;     // [nchunks+1] x {first slice, first entry column} of every stage
  const int32_t* pipe_blk_chunk;  // [pipe_grid+1] stage range of every block
  int32_t use_pipe;               // 1: iterations with u_r = FP32 run k_spmv_pipe, those with u_r = FP64 the direct k_spmv
  // Chebyshev-accelerated Jacobi (cheb_s = 0: not in use): sweeps, 1/theta, c1_i = rho_i rho_{i-1}, c2_i = 2 rho_i / dc
  int32_t cheb_s;
  double cheb_inv_theta;
  double cheb_c1[kMaxChebDegree], cheb_c2[kMaxChebDegree];
  cudaGraphConditionalHandle cond;  // WHILE-node handle (graph loop only)
  int32_t use_cond;
  // block row of a sharded system (create opts halo_lo / halo_hi): stored column indices are relative to the first owned
  // entry of p, gathers may reach col_min .. col_max (halo bands, then zero guard); col_shift = halo_lo is subtracted from
  // the borrowed CSR column indices (long rows)
  int32_t col_shift, col_min, col_max;
  // uniform stencil (spmv.cuh): slices flagged kUniformFlag in sell_wptr are diagonal-aligned, uni_w wide and share these
  // diagonal offsets, so their columns are row + a constant; uni_noclamp: the operand vector has a guard band that covers
  // every row + offset (the handle's own p / z), so no clamp is needed either
  int32_t uni_w, uni_noclamp;
  int32_t uni_base[8];
  // fused loop (vec_fused.cuh): the mat-vec only publishes its per-block partial sums of gamma; every block of
  // k_vec_fused adds them in index order and computes alpha on its replica (no last-block tail in the mat-vec)
  int32_t defer_gamma;
  int32_t spmv_grid_direct, spmv_grid_pipe;  // blocks of k_spmv / k_spmv_uni and of k_spmv_pipe (how many partials there are)
  int64_t n_scale;                  // rows of the WHOLE system (= n unless sharded): the n of the RMS scale sqrt(n)/||r||
  const ShardCtx* sh;               // device pointer, nullptr unless attached to a group (amp_pcg_shard_attach*)
};

// Programmatic dependent launch (sm_90+): every loop kernel lets its successor start launching at
// once and itself waits for its predecessor (completion + visibility of its writes) before the first
// access to anything the predecessor writes, so the launch latency of kernel N+1 overlaps the
// reduction tail of kernel N.  Both instructions are no-ops in a launch without the attribute.
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }

// ------------------------------------------------------------------ typed storage access ----
template <int P> struct Store;
template <> struct Store<P64> { using T = double; };
template <> struct Store<P32> { using T = float; };
template <> struct Store<P16> { using T = __half; };

template <int P> __device__ __forceinline__ typename Store<P>::T* rvec(const Ctx& c);
template <> __device__ __forceinline__ double* rvec<P64>(const Ctx& c) { return c.r64; }
template <> __device__ __forceinline__ float* rvec<P32>(const Ctx& c) { return c.r32; }
template <int P> __device__ __forceinline__ typename Store<P>::T* qvec(const Ctx& c);
template <> __device__ __forceinline__ double* qvec<P64>(const Ctx& c) { return c.q64; }
template <> __device__ __forceinline__ float* qvec<P32>(const Ctx& c) { return c.q32; }
template <int P> __device__ __forceinline__ typename Store<P>::T* zvec(const Ctx& c);
template <> __device__ __forceinline__ double* zvec<P64>(const Ctx& c) { return c.z64; }
template <> __device__ __forceinline__ float* zvec<P32>(const Ctx& c) { return c.z32; }
template <> __device__ __forceinline__ __half* zvec<P16>(const Ctx& c) { return c.z16; }
template <int P> __device__ __forceinline__ typename Store<P>::T* dvec(const Ctx& c);
template <> __device__ __forceinline__ double* dvec<P64>(const Ctx& c) { return c.d64; }
template <> __device__ __forceinline__ float* dvec<P32>(const Ctx& c) { return c.d32; }
template <> __device__ __forceinline__ __half* dvec<P16>(const Ctx& c) { return c.d16; }
template <int P> __device__ __forceinline__ typename Store<P>::T* pvec(const Ctx& c);
template <> __device__ __forceinline__ double* pvec<P64>(const Ctx& c) { return c.p64; }
template <> __device__ __forceinline__ float* pvec<P32>(const Ctx& c) { return c.p32; }
template <> __device__ __forceinline__ __half* pvec<P16>(const Ctx& c) { return c.p16; }

// one IEEE round-to-nearest-even of an FP64 value to the storage precision, returned as FP64
template <int P> __device__ __forceinline__ double round_to(double v);
template <> __device__ __forceinline__ double round_to<P64>(double v) { return v; }
template <> __device__ __forceinline__ double round_to<P32>(double v) { return (double)__double2float_rn(v); }
template <> __device__ __forceinline__ double round_to<P16>(double v) { return (double)__half2float(__double2half(v)); }

// load / store of 2 consecutive elements (element index 2*pair).  Loads return the raw packed
// pair so that many can be in flight in few registers; unpack() converts to FP64 exactly;
// stores round once (RN-even, direct from the double).
template <class T> struct Raw2;
template <> struct Raw2<double> { using T = double2; };
template <> struct Raw2<float> { using T = float2; };
template <> struct Raw2<__half> { using T = __half2; };
__device__ __forceinline__ double2 load_raw(const double* a, int64_t pair) { return reinterpret_cast<const double2*>(a)[pair]; }
__device__ __forceinline__ float2 load_raw(const float* a, int64_t pair) { return reinterpret_cast<const float2*>(a)[pair]; }
__device__ __forceinline__ __half2 load_raw(const __half* a, int64_t pair) { return reinterpret_cast<const __half2*>(a)[pair]; }
__device__ __forceinline__ void unpack(const double2 t, double& v0, double& v1) { v0 = t.x; v1 = t.y; }
__device__ __forceinline__ void unpack(const float2 t, double& v0, double& v1) { v0 = (double)t.x; v1 = (double)t.y; }
__device__ __forceinline__ void unpack(const __half2 t, double& v0, double& v1) {
  const float2 f = __half22float2(t);
  v0 = (double)f.x; v1 = (double)f.y;
}
template <class T> __device__ __forceinline__ void load2(const T* a, int64_t pair, double& v0, double& v1) {
  unpack(load_raw(a, pair), v0, v1);
}
__device__ __forceinline__ void store2(double* a, int64_t pair, double v0, double v1) {
  reinterpret_cast<double2*>(a)[pair] = make_double2(v0, v1);
}
__device__ __forceinline__ void store2(float* a, int64_t pair, double v0, double v1) {
  reinterpret_cast<float2*>(a)[pair] = make_float2(__double2float_rn(v0), __double2float_rn(v1));
}
__device__ __forceinline__ void store2(__half* a, int64_t pair, double v0, double v1) {
  reinterpret_cast<__half2*>(a)[pair] = __halves2half2(__double2half(v0), __double2half(v1));
}

// ------------------------------------------------------------------ chunked vector access ---
// The vector kernels give every thread chunks of E consecutive elements; a chunk of an array of
// type T is E*sizeof(T) contiguous bytes, moved with 128-bit accesses (64-bit for 4 halves).
// E = min(16 / smallest element, 32 / largest element) over the arrays of a kernel, so the
// narrowest array moves 16 bytes per access and the widest at most 32 bytes (one sector) per
// thread.  Raw words are kept packed until they are used (many chunks in flight, few registers).
template <class T, int E> struct Chunk {
  static constexpr int W = E * (int)sizeof(T) / 4;  // 32-bit words
  static_assert(W == 2 || W % 4 == 0, "chunk must be 8 bytes or a multiple of 16");
  uint32_t w[W];
};
template <class T, int E> __device__ __forceinline__ void chunk_load(Chunk<T, E>& k, const T* a, int64_t chunk) {
  constexpr int W = Chunk<T, E>::W;
  const char* src = reinterpret_cast<const char*>(a) + chunk * (int64_t)(E * sizeof(T));
  if constexpr (W == 2) {
    const uint2 t = *reinterpret_cast<const uint2*>(src);
    k.w[0] = t.x; k.w[1] = t.y;
  } else {
#pragma unroll
    for (int i = 0; i < W / 4; ++i) {
      const uint4 t = *reinterpret_cast<const uint4*>(src + 16 * i);
      k.w[4 * i] = t.x; k.w[4 * i + 1] = t.y; k.w[4 * i + 2] = t.z; k.w[4 * i + 3] = t.w;
    }
  }
}
template <class T, int E> __device__ __forceinline__ void chunk_store(const Chunk<T, E>& k, T* a, int64_t chunk) {
  constexpr int W = Chunk<T, E>::W;
  char* dst = reinterpret_cast<char*>(a) + chunk * (int64_t)(E * sizeof(T));
  if constexpr (W == 2) {
    *reinterpret_cast<uint2*>(dst) = make_uint2(k.w[0], k.w[1]);
  } else {
#pragma unroll
    for (int i = 0; i < W / 4; ++i)
      *reinterpret_cast<uint4*>(dst + 16 * i) = make_uint4(k.w[4 * i], k.w[4 * i + 1], k.w[4 * i + 2], k.w[4 * i + 3]);
  }
}
// exact conversion of the stored values to FP64
template <int E> __device__ __forceinline__ void chunk_unpack(const Chunk<double, E>& k, double (&v)[E]) {
#pragma unroll
  for (int i = 0; i < E; ++i) v[i] = __hiloint2double((int)k.w[2 * i + 1], (int)k.w[2 * i]);
}
template <int E> __device__ __forceinline__ void chunk_unpack(const Chunk<float, E>& k, double (&v)[E]) {
#pragma unroll
  for (int i = 0; i < E; ++i) v[i] = (double)__uint_as_float(k.w[i]);
}
template <int E> __device__ __forceinline__ void chunk_unpack(const Chunk<__half, E>& k, double (&v)[E]) {
#pragma unroll
  for (int i = 0; i < E / 2; ++i) {
    const float2 f = __half22float2(*reinterpret_cast<const __half2*>(&k.w[i]));
    v[2 * i] = (double)f.x; v[2 * i + 1] = (double)f.y;
  }
}
// one IEEE round-to-nearest-even from FP64 to the storage type (direct, no double rounding)
template <int E> __device__ __forceinline__ void chunk_pack(Chunk<double, E>& k, const double (&v)[E]) {
#pragma unroll
  for (int i = 0; i < E; ++i) { k.w[2 * i] = (uint32_t)__double2loint(v[i]); k.w[2 * i + 1] = (uint32_t)__double2hiint(v[i]); }
}
template <int E> __device__ __forceinline__ void chunk_pack(Chunk<float, E>& k, const double (&v)[E]) {
#pragma unroll
  for (int i = 0; i < E; ++i) k.w[i] = __float_as_uint(__double2float_rn(v[i]));
}
template <int E> __device__ __forceinline__ void chunk_pack(Chunk<__half, E>& k, const double (&v)[E]) {
#pragma unroll
  for (int i = 0; i < E / 2; ++i) {
    const __half2 h = __halves2half2(__double2half(v[2 * i]), __double2half(v[2 * i + 1]));
    k.w[i] = *reinterpret_cast<const uint32_t*>(&h);
  }
}
__host__ __device__ constexpr int cmin(int a, int b) { return a < b ? a : b; }
__host__ __device__ constexpr int cmax(int a, int b) { return a > b ? a : b; }
// elements per chunk for a kernel whose arrays have element sizes in [smin, smax] bytes
__host__ __device__ constexpr int chunk_elems(int smin, int smax) { return cmin(16 / smin, 32 / smax); }
#ifndef AMP_VEC_BIF
#define AMP_VEC_BIF 192
#endif
constexpr int kVecBytesInFlight = AMP_VEC_BIF;  // target bytes of loads in flight per thread of a vector kernel

// Row-sharded solve: where the chunks of p that a neighbour needs go: element index e of this rank's p lands at lo[e] (e < send_lo) and at
// hi[e - hi0] (e >= hi0 = n - send_hi)
template <class T> struct HaloPush {
  T* lo;
  T* hi;
  int64_t send_lo, hi0, n;
};
template <int P> __device__ __forceinline__ HaloPush<typename Store<P>::T> halo_push_of(const Ctx& c) {
  using T = typename Store<P>::T;
  HaloPush<T> h{nullptr, nullptr, 0, 0, 0};
  const ShardCtx* sh = c.sh;
  if (sh != nullptr) {
    h.lo = reinterpret_cast<T*>(sh->peer_lo_band[P]);
    h.hi = reinterpret_cast<T*>(sh->peer_hi_band[P]);
    h.send_lo = h.lo ? sh->send_lo : 0;
    h.n = c.n;
    h.hi0 = h.hi ? c.n - sh->send_hi : c.npad;
  }
  return h;
}
template <class T, int E> __device__ __forceinline__ void halo_push_chunk(const HaloPush<T>& h, const Chunk<T, E>& k, int64_t chunk) {
  const int64_t e = chunk * E;  // E divides 8 and the send ranges are multiples of 8: a chunk is inside a range or outside
  if (e < h.send_lo) chunk_store(k, h.lo, chunk);
  if (e >= h.hi0 && e < h.n) chunk_store(k, h.hi, chunk - h.hi0 / E);
}

// gather of one element of p as the SpMV working type.  COH = false: read-only path (p is not
// written by the running kernel); COH = true: plain coherent load.
template <bool COH, class T> __device__ __forceinline__ T ldp(const T* p, int j) { return COH ? p[j] : __ldg(p + j); }
template <bool COH> __device__ __forceinline__ double gather64(const double* p, int j) { return ldp<COH>(p, j); }
template <bool COH> __device__ __forceinline__ double gather64(const float* p, int j) { return (double)ldp<COH>(p, j); }
template <bool COH> __device__ __forceinline__ double gather64(const __half* p, int j) { return (double)__half2float(ldp<COH>(p, j)); }
template <bool COH> __device__ __forceinline__ float gather32(const double* p, int j) { return __double2float_rn(ldp<COH>(p, j)); }
template <bool COH> __device__ __forceinline__ float gather32(const float* p, int j) { return ldp<COH>(p, j); }
template <bool COH> __device__ __forceinline__ float gather32(const __half* p, int j) { return __half2float(ldp<COH>(p, j)); }

// ------------------------------------------------------------------ reductions --------------
__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

// Sum over the block; the result is valid in warp 0.  Fixed tree => deterministic.
template <int NT> __device__ __forceinline__ double block_sum(double v, double* sm /* [32] */) {
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  v = warp_sum(v);
  __syncthreads();
  if (lane == 0) sm[w] = v;
  __syncthreads();
  double t = (threadIdx.x < NT / 32) ? sm[threadIdx.x] : 0.0;
  if (w == 0) t = warp_sum(t);
  return t;
}

// Single-pass deterministic grid reduction: every block publishes its partial sum, the block
// that takes the last ticket adds the partials in index order and runs epi(total) on thread 0.
template <int NT, class Epi>
__device__ __forceinline__ void grid_reduce(double v, double* partials, unsigned int* counter, int bid, int nb,
                                            double* sm, Epi epi) {
  __shared__ int s_last;
  const double bs = block_sum<NT>(v, sm);
  if (threadIdx.x == 0) {
    __stcg(partials + bid, bs);
    __threadfence();
    const unsigned int t = atomicAdd(counter, 1u);
    s_last = (t == (unsigned int)nb - 1u);
  }
  __syncthreads();
  if (s_last) {
    __threadfence();
    double s = 0.0;
    for (int i = threadIdx.x; i < nb; i += NT) s += __ldcg(partials + i);
    const double tot = block_sum<NT>(s, sm);
    if (threadIdx.x == 0) {
      *counter = 0u;
      epi(tot);
    }
  }
}

// first half of grid_reduce only: publish this block's partial sum (the consumer kernel adds the partials itself)
template <int NT>
__device__ __forceinline__ void grid_publish(double v, double* partials, int bid, double* sm) {
  const double bs = block_sum<NT>(v, sm);
  if (threadIdx.x == 0) __stcg(partials + bid, bs);
}

// the same for two sums at once (partials interleaved: [2*bid], [2*bid+1])
template <int NT, class Epi>
__device__ __forceinline__ void grid_reduce2(double v0, double v1, double* partials, unsigned int* counter, int bid, int nb,
                                             double* sm, Epi epi) {
  __shared__ int s_last2;
  const double b0 = block_sum<NT>(v0, sm);
  const double b1 = block_sum<NT>(v1, sm);
  if (threadIdx.x == 0) {
    __stcg(partials + 2 * bid, b0);
    __stcg(partials + 2 * bid + 1, b1);
    __threadfence();
    const unsigned int t = atomicAdd(counter, 1u);
    s_last2 = (t == (unsigned int)nb - 1u);
  }
  __syncthreads();
  if (s_last2) {
    __threadfence();
    double s0 = 0.0, s1 = 0.0;
    for (int i = threadIdx.x; i < nb; i += NT) { s0 += __ldcg(partials + 2 * i); s1 += __ldcg(partials + 2 * i + 1); }
    const double t0 = block_sum<NT>(s0, sm);
    const double t1 = block_sum<NT>(s1, sm);
    if (threadIdx.x == 0) {
      *counter = 0u;
      epi(t0, t1);
    }
  }
}

}  // namespace amp
