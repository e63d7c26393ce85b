// xr_static.cu — amp_xr_update_static(): step a5 of the loop (Alg 4.1 lines 15-17) for callers that
// must not allocate device memory.
//
// Everything else in this library hangs off a handle whose create() calls cudaMalloc for the work vectors, the partial
// sums and the ticket counters of the grid reductions.  Two kinds of caller can't use that:
//   * a process that handed all device memory to a pool of its own at start-up (a solver service that reserved the HBM
//     for its matrices, a framework with a fixed arena): a cudaMalloc made later fails with out-of-memory, or eats into
//     a budget somebody else planned;
//   * a time-step or control loop with a latency bound: cudaMalloc / cudaFree may synchronise the whole device and take
//     an unbounded time, which such a loop can't afford between two launches.
// For them this file offers ONE entry point that allocates nothing.  The x / r update needs scratch memory for its
// single-pass grid reduction of ||r||^2 (one partial sum per block + one ticket); here that scratch is a file-scope
// __device__ array of kXrStaticScratchBytes = 131 328 bytes.  It is part of the library image: every GPU that loads the
// library holds these bytes until the process exits, whether the entry point is used or not.
//
// What follows from the scratch being one fixed array:
//   * size limit: one block owns a tile of 4096 elements and one partial sum, the array holds 16 384 partial sums, so
//     n <= AMP_XR_STATIC_MAX_N = 67 108 864 (larger n is rejected, nothing is launched);
//   * every call on a device uses the SAME array, and the array keeps what the last call left.  Each call therefore
//     clears the ticket itself (a cudaMemsetAsync ahead of the kernel, in stream order); the partial sums need no clearing,
//     every one that is read was written by the same launch.  Two calls that overlap on one GPU (different streams, or
//     different host threads without ordering between their streams) race on the array: give them a common order.
//   * the host-side name of a __device__ array is not a device address.  The address is looked up once per device with
//     cudaGetSymbolAddress, with that device current, inside the first call made on that device; that first call
//     should therefore come before any stream capture is begun.  Later calls only read the cached address.
//
// Arithmetic: exactly that of phases.cuh xr_chunk<P64, P64> (FP64 x, p, q, r): x_i = fma(alpha, p_i, x_i),
// r_i = fma(-alpha, q_i, r_i), delta = sqrt(sum r_i^2); x and r are bit-identical to the handle path, the sum is added
// in another fixed order (per thread in element order, fixed tree in the block, blocks in index order).
#include <cuda_runtime.h>
#include <stdint.h>

#include <cstdarg>
#include <cstdio>
#include <mutex>

#include "../../include/amp_pcg.h"
#include "common.cuh"

namespace amp {
void set_error_text(const char* msg);  // amp_pcg.cu: the thread-local message behind amp_pcg_last_error()
}

namespace {

constexpr int kThreads = 256;
constexpr int kPairsPerThread = 8;                                     // 8 x double2 of each of x, p, q, r in flight per thread
constexpr int kTile = kThreads * kPairsPerThread * 2;                  // 4096 elements per block
constexpr int kMaxBlocks = 16384;                                      // partial sums the scratch array holds
constexpr int64_t kMaxN = (int64_t)kMaxBlocks * kTile;                 // 67 108 864
constexpr size_t kTicketOffset = sizeof(double) * (size_t)kMaxBlocks;  // the ticket sits behind the partial sums
constexpr size_t kXrStaticScratchBytes = kTicketOffset + 256;          // 131 328
constexpr int kMaxDevices = 64;
static_assert(kMaxN == AMP_XR_STATIC_MAX_N, "header and kernel disagree about the size limit");

}  // namespace

// the scratch memory of amp_xr_update_static: [kMaxBlocks] partial sums, then the ticket (first 4 bytes of the last 256)
static __device__ __align__(256) unsigned char g_xr_static_scratch[kXrStaticScratchBytes];

namespace {

__global__ void __launch_bounds__(kThreads) k_xr_static(const int64_t n, const double alpha, const double* __restrict__ p,
                                                        const double* __restrict__ q, double* __restrict__ x,
                                                        double* __restrict__ r, double* __restrict__ delta_out,
                                                        unsigned char* scratch) {
  __shared__ double red[32];
  __shared__ int s_last;
  double* partials = reinterpret_cast<double*>(scratch);
  unsigned int* ticket = reinterpret_cast<unsigned int*>(scratch + kTicketOffset);
  const int64_t npair = (n + 1) / 2;  // the last pair is half empty when n is odd
  const int64_t first = (int64_t)blockIdx.x * (kThreads * kPairsPerThread) + threadIdx.x;
  double2 xx[kPairsPerThread], pp[kPairsPerThread], qq[kPairsPerThread], rr[kPairsPerThread];
#pragma unroll
  for (int u = 0; u < kPairsPerThread; ++u) {
    const int64_t i = first + (int64_t)u * kThreads;
    if (2 * i + 1 < n) {
      xx[u] = reinterpret_cast<const double2*>(x)[i];
      pp[u] = reinterpret_cast<const double2*>(p)[i];
      qq[u] = reinterpret_cast<const double2*>(q)[i];
      rr[u] = reinterpret_cast<const double2*>(r)[i];
    } else if (i < npair) {
      xx[u] = make_double2(x[2 * i], 0.0);
      pp[u] = make_double2(p[2 * i], 0.0);
      qq[u] = make_double2(q[2 * i], 0.0);
      rr[u] = make_double2(r[2 * i], 0.0);
    }
  }
  double sum = 0.0;
#pragma unroll
  for (int u = 0; u < kPairsPerThread; ++u) {
    const int64_t i = first + (int64_t)u * kThreads;
    if (i >= npair) continue;
    const double x0 = fma(alpha, pp[u].x, xx[u].x), x1 = fma(alpha, pp[u].y, xx[u].y);     // line 15, FP64
    const double r0 = fma(-alpha, qq[u].x, rr[u].x), r1 = fma(-alpha, qq[u].y, rr[u].y);   // line 16
    if (2 * i + 1 < n) {
      reinterpret_cast<double2*>(x)[i] = make_double2(x0, x1);
      reinterpret_cast<double2*>(r)[i] = make_double2(r0, r1);
      sum = fma(r0, r0, sum);
      sum = fma(r1, r1, sum);
    } else {
      x[2 * i] = x0;
      r[2 * i] = r0;
      sum = fma(r0, r0, sum);
    }
  }
  // single-pass grid reduction through the static scratch: publish, take a ticket, the last block adds in index order
  const int nb = gridDim.x;
  const double bs = amp::block_sum<kThreads>(sum, red);
  if (threadIdx.x == 0) {
    __stcg(partials + blockIdx.x, bs);
    __threadfence();
    s_last = (atomicAdd(ticket, 1u) == (unsigned int)nb - 1u);
  }
  __syncthreads();
  if (s_last) {
    __threadfence();
    double s = 0.0;
    for (int i = threadIdx.x; i < nb; i += kThreads) s += __ldcg(partials + i);
    const double tot = amp::block_sum<kThreads>(s, red);
    if (threadIdx.x == 0) {
      *ticket = 0u;
      *delta_out = sqrt(tot);  // line 17
    }
  }
}

std::mutex g_mu;
unsigned char* g_scratch_of_device[kMaxDevices] = {};  // device address of g_xr_static_scratch, per device ordinal

void fail(const char* fmt, ...) {
  char buf[512];
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(buf, sizeof(buf), fmt, ap);
  va_end(ap);
  amp::set_error_text(buf);
}

// Set-up, once per device, with that device current: the device address behind the host-side name.
int scratch_of_current_device(unsigned char** out) {
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) {
    fail("amp_xr_update_static: cudaGetDevice failed (%s): no usable CUDA device, and this library has no CPU fallback", cudaGetErrorString(e));
    cudaGetLastError();
    return AMP_ERR_CUDA;
  }
  if (dev < 0 || dev >= kMaxDevices) {
    fail("amp_xr_update_static: device ordinal %d is beyond the %d devices this entry point keeps addresses for", dev, kMaxDevices);
    return AMP_ERR_INVALID;
  }
  std::lock_guard<std::mutex> lock(g_mu);
  if (g_scratch_of_device[dev] == nullptr) {
    unsigned char* ptr = nullptr;
    e = cudaGetSymbolAddress((void**)&ptr, g_xr_static_scratch);
    if (e != cudaSuccess || ptr == nullptr) {
      fail("amp_xr_update_static: cudaGetSymbolAddress of the static scratch failed on device %d: %s", dev, cudaGetErrorString(e));
      cudaGetLastError();
      return AMP_ERR_CUDA;
    }
    g_scratch_of_device[dev] = ptr;
  }
  *out = g_scratch_of_device[dev];
  return AMP_OK;
}

bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

}  // namespace

extern "C" int amp_xr_update_static(int64_t n, double alpha, const double* p, const double* q, double* x, double* r,
                                    double* delta_out, void* cuda_stream) {
  if (n <= 0) {
    fail("amp_xr_update_static: n must be positive (got %lld)", (long long)n);
    return AMP_ERR_INVALID;
  }
  if (n > kMaxN) {
    fail("amp_xr_update_static: n = %lld is beyond AMP_XR_STATIC_MAX_N = %lld, the most the fixed static scratch array serves; "
         "use a handle (amp_pcg_create) for larger systems", (long long)n, (long long)kMaxN);
    return AMP_ERR_INVALID;
  }
  if (!p || !q || !x || !r || !delta_out || !aligned16(p) || !aligned16(q) || !aligned16(x) || !aligned16(r) ||
      (reinterpret_cast<uintptr_t>(delta_out) & 7u) != 0) {
    fail("amp_xr_update_static: p, q, x, r must be 16-byte aligned device pointers and delta_out an 8-byte aligned one");
    return AMP_ERR_INVALID;
  }
  unsigned char* scratch = nullptr;
  const int rc = scratch_of_current_device(&scratch);
  if (rc != AMP_OK) return rc;
  cudaStream_t st = reinterpret_cast<cudaStream_t>(cuda_stream);
  // the array keeps the last call's contents: the ticket must start at zero (an earlier launch may have been cut short)
  cudaError_t e = cudaMemsetAsync(scratch + kTicketOffset, 0, 256, st);
  if (e == cudaSuccess) {
    const int blocks = (int)((n + kTile - 1) / kTile);
    k_xr_static<<<blocks, kThreads, 0, st>>>(n, alpha, p, q, x, r, delta_out, scratch);
    e = cudaGetLastError();
  }
  if (e != cudaSuccess) {
    fail("amp_xr_update_static: memset or launch failed: %s", cudaGetErrorString(e));
    cudaGetLastError();
    return AMP_ERR_CUDA;
  }
  return AMP_OK;
}
