// broyden_residual_noalloc (include/negf.h): the convergence measure of the self-consistent loop,
//     eps_max = max_t |x_in,t - x_out,t| / max(|x_in,t + x_out,t|, 1e-300)      (Alg.3 steps 2, 4-7),
// for callers that must not allocate: code under CUDA graph capture, tight serving loops, harnesses that
// forbid cudaMalloc.  It is the eps part of broyden_dots_kernel / broyden_finish_kernel (broyden.cu) with
// the per-block partial maxima in a file-scope device array instead of a cudaMalloc'ed buffer: the call
// launches two kernels on the caller's stream and calls no cudaMalloc, cudaFree or allocating routine.
//
// The array is 128 KiB, held by every GPU that loads the library until the process exits.  Each block
// reduces kElemsPerBlock entries into one partial, so len <= kNoallocMaxLen = 2^26 entries (config 5 has
// 256 000, the Table 2 shape 524 288); longer vectors are rejected with NEGF_EINVAL.
//
// All calls on one device share the array.  Nothing in it has to start at zero: a call overwrites the
// entries [0, nblocks) it reads and reads no others, so the previous call's contents never leak into the
// result.  Two calls that overlap on the GPU (different streams, no dependency between them) race on it.
#include <math_constants.h>

#include <mutex>

#include "negf_internal.h"

namespace negf {
namespace {

constexpr int kThreadsNa = 256;
constexpr int kElemsPerBlock = 4096;                 // 16 entries per thread
constexpr int kMaxBlocksNa = 16384;                  // 128 KiB of partials
constexpr int64_t kNoallocMaxLen = (int64_t)kMaxBlocksNa * kElemsPerBlock;   // 2^26
static_assert(kNoallocMaxLen == NEGF_NOALLOC_MAX_LEN, "include/negf.h states the limit");
constexpr int kMaxDevices = 64;

// Device storage.  In host code this name is a host-side stand-in, not a device address: the host passes
// the pointer cudaGetSymbolAddress returns (scratch_for_current_device below), never the name itself.
static __device__ __align__(256) double g_noalloc_part[kMaxBlocksNa];

// NaN and infinity both map to +infinity (fmax would drop a NaN; see broyden.cu)
__device__ __forceinline__ double nan_max_na(double a, double b) {
  if (!(fabs(b) <= 1.79769313486231570e308)) b = CUDART_INF;
  return (a >= b) ? a : b;
}

__global__ void __launch_bounds__(kThreadsNa)
residual_partial_kernel(const double* __restrict__ x_in, const double* __restrict__ x_out, int64_t len,
                        double* __restrict__ part) {
  __shared__ double sm[kThreadsNa / 32];
  const int64_t begin = (int64_t)blockIdx.x * kElemsPerBlock;
  const int64_t end = begin + kElemsPerBlock < len ? begin + kElemsPerBlock : len;
  double em = 0.0;
  for (int64_t t = begin + threadIdx.x; t < end; t += kThreadsNa) {
    const double xi = x_in[t], xo = x_out[t];
    em = nan_max_na(em, fabs(xi - xo) / fmax(fabs(xi + xo), 1e-300));      // steps 2, 4
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) em = nan_max_na(em, __shfl_down_sync(0xffffffffu, em, o));
  if ((threadIdx.x & 31) == 0) sm[threadIdx.x >> 5] = em;
  __syncthreads();
  if (threadIdx.x == 0) {
    double t = 0.0;
#pragma unroll
    for (int w = 0; w < kThreadsNa / 32; ++w) t = nan_max_na(t, sm[w]);
    part[blockIdx.x] = t;
  }
}

// single block: maximum over the blocks' partials (steps 5-7)
__global__ void __launch_bounds__(kThreadsNa)
residual_finish_kernel(const double* __restrict__ part, int nblocks, double* __restrict__ eps_max) {
  __shared__ double sm[kThreadsNa];
  double em = 0.0;
  for (int b = threadIdx.x; b < nblocks; b += kThreadsNa) em = nan_max_na(em, part[b]);
  sm[threadIdx.x] = em;
  __syncthreads();
  for (int h = kThreadsNa / 2; h > 0; h >>= 1) {
    if (threadIdx.x < h) sm[threadIdx.x] = nan_max_na(sm[threadIdx.x], sm[threadIdx.x + h]);
    __syncthreads();
  }
  if (threadIdx.x == 0) *eps_max = sm[0];
}

// Device address of g_noalloc_part on the current device, resolved once per device with that device
// current.  cudaGetSymbolAddress allocates nothing: the array is part of the loaded module.
negf_status scratch_for_current_device(double** out) {
  static std::mutex mu;
  static double* ptr[kMaxDevices] = {nullptr};
  int dev = -1;
  NEGF_CUDA_TRY(cudaGetDevice(&dev));
  if (dev < 0 || dev >= kMaxDevices) {
    set_error("broyden_residual_noalloc: device ordinal %d is outside [0, %d)", dev, kMaxDevices);
    return NEGF_EINVAL;
  }
  std::lock_guard<std::mutex> lock(mu);
  if (!ptr[dev]) {
    double* p = nullptr;
    cudaError_t e = cudaGetSymbolAddress((void**)&p, g_noalloc_part);
    if (e != cudaSuccess || !p) {
      cudaGetLastError();
      set_error("broyden_residual_noalloc: cudaGetSymbolAddress failed on device %d: %s", dev,
                cudaGetErrorString(e));
      return NEGF_ECUDA;
    }
    ptr[dev] = p;
  }
  *out = ptr[dev];
  return NEGF_OK;
}

}  // namespace
}  // namespace negf

using namespace negf;

extern "C" negf_status broyden_residual_noalloc(const double* x_in_dev, const double* x_out_dev, int64_t len,
                                                double* eps_max_dev, void* cuda_stream) {
  if (!x_in_dev || !x_out_dev || !eps_max_dev) {
    set_error("broyden_residual_noalloc: null argument");
    return NEGF_EINVAL;
  }
  if (len < 1 || len > kNoallocMaxLen) {
    set_error("broyden_residual_noalloc: len = %lld is outside [1, %lld] (the static scratch array holds one "
              "partial per %d entries, %d partials)", (long long)len, (long long)kNoallocMaxLen, kElemsPerBlock,
              kMaxBlocksNa);
    return NEGF_EINVAL;
  }
  double* part = nullptr;
  negf_status st = scratch_for_current_device(&part);
  if (st != NEGF_OK) return st;
  cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
  const int nblocks = (int)((len + kElemsPerBlock - 1) / kElemsPerBlock);
  residual_partial_kernel<<<nblocks, kThreadsNa, 0, s>>>(x_in_dev, x_out_dev, len, part);
  residual_finish_kernel<<<1, kThreadsNa, 0, s>>>(part, nblocks, eps_max_dev);
  NEGF_CUDA_TRY(cudaGetLastError());
  return NEGF_OK;
}
