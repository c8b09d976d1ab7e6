// Diagnostic: measured FP64 peaks of the device (DFMA chains and DMMA m8n8k4 chains).  The block path
// is FP64-compute bound and MEASURED_PEAKS.json holds no FP64 figure, so bench.py
// measures the denominator of that roofline on the box it runs on.
#include "negf_internal.h"

namespace negf {
namespace {

constexpr int kIters = 2048;

__global__ void __launch_bounds__(256) dfma_kernel(double* out, double a, double b) {
  double x0 = threadIdx.x, x1 = x0 + 1, x2 = x0 + 2, x3 = x0 + 3, x4 = x0 + 4, x5 = x0 + 5, x6 = x0 + 6,
         x7 = x0 + 7;
#pragma unroll 4
  for (int i = 0; i < kIters; ++i) {
    x0 = fma(x0, a, b); x1 = fma(x1, a, b); x2 = fma(x2, a, b); x3 = fma(x3, a, b);
    x4 = fma(x4, a, b); x5 = fma(x5, a, b); x6 = fma(x6, a, b); x7 = fma(x7, a, b);
  }
  out[blockIdx.x * blockDim.x + threadIdx.x] = x0 + x1 + x2 + x3 + x4 + x5 + x6 + x7;
}

__device__ __forceinline__ void dmma(double& d0, double& d1, double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
               : "+d"(d0), "+d"(d1)
               : "d"(a), "d"(b));
}

__global__ void __launch_bounds__(256) dmma_kernel(double* out, double a, double b) {
  double c[8][2];
#pragma unroll
  for (int j = 0; j < 8; ++j) c[j][0] = c[j][1] = threadIdx.x + j;
#pragma unroll 2
  for (int i = 0; i < kIters; ++i) {
#pragma unroll
    for (int j = 0; j < 8; ++j) dmma(c[j][0], c[j][1], a, b);
  }
  double s = 0;
#pragma unroll
  for (int j = 0; j < 8; ++j) s += c[j][0] + c[j][1];
  out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

}  // namespace
}  // namespace negf

using namespace negf;

extern "C" negf_status negf_fp64_peak(double* dfma_tflops, double* dmma_tflops) {
  int dev = 0, sms = 0;
  NEGF_CUDA_TRY(cudaGetDevice(&dev));
  NEGF_CUDA_TRY(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
  const int blocks = sms * 8, threads = 256;
  double* buf = nullptr;
  NEGF_CUDA_TRY(cudaMalloc((void**)&buf, sizeof(double) * blocks * threads));
  cudaEvent_t e0, e1;
  NEGF_CUDA_TRY(cudaEventCreate(&e0));
  NEGF_CUDA_TRY(cudaEventCreate(&e1));
  double best[2] = {0.0, 0.0};
  for (int which = 0; which < 2; ++which) {
    for (int rep = 0; rep < 6; ++rep) {
      cudaEventRecord(e0);
      if (which == 0) dfma_kernel<<<blocks, threads>>>(buf, 0.999999, 1e-9);
      else dmma_kernel<<<blocks, threads>>>(buf, 0.999999, 1e-9);
      cudaEventRecord(e1);
      cudaError_t err = cudaEventSynchronize(e1);
      if (err != cudaSuccess) { cudaFree(buf); set_error("fp64 peak kernel: %s", cudaGetErrorString(err)); return NEGF_ECUDA; }
      float ms = 0.f;
      cudaEventElapsedTime(&ms, e0, e1);
      const double flop = which == 0 ? 2.0 * 8 * kIters * (double)blocks * threads
                                     : 2.0 * 256 * 8 * kIters * (double)blocks * threads / 32;
      if (rep > 0) best[which] = fmax(best[which], flop / (ms * 1e-3) * 1e-12);
    }
  }
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  cudaFree(buf);
  if (dfma_tflops) *dfma_tflops = best[0];
  if (dmma_tflops) *dmma_tflops = best[1];
  return NEGF_OK;
}
