// Second stage of the energy reduction (a5 of SURVEY.md 8(a); eq.(4)): deterministic
// sums of the per-warp partial charges, mode sum of T(E), and the Landauer reductions of T(E)
// (eq.(5)-(6)).
#include "negf_internal.h"

namespace negf {
namespace {

constexpr int kSliceRows = 64;    // rows summed by one block of the first level

// level 1: grid (ceil(cols/32), nslice, n_out), block (32, 8)
__global__ void reduce_rows_l1(const double* __restrict__ in, double* __restrict__ scratch,
                               int rows_per_out, int cols, int nslice) {
  __shared__ double sm[8][33];
  const int col = blockIdx.x * 32 + threadIdx.x;
  const int sl = blockIdx.y, r = blockIdx.z;
  const int j0 = sl * kSliceRows;
  const int j1 = min(j0 + kSliceRows, rows_per_out);
  double acc = 0.0;
  if (col < cols) {
    const double* base = in + (size_t)r * rows_per_out * cols + col;
    for (int j = j0 + threadIdx.y; j < j1; j += 8) acc += base[(size_t)j * cols];
  }
  sm[threadIdx.y][threadIdx.x] = acc;
  __syncthreads();
  if (threadIdx.y == 0 && col < cols) {
    double t = 0.0;
#pragma unroll
    for (int y = 0; y < 8; ++y) t += sm[y][threadIdx.x];
    scratch[((size_t)r * nslice + sl) * cols + col] = t;
  }
}

__global__ void reduce_rows_l2(const double* __restrict__ scratch, double* __restrict__ out, int n_out,
                               int nslice, int cols, double scale) {
  const int col = blockIdx.x * blockDim.x + threadIdx.x;
  const int r = blockIdx.y;
  if (col >= cols || r >= n_out) return;
  double t = 0.0;
  for (int s = 0; s < nslice; ++s) t += scratch[((size_t)r * nslice + s) * cols + col];
  out[(size_t)r * cols + col] = scale * t;
}

__global__ void reduce_modes_kernel(const double* __restrict__ Tp, double* __restrict__ T, int C,
                                    int n_modes, int K) {
  const int k = blockIdx.x * blockDim.x + threadIdx.x;
  const int c = blockIdx.y;
  if (k >= K) return;
  double t = 0.0;
  for (int m = 0; m < n_modes; ++m) t += Tp[((size_t)c * n_modes + m) * K + k];
  T[(size_t)c * K + k] = t;
}

__global__ void negate_kernel(const double* __restrict__ in, double* __restrict__ out, int64_t n) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) out[i] = -in[i];
}

__device__ __forceinline__ double fermi(double E, double mu, double kT) {
  double x = (E - mu) / kT;
  double e = exp(-fabs(x));
  return x > 0.0 ? e / (1.0 + e) : 1.0 / (1.0 + e);
}

// one block per channel; fixed-order tree reduction => deterministic
__global__ void landauer_kernel(const double* __restrict__ T, const double2* __restrict__ z,
                                const double* __restrict__ w, int K, double mu_s, double mu_d,
                                double kT, double* __restrict__ cur, double* __restrict__ cond) {
  __shared__ double s1[256], s2[256];
  const int c = blockIdx.x;
  double a = 0.0, b = 0.0;
  for (int k = threadIdx.x; k < K; k += 256) {
    const double E = z[k].x;
    const double t = T[(size_t)c * K + k] * w[k];
    const double fs = fermi(E, mu_s, kT), fd = fermi(E, mu_d, kT);
    a += t * (fs - fd);
    b += t * fs * (1.0 - fs) / kT;          // -df/dE
  }
  s1[threadIdx.x] = a;
  s2[threadIdx.x] = b;
  __syncthreads();
  for (int h = 128; h > 0; h >>= 1) {
    if (threadIdx.x < h) {
      s1[threadIdx.x] += s1[threadIdx.x + h];
      s2[threadIdx.x] += s2[threadIdx.x + h];
    }
    __syncthreads();
  }
  if (threadIdx.x == 0) {
    if (cur) cur[c] = s1[0];
    if (cond) cond[c] = s2[0];
  }
}

}  // namespace

cudaError_t launch_reduce_rows(const double* in, double* out, int n_out, int rows_per_out, int cols,
                               double scale, double* scratch, cudaStream_t s) {
  const int nslice = (rows_per_out + kSliceRows - 1) / kSliceRows;
  dim3 g1((cols + 31) / 32, nslice, n_out), b1(32, 8);
  reduce_rows_l1<<<g1, b1, 0, s>>>(in, scratch, rows_per_out, cols, nslice);
  dim3 g2((cols + 127) / 128, n_out);
  reduce_rows_l2<<<g2, 128, 0, s>>>(scratch, out, n_out, nslice, cols, scale);
  return cudaGetLastError();
}

cudaError_t launch_reduce_modes(const double* T_part, double* T, int C, int n_modes, int K,
                                cudaStream_t s) {
  if (K <= 0) return cudaSuccess;
  dim3 g((K + 127) / 128, C);
  reduce_modes_kernel<<<g, 128, 0, s>>>(T_part, T, C, n_modes, K);
  return cudaGetLastError();
}

cudaError_t launch_negate(const double* in, double* out, int64_t n, cudaStream_t s) {
  negate_kernel<<<(unsigned)((n + 255) / 256), 256, 0, s>>>(in, out, n);
  return cudaGetLastError();
}

cudaError_t launch_landauer(const double* T, const double2* z_neq, const double* w_neq, int C, int K,
                            double mu_s, double mu_d, double kT, double* current,
                            double* conductance, cudaStream_t s) {
  landauer_kernel<<<C, 256, 0, s>>>(T, z_neq, w_neq, K, mu_s, mu_d, kT, current, conductance);
  return cudaGetLastError();
}

}  // namespace negf
