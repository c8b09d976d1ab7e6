// Internal declarations shared by the translation units of libnegf_b200 (not part of the C-ABI).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "negf.h"

namespace negf {

// ---------------------------------------------------------------- error plumbing
void set_error(const char* fmt, ...);
#define NEGF_CUDA_TRY(expr)                                                        \
  do {                                                                             \
    cudaError_t _e = (expr);                                                       \
    if (_e != cudaSuccess) {                                                       \
      ::negf::set_error("%s failed: %s (%s:%d)", #expr, cudaGetErrorString(_e),    \
                        __FILE__, __LINE__);                                       \
      return NEGF_ECUDA;                                                           \
    }                                                                              \
  } while (0)

// ---------------------------------------------------------------- scalar (mode-space) path
// One half-sweep task = (channel, mode, energy, direction); a warp holds 32 tasks of the same
// channel and direction.  Warp numbering inside a launch:
//   [0, n_cwarps)                      contour tasks, even = left-to-right, odd = right-to-left
//   [n_cwarps, n_cwarps + 2*n_rwarps)  real-axis tasks, even = left-to-right, odd = right-to-left
struct ScalarLaunch {
  int C, N, n_modes, K_eq, K_neq;
  int rwarps_per_channel;   // ceil(n_modes*K_neq/32)
  int cwarps_per_channel;   // 2 * ceil(n_modes*K_eq/32)
  const double* U;          // [C][N] on-site energy = -phi
  const double* bsq_even;   // [n_modes] |H_{i,i+1}|^2, i even
  const double* bsq_odd;    // [n_modes]
  const double* mode_w;     // [n_modes] deg * mode_weight
  const double* mode_w_T;   // [n_modes] mode_weight (for T(E))
  const double2* z_neq;     // [K_neq]
  const double* w_neq;      // [K_neq]
  const double2* z_eq;      // [K_eq]
  const double2* w_eq;      // [K_eq]
  double mu_s, mu_d, kT;
  double* hist_r;           // real-axis history: [warp][N][32] doubles
  double2* hist_c;          // contour history:   [warp][N][32] double2
  double* partial;          // [total warps][N] per-warp partial charge
  double* T_part;           // [C][n_modes][K_neq]
  int probe_ring;           // >= 0: ring whose per-energy charge contributions are recorded
  double* probe;            // [C][2 directions][n_modes][K_neq], or nullptr
  // parallel-in-N contour path (scalar_sweep.cu): steps 1 .. N-1 in seg_S segments of seg_L steps; nullptr = serial
  double2* seg_M;           // [contour warp of the launch][segment][4 components][32 lanes]
  double2* seg_v;           // [contour warp of the launch][segment][2 components][32 lanes]
  int seg_S, seg_L;
  int warp_begin, warp_end; // global warp range of this launch
  cudaStream_t side;        // host only: stream of the contour kernel (forked from / joined to s)
  cudaEvent_t ev_fork, ev_join;
};
cudaError_t launch_scalar_sweep(const ScalarLaunch& p, cudaStream_t s);

// ---------------------------------------------------------------- reductions
// out[r][col] = scale * sum_{j<rows_per_out} in[(r*rows_per_out + j)][col], deterministic order.
cudaError_t launch_reduce_rows(const double* in, double* out, int n_out, int rows_per_out,
                               int cols, double scale, double* scratch, cudaStream_t s);
// T[c][k] = sum_m T_part[c][m][k]
cudaError_t launch_reduce_modes(const double* T_part, double* T, int C, int n_modes, int K,
                                cudaStream_t s);
cudaError_t launch_negate(const double* in, double* out, int64_t n, cudaStream_t s);
// current / conductance reductions of T(E)  (eq.(5)-(6))
// Integrand of the real-axis part of eq.(4) at the probe ring and its peak:
// integrand[c][k] = 2 pi / (deg w_k) * sum_{dir, mode} probe[c][dir][mode][k]; k_peak[c] = first arg-max over k.
cudaError_t launch_integrand_peak(const double* probe, int C, int n_modes, int K, const double2* z_neq,
                                  const double* w_neq, double deg, double* integrand, int* k_peak,
                                  double* E_peak, cudaStream_t s);
cudaError_t launch_landauer(const double* T, const double2* z_neq, const double* w_neq, int C, int K,
                            double mu_s, double mu_d, double kT, double* current,
                            double* conductance, cudaStream_t s);

// ---------------------------------------------------------------- block (real-space) path
struct BlockLaunch;   // defined in block_sweep.cuh
}  // namespace negf
