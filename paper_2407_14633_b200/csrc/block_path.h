// Block (real-space, n x n) path: Sancho-Rubio self-energies + block RGF sweeps (configs[2..4]).
// Host-side interface used by negf_api.cu, and the launch descriptors shared by the kernels'
// translation units (sancho_rubio.cu, block_sweep.cu, block_path.cu).
#pragma once
#include <cuda_runtime.h>

#include "negf.h"

// Block sizes the kernels are instantiated for (registers hold one matrix row per thread, so the
// size is a compile-time constant).  17 = (17,0) tube; the small ones serve the brute-force tests.
#define NEGF_BLOCK_SIZES(X) X(2) X(3) X(4) X(5) X(8) X(17)

namespace negf {

struct BlockPath;

struct ProfHook {                 // optional per-kernel timing callbacks (kinds: 0 SR, 1 sweep, 2 reduce, 3 combine)
  void* ctx;
  void (*begin)(void* ctx, int kind);
  void (*end)(void* ctx);
};

negf_status block_path_create(const negf_config* cfg, const double2* z_eq_dev, const double2* w_eq_dev,
                              const double2* z_neq_dev, const double* w_neq_dev, BlockPath** out);
// to be called before U is overwritten by a new potential (joins a contour sweep still in flight)
negf_status block_path_before_potential(BlockPath* bp, cudaStream_t s);
negf_status block_path_self_energy(BlockPath* bp, const double* U_dev, cudaStream_t s, ProfHook hook);
negf_status block_path_run(BlockPath* bp, const double* U_dev, double* n_res, double* T_res, int probe_ring,
                           double* probe, cudaStream_t s, ProfHook hook);
negf_status block_path_check(BlockPath* bp);
negf_status block_path_copy_sigma(BlockPath* bp, double2* sigma_dev, cudaStream_t s);
void block_path_plan(BlockPath* bp, negf_plan_info* out);
void block_path_destroy(BlockPath* bp);

namespace blk {

// Sparse coupling matrices on the device: four CSR matrices E, E^dagger, O, O^dagger
// (E = coup_even = H_{i,i+1} for even i, O = coup_odd), concatenated.
struct CsrSet {
  const int* rowptr;     // [4][nb + 1], each starting at 0
  const int* col;        // [4][nnz_cap]
  const double2* val;    // [4][nnz_cap]
  int nnz_cap;           // max nnz over the four
  int row_nnz_max;       // max nnz of a row over the four (width of the padded row tables of block_fwd17.cu)
  const double2* diag;   // [4][nb] diagonal entries of the four matrices
  int diag_mask;         // bit m set: matrix m is diagonal (its products stay in registers)
};
enum { CSR_E = 0, CSR_EDAG = 1, CSR_O = 2, CSR_ODAG = 3 };

constexpr int kLeadMats = 10;
struct SrLaunch {
  int C, N, K_eq, K_neq;
  const double* U;            // [C][N]
  const double2* z_eq;        // [K_eq]
  const double2* z_neq;       // [K_neq]
  const double2* lead_mats;   // [2 leads][kLeadMats][nb*nb]: V0 V0^+, V1^+ V1 + V0 V0^+, V0 V1, V1^+ V0^+,
                              //   L, R, V0, V1, V0^+, V1^+
  double2* table;             // [C][K_eq + K_neq][2 leads][2: Sigma, F][nb*nb]
  double tol;
  double shift;               // imaginary energy shift of the fallback decimation (sancho_rubio.cu)
  double theta2;              // pivot acceptance threshold (block_ops.cuh)
  int maxit;
  int* max_iters;             // device scalar, atomicMax
  int* noconv_flag;           // device scalar
  unsigned long long* iters_total;   // device scalar: decimation passes summed over all tasks
  long long task_begin, task_end;    // this launch covers the tasks [task_begin, task_end) of the C * K_all * 2
};
cudaError_t launch_sancho_rubio(int nb, const SrLaunch& p, cudaStream_t s);

// One launch of the sweep kernel covers the global CTA range [cta_begin, cta_begin + n_cta).
// Global CTA numbering: contour CTAs first, (channel, energy group, direction) with direction
// fastest, then real-axis CTAs in the same order.  CTA j of the launch owns history slot j.
struct SweepLaunch {
  int C, N, K_eq, K_neq;
  int geq, gneq;              // energy groups per channel: ceil(K / TPC)
  long long n_eq_cta;         // number of contour CTAs = C * geq * 2 (they come first in the global numbering)
  long long cta_begin;
  int n_cta;
  const double* U;
  const double2 *z_eq, *w_eq, *z_neq;
  const double* w_neq;
  const double2* table;       // Sigma / F table of SrLaunch
  double mu_s, mu_d, kT, deg;
  double theta2;              // pivot acceptance threshold (block_ops.cuh)
  double2* hist;              // [slots][N][2 row slots][nb][THREADS]
  double* partial;            // [C][geq + 2 gneq][N]
  double* T;                  // [C][K_neq]
  int probe_ring;             // >= 0: ring whose per-energy charge contributions are recorded
  double* probe;              // [C][2 directions][K_neq], or nullptr
  CsrSet csr;
};
cudaError_t launch_block_sweep(int nb, const SweepLaunch& p, cudaStream_t s);
// n = 17: the way back of the real-axis CTAs of a finished sweep launch on the FP64 tensor cores
// (block_back.cu).  Other block sizes do the way back inside block_sweep_kernel.
constexpr int kHistLd17 = 18;         // row stride of a history matrix: 288 B rows start on 32-byte sectors
constexpr int kHistRec17 = 17 * kHistLd17;   // history elements per task and ring
constexpr int kBackThreads17 = 256;   // 8 warps = the 8 tasks of one block_fwd17 CTA
cudaError_t launch_block_back17(const SweepLaunch& p, cudaStream_t s);
cudaError_t launch_block_fwd17(const SweepLaunch& p, cudaStream_t s);    // block_fwd17.cu
int block_fwd17_ctas_per_sm(int row_nnz_max);
// Contour combine over the pairs of contour CTAs [cta_begin, cta_begin + 2 n_pairs) of a finished
// sweep launch whose first CTA was launch_cta_begin.
cudaError_t launch_block_combine(int nb, const SweepLaunch& p, long long pair_cta_begin, int n_pairs,
                                 cudaStream_t s);
// Geometry queries (host).
int block_tasks_per_cta(int nb);
int block_tasks_per_cta_real(int nb);   // real-axis CTAs (n = 17: block_fwd17.cu holds 8)
int block_threads(int nb);
long long block_step_elems(int nb);   // history elements per ring step per CTA
size_t block_sweep_smem(int nb, int nnz_cap);
int block_sweep_ctas_per_sm(int nb, int nnz_cap, int row_nnz_max);
bool block_size_supported(int nb);

}  // namespace blk
}  // namespace negf
