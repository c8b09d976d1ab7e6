// Host side of the block (real-space, n x n) path: coupling tables, workspace plan, launch
// sequencing of sancho_rubio.cu / block_sweep.cu / reduce.cu.  No arithmetic of the method runs
// here except the constant n x n products of the coupling blocks that define the lead's reduced
// chain (sancho_rubio.cu header), computed once at creation.
#include <algorithm>
#include <complex>
#include <cstdlib>
#include <cstring>
#include <new>
#include <vector>

#include "block_ops.cuh"
#include "block_path.h"
#include "negf_internal.h"

namespace negf {

using blk::CsrSet;
typedef std::complex<double> zc;

struct BlockPath {
  int C, N, n, K_eq, K_neq;
  double mu_s, mu_d, kT, deg, sr_tol, sr_shift;
  int sr_maxit;
  const double2 *z_eq, *w_eq, *z_neq;   // owned by the negf_handle
  const double* w_neq;
  double theta2;        // pivot acceptance threshold squared (negf_config.pivot_theta)
  // geometry
  int tpc, threads, geq, gneq;
  long long total_cta, n_eq_cta;
  int slots, wave, ctas_per_sm, n_launches;
  int64_t slot_bytes, hist_bytes, partial_bytes, table_bytes;
  // device
  int* csr_rowptr;
  int* csr_col;
  double2* csr_val;
  double2* csr_diag;
  int diag_mask;
  int nnz_cap;
  int row_nnz_max;
  double2* lead_mats;
  double2* table;
  double2* hist;
  double* partial;
  double* scratch;
  // Overlap plan (C = 1, one launch, the real-axis CTAs alone fit one wave but all CTAs do not -- config 3):
  // negf_set_potential runs the self-energies of the contour energies first and then starts the contour
  // half-sweeps + combine on a side stream, beside the self-energies of the real-axis energies; negf_charge
  // launches the real-axis CTAs only and joins.  Without it the few contour CTAs cost a second forward wave.
  bool overlap, contour_started;
  cudaStream_t side;
  cudaEvent_t ev_fork, ev_join;
  const double* U_last;   // potential the contour sweep was started for
  int* flags;       // [0] max SR iterations, [1] non-convergence flag
  unsigned long long* counters;   // [0] Sancho-Rubio passes of the last set_potential, summed over all tasks
  int last_max_iters;
  long long last_sr_passes;
};

namespace {

std::vector<zc> mat_mul(const std::vector<zc>& A, const std::vector<zc>& B, int n) {
  std::vector<zc> Cm((size_t)n * n, zc(0, 0));
  for (int i = 0; i < n; ++i)
    for (int k = 0; k < n; ++k) {
      const zc a = A[(size_t)i * n + k];
      if (a == zc(0, 0)) continue;
      for (int j = 0; j < n; ++j) Cm[(size_t)i * n + j] += a * B[(size_t)k * n + j];
    }
  return Cm;
}
std::vector<zc> mat_dag(const std::vector<zc>& A, int n) {
  std::vector<zc> D((size_t)n * n);
  for (int i = 0; i < n; ++i)
    for (int j = 0; j < n; ++j) D[(size_t)j * n + i] = std::conj(A[(size_t)i * n + j]);
  return D;
}
std::vector<zc> mat_add(const std::vector<zc>& A, const std::vector<zc>& B) {
  std::vector<zc> Cm(A.size());
  for (size_t i = 0; i < A.size(); ++i) Cm[i] = A[i] + B[i];
  return Cm;
}

template <typename T>
cudaError_t upload_vec(T** dst, const void* src, size_t count) {
  *dst = nullptr;
  cudaError_t e = cudaMalloc((void**)dst, sizeof(T) * std::max<size_t>(count, 1));
  if (e != cudaSuccess) return e;
  if (count == 0) return cudaSuccess;
  return cudaMemcpy(*dst, src, sizeof(T) * count, cudaMemcpyHostToDevice);
}

}  // namespace

void block_path_destroy(BlockPath* bp) {
  if (!bp) return;
  cudaFree(bp->csr_rowptr); cudaFree(bp->csr_col); cudaFree(bp->csr_val); cudaFree(bp->csr_diag);
  cudaFree(bp->lead_mats); cudaFree(bp->table); cudaFree(bp->hist);
  cudaFree(bp->partial); cudaFree(bp->scratch); cudaFree(bp->flags); cudaFree(bp->counters);
  if (bp->side) { cudaStreamSynchronize(bp->side); cudaStreamDestroy(bp->side); }
  if (bp->ev_fork) cudaEventDestroy(bp->ev_fork);
  if (bp->ev_join) cudaEventDestroy(bp->ev_join);
  delete bp;
}

negf_status block_path_create(const negf_config* cfg, const double2* z_eq_dev, const double2* w_eq_dev,
                              const double2* z_neq_dev, const double* w_neq_dev, BlockPath** out) {
  *out = nullptr;
  const int n = cfg->block;
  if (!blk::block_size_supported(n)) {
    set_error("negf_create: block size %d is not instantiated in this build of libnegf_b200 "
              "(see NEGF_BLOCK_SIZES in csrc/block_path.h)", n);
    return NEGF_EINVAL;
  }
  BlockPath* bp = new (std::nothrow) BlockPath();
  if (!bp) { set_error("negf_create: out of host memory"); return NEGF_ENOMEM; }
  std::memset(bp, 0, sizeof(*bp));
  bp->C = cfg->n_channels; bp->N = cfg->n_rings; bp->n = n;
  bp->K_eq = cfg->n_eq; bp->K_neq = cfg->n_neq;
  bp->mu_s = cfg->mu_s; bp->mu_d = cfg->mu_d; bp->kT = cfg->kT; bp->deg = cfg->deg;
  bp->sr_tol = cfg->sr_tol; bp->sr_maxit = cfg->sr_maxit;
  bp->theta2 = cfg->pivot_theta > 0.0 ? cfg->pivot_theta * cfg->pivot_theta : blk::kTheta2Default;
  bp->z_eq = z_eq_dev; bp->w_eq = w_eq_dev; bp->z_neq = z_neq_dev; bp->w_neq = w_neq_dev;
  auto fail = [&](negf_status st) { block_path_destroy(bp); return st; };

  // ---- coupling blocks: dense copies, the four CSR matrices, the lead's constant products
  const size_t nn = (size_t)n * n;
  std::vector<zc> E(nn), O(nn);
  for (size_t i = 0; i < nn; ++i) {
    E[i] = zc(cfg->coup_even[i].re, cfg->coup_even[i].im);
    O[i] = zc(cfg->coup_odd[i].re, cfg->coup_odd[i].im);
  }
  {
    double vmax = 0.0;
    for (size_t i = 0; i < nn; ++i) vmax = std::max(vmax, std::max(std::abs(E[i]), std::abs(O[i])));
    bp->sr_shift = 1e-4 * vmax;
  }
  const std::vector<zc> Ed = mat_dag(E, n), Od = mat_dag(O, n);
  const std::vector<zc>* four[4] = {&E, &Ed, &O, &Od};     // CSR_E, CSR_EDAG, CSR_O, CSR_ODAG
  int nnz_cap = 1;
  for (int m = 0; m < 4; ++m) {
    int c = 0;
    for (size_t i = 0; i < nn; ++i) c += ((*four[m])[i] != zc(0, 0));
    nnz_cap = std::max(nnz_cap, c);
  }
  bp->nnz_cap = nnz_cap;
  std::vector<int> rowptr(4 * (n + 1), 0), col((size_t)4 * nnz_cap, 0);
  std::vector<double2> val((size_t)4 * nnz_cap, make_double2(0.0, 0.0));
  for (int m = 0; m < 4; ++m) {
    int e = 0;
    for (int r = 0; r < n; ++r) {
      rowptr[m * (n + 1) + r] = e;
      for (int c = 0; c < n; ++c) {
        const zc v = (*four[m])[(size_t)r * n + c];
        if (v != zc(0, 0)) {
          col[(size_t)m * nnz_cap + e] = c;
          val[(size_t)m * nnz_cap + e] = make_double2(v.real(), v.imag());
          ++e;
        }
      }
    }
    rowptr[m * (n + 1) + n] = e;
  }
  bp->row_nnz_max = 1;
  for (int m = 0; m < 4; ++m)
    for (int r = 0; r < n; ++r)
      bp->row_nnz_max = std::max(bp->row_nnz_max, rowptr[m * (n + 1) + r + 1] - rowptr[m * (n + 1) + r]);
  // lead 0 (left, rings -1, -2, ...): V0 = H_{-1,-2} = E^dagger, V1 = H_{-2,-3} = O^dagger,
  //   Sigma_L = tau^dagger g tau with tau = H_{-1,0} = O          -> (L, R) = (O^dagger, O)
  // lead 1 (right, rings N, N+1, ...): V0 = H_{N,N+1}, V1 = H_{N+1,N+2},
  //   Sigma_R = H_{N-1,N} g H_{N-1,N}^dagger                     -> (L, R) = (bond(N-1), bond(N-1)^dagger)
  auto bond = [&](int j) -> const std::vector<zc>& { return (j % 2 == 0) ? E : O; };
  auto bond_dag = [&](int j) -> const std::vector<zc>& { return (j % 2 == 0) ? Ed : Od; };
  std::vector<double2> lead((size_t)2 * blk::kLeadMats * nn);
  for (int l = 0; l < 2; ++l) {
    const std::vector<zc>& V0 = l == 0 ? Ed : bond(bp->N);
    const std::vector<zc>& V1 = l == 0 ? Od : bond(bp->N + 1);
    const std::vector<zc> V0d = mat_dag(V0, n), V1d = mat_dag(V1, n);
    const std::vector<zc> P00 = mat_mul(V0, V0d, n);
    const std::vector<zc> PE = mat_add(mat_mul(V1d, V1, n), P00);
    const std::vector<zc> PA = mat_mul(V0, V1, n);
    const std::vector<zc> PB = mat_mul(V1d, V0d, n);
    const std::vector<zc>& Lm = l == 0 ? Od : bond(bp->N - 1);
    const std::vector<zc>& Rm = l == 0 ? O : bond_dag(bp->N - 1);
    const std::vector<zc>* all[blk::kLeadMats] = {&P00, &PE, &PA, &PB, &Lm, &Rm, &V0, &V1, &V0d, &V1d};
    for (int m = 0; m < blk::kLeadMats; ++m)
      for (size_t i = 0; i < nn; ++i)
        lead[((size_t)l * blk::kLeadMats + m) * nn + i] = make_double2((*all[m])[i].real(), (*all[m])[i].imag());
  }
  cudaError_t e = cudaSuccess;
  auto chk = [&](cudaError_t r) { if (e == cudaSuccess) e = r; };
  chk(upload_vec(&bp->csr_rowptr, rowptr.data(), rowptr.size()));
  chk(upload_vec(&bp->csr_col, col.data(), col.size()));
  chk(upload_vec(&bp->csr_val, val.data(), val.size()));
  {
    std::vector<double2> dg((size_t)4 * n);
    bp->diag_mask = 0;
    for (int m = 0; m < 4; ++m) {
      bool is_diag = true;
      for (int r = 0; r < n; ++r)
        for (int c = 0; c < n; ++c) {
          const zc v = (*four[m])[(size_t)r * n + c];
          if (r == c) dg[(size_t)m * n + r] = make_double2(v.real(), v.imag());
          else if (v != zc(0, 0)) is_diag = false;
        }
      if (is_diag) bp->diag_mask |= 1 << m;
    }
    chk(upload_vec(&bp->csr_diag, dg.data(), dg.size()));
  }
  chk(upload_vec(&bp->lead_mats, lead.data(), lead.size()));

  // ---- geometry and workspace plan
  bp->tpc = blk::block_tasks_per_cta(n);
  bp->threads = blk::block_threads(n);
  bp->geq = (bp->K_eq + bp->tpc - 1) / bp->tpc;
  const int tpc_real = blk::block_tasks_per_cta_real(n);
  bp->gneq = (bp->K_neq + tpc_real - 1) / tpc_real;
  bp->n_eq_cta = (long long)bp->C * bp->geq * 2;
  bp->total_cta = (long long)bp->C * 2 * (bp->geq + bp->gneq);
  const size_t K_all = (size_t)bp->K_eq + bp->K_neq;
  bp->table_bytes = (int64_t)(sizeof(double2) * (size_t)bp->C * K_all * 2 * 2 * nn);
  const int R = bp->geq + 2 * bp->gneq;
  bp->partial_bytes = (int64_t)(sizeof(double) * (size_t)bp->C * R * bp->N);
  const int nslice = (R + 63) / 64;
  chk(cudaMalloc((void**)&bp->table, (size_t)bp->table_bytes));
  chk(cudaMalloc((void**)&bp->partial, (size_t)bp->partial_bytes));
  chk(cudaMalloc((void**)&bp->scratch, sizeof(double) * (size_t)bp->C * nslice * bp->N));
  chk(cudaMalloc((void**)&bp->flags, 2 * sizeof(int)));
  if (e == cudaSuccess) chk(cudaMemset(bp->flags, 0, 2 * sizeof(int)));
  chk(cudaMalloc((void**)&bp->counters, sizeof(unsigned long long)));
  if (e == cudaSuccess) chk(cudaMemset(bp->counters, 0, sizeof(unsigned long long)));
  if (e != cudaSuccess) {
    set_error("negf_create (block path): device allocation failed: %s", cudaGetErrorString(e));
    return fail(e == cudaErrorMemoryAllocation ? NEGF_ENOMEM : NEGF_ECUDA);
  }
  int dev = 0, sms = 0;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  bp->ctas_per_sm = blk::block_sweep_ctas_per_sm(n, nnz_cap, bp->row_nnz_max);
  if (bp->ctas_per_sm < 1) {
    cudaGetLastError();
    set_error("negf_create: the block sweep kernel does not fit on this device (n = %d, nnz = %d)", n, nnz_cap);
    return fail(NEGF_ECUDA);
  }
  bp->wave = std::max(2, bp->ctas_per_sm * sms);
  bp->slot_bytes = (int64_t)sizeof(double2) * bp->N * blk::block_step_elems(n);
  size_t free_b = 0, total_b = 0;
  cudaMemGetInfo(&free_b, &total_b);
  // default (workspace_bytes = 0): what two waves of resident CTAs need, never more than 85 % of the free
  // device memory (include/negf.h)
  int64_t budget = cfg->workspace_bytes > 0 ? cfg->workspace_bytes : (int64_t)((double)free_b * 0.85);
  budget = std::min<int64_t>(budget, (int64_t)((double)free_b * 0.95));
  long long slots = std::min<long long>(bp->total_cta, budget / bp->slot_bytes);
  slots = std::min<long long>(slots, 2LL * bp->wave);
  if (slots > bp->wave && slots < bp->total_cta) slots = slots / bp->wave * bp->wave;
  slots &= ~1LL;
  if (slots < 2) {
    set_error("negf_create: recursion-history workspace too small (need >= %lld bytes for two CTAs)",
              (long long)(2 * bp->slot_bytes));
    return fail(NEGF_ENOMEM);
  }
  bp->slots = (int)slots;
  bp->hist_bytes = bp->slot_bytes * slots;
  bp->n_launches = (int)((bp->total_cta + slots - 1) / slots);
  {
    const char* force = getenv("NEGF_FORCE_OVERLAP");   // test hook: "1" forces the plan on small devices, "0" forbids it
    const bool possible = bp->C == 1 && bp->n_launches == 1 && bp->n_eq_cta > 0 && bp->total_cta > bp->n_eq_cta;
    // n = 17: the contour and the real-axis CTAs are different kernels (block_sweep.cu, block_fwd17.cu), so
    // the contour sweep always gains from running beside the self-energies of the real-axis energies
    const bool pays = bp->n == 17 || (bp->total_cta > bp->wave && bp->total_cta - bp->n_eq_cta <= bp->wave);
    bp->overlap = possible && (force ? force[0] == '1' : pays);
  }
  if (bp->overlap || bp->n == 17) {
    // (n = 17 without the overlap plan: block_path_run puts the contour CTAs of a launch on the side stream)
    // highest priority: when the contour CTAs and the second Sancho-Rubio launch become ready together, the
    // few contour CTAs must be placed first (a Sancho-Rubio CTA takes a whole SM's registers)
    int prio_lo = 0, prio_hi = 0;
    cudaDeviceGetStreamPriorityRange(&prio_lo, &prio_hi);
    chk(cudaStreamCreateWithPriority(&bp->side, cudaStreamNonBlocking, prio_hi));
    chk(cudaEventCreateWithFlags(&bp->ev_fork, cudaEventDisableTiming));
    chk(cudaEventCreateWithFlags(&bp->ev_join, cudaEventDisableTiming));
    if (e != cudaSuccess) {
      set_error("negf_create: cannot create the side stream: %s", cudaGetErrorString(e));
      return fail(NEGF_ECUDA);
    }
  }
  e = cudaMalloc((void**)&bp->hist, (size_t)bp->hist_bytes);
  if (e != cudaSuccess) {
    set_error("negf_create: cannot allocate %lld bytes of recursion history: %s", (long long)bp->hist_bytes,
              cudaGetErrorString(e));
    return fail(NEGF_ENOMEM);
  }
  *out = bp;
  return NEGF_OK;
}

namespace {

blk::SweepLaunch sweep_launch(const BlockPath* bp, const double* U_dev, double* T_res, int probe_ring, double* probe) {
  blk::SweepLaunch p;
  p.C = bp->C; p.N = bp->N; p.K_eq = bp->K_eq; p.K_neq = bp->K_neq;
  p.geq = bp->geq; p.gneq = bp->gneq; p.n_eq_cta = bp->n_eq_cta;
  p.U = U_dev; p.z_eq = bp->z_eq; p.w_eq = bp->w_eq; p.z_neq = bp->z_neq; p.w_neq = bp->w_neq;
  p.table = bp->table;
  p.mu_s = bp->mu_s; p.mu_d = bp->mu_d; p.kT = bp->kT; p.deg = bp->deg; p.theta2 = bp->theta2;
  p.hist = bp->hist; p.partial = bp->partial; p.T = T_res;
  p.probe_ring = probe_ring; p.probe = probe;
  p.csr.rowptr = bp->csr_rowptr; p.csr.col = bp->csr_col; p.csr.val = bp->csr_val;
  p.csr.nnz_cap = bp->nnz_cap;
  p.csr.row_nnz_max = bp->row_nnz_max;
  p.csr.diag = bp->csr_diag; p.csr.diag_mask = bp->diag_mask;
  p.cta_begin = 0;
  p.n_cta = 0;
  return p;
}

}  // namespace

negf_status block_path_before_potential(BlockPath* bp, cudaStream_t s) {
  // Overlap plan: a contour sweep started for the previous potential and never joined (two
  // negf_set_potential calls in a row) still reads U and the table: the stream waits for it first.
  if (bp->overlap && bp->contour_started) {
    NEGF_CUDA_TRY(cudaStreamWaitEvent(s, bp->ev_join, 0));
    bp->contour_started = false;
  }
  return NEGF_OK;
}

negf_status block_path_self_energy(BlockPath* bp, const double* U_dev, cudaStream_t s, ProfHook hook) {
  blk::SrLaunch p;
  p.C = bp->C; p.N = bp->N; p.K_eq = bp->K_eq; p.K_neq = bp->K_neq;
  p.U = U_dev; p.z_eq = bp->z_eq; p.z_neq = bp->z_neq;
  p.lead_mats = bp->lead_mats; p.table = bp->table;
  p.tol = bp->sr_tol; p.shift = bp->sr_shift; p.maxit = bp->sr_maxit; p.theta2 = bp->theta2;
  p.max_iters = bp->flags; p.noconv_flag = bp->flags + 1; p.iters_total = bp->counters;
  NEGF_CUDA_TRY(cudaMemsetAsync(bp->counters, 0, sizeof(unsigned long long), s));
  // [0] = largest iteration count of THIS call; [1] = non-convergence flag, sticky until block_path_check
  // has reported it (a Broyden loop that never syncs in between must not lose it)
  NEGF_CUDA_TRY(cudaMemsetAsync(bp->flags, 0, sizeof(int), s));
  const long long n_task = (long long)bp->C * ((long long)bp->K_eq + bp->K_neq) * 2;
  if (!bp->overlap) {
    p.task_begin = 0;
    p.task_end = n_task;
    hook.begin(hook.ctx, 0);
    cudaError_t e = blk::launch_sancho_rubio(bp->n, p, s);
    hook.end(hook.ctx);
    NEGF_CUDA_TRY(e);
    return NEGF_OK;
  }
  // overlap plan (C = 1: the contour energies are the first 2 K_eq tasks): self-energies of the contour
  // energies, then the contour half-sweeps + combine on the side stream beside the rest of the self-energies
  p.task_begin = 0;
  p.task_end = 2LL * bp->K_eq;
  hook.begin(hook.ctx, 0);
  cudaError_t e = blk::launch_sancho_rubio(bp->n, p, s);
  hook.end(hook.ctx);
  NEGF_CUDA_TRY(e);
  NEGF_CUDA_TRY(cudaEventRecord(bp->ev_fork, s));
  NEGF_CUDA_TRY(cudaStreamWaitEvent(bp->side, bp->ev_fork, 0));
  {
    blk::SweepLaunch q = sweep_launch(bp, U_dev, nullptr, -1, nullptr);
    q.cta_begin = 0;
    q.n_cta = (int)bp->n_eq_cta;
    NEGF_CUDA_TRY(blk::launch_block_sweep(bp->n, q, bp->side));
    NEGF_CUDA_TRY(blk::launch_block_combine(bp->n, q, 0, (int)(bp->n_eq_cta / 2), bp->side));
  }
  NEGF_CUDA_TRY(cudaEventRecord(bp->ev_join, bp->side));
  bp->contour_started = true;
  bp->U_last = U_dev;
  p.task_begin = 2LL * bp->K_eq;
  p.task_end = n_task;
  hook.begin(hook.ctx, 0);
  e = blk::launch_sancho_rubio(bp->n, p, s);
  hook.end(hook.ctx);
  NEGF_CUDA_TRY(e);
  return NEGF_OK;
}

negf_status block_path_run(BlockPath* bp, const double* U_dev, double* n_res, double* T_res, int probe_ring,
                           double* probe, cudaStream_t s, ProfHook hook) {
  blk::SweepLaunch p = sweep_launch(bp, U_dev, T_res, probe_ring, probe);
  if (bp->overlap && bp->contour_started && bp->U_last == U_dev) {
    // the contour CTAs run (or ran) on the side stream in the slots [0, n_eq_cta): the real-axis CTAs go to
    // the slots after them, in one wave
    p.cta_begin = bp->n_eq_cta;
    p.n_cta = (int)(bp->total_cta - bp->n_eq_cta);
    p.hist = bp->hist + (size_t)bp->n_eq_cta * bp->N * blk::block_step_elems(bp->n);
    hook.begin(hook.ctx, 1);
    cudaError_t e = blk::launch_block_sweep(bp->n, p, s);
    hook.end(hook.ctx);
    NEGF_CUDA_TRY(e);
    NEGF_CUDA_TRY(cudaStreamWaitEvent(s, bp->ev_join, 0));
    bp->contour_started = false;
  } else {
    if (bp->overlap && bp->contour_started) {          // started for another potential buffer: join, redo below
      NEGF_CUDA_TRY(cudaStreamWaitEvent(s, bp->ev_join, 0));
      bp->contour_started = false;
    }
    for (long long begin = 0; begin < bp->total_cta; begin += bp->slots) {
      p.cta_begin = begin;
      p.n_cta = (int)std::min<long long>(bp->slots, bp->total_cta - begin);
      const long long eq_end = std::min<long long>(begin + p.n_cta, bp->n_eq_cta);
      if (bp->n == 17 && eq_end > begin && begin + p.n_cta > bp->n_eq_cta) {
        // n = 17, a launch with both kinds of CTA: two kernels, which must not run one after the other (the
        // few contour CTAs would hold the device for a whole sweep).  Contour CTAs + combine go to the side
        // stream, the real-axis CTAs stay here in the slots after them; joined before the slots are reused.
        NEGF_CUDA_TRY(cudaEventRecord(bp->ev_fork, s));
        NEGF_CUDA_TRY(cudaStreamWaitEvent(bp->side, bp->ev_fork, 0));
        blk::SweepLaunch q = p;
        q.n_cta = (int)(eq_end - begin);
        NEGF_CUDA_TRY(blk::launch_block_sweep(bp->n, q, bp->side));
        NEGF_CUDA_TRY(blk::launch_block_combine(bp->n, q, begin, (int)((eq_end - begin) / 2), bp->side));
        NEGF_CUDA_TRY(cudaEventRecord(bp->ev_join, bp->side));
        blk::SweepLaunch r = p;
        r.cta_begin = eq_end;
        r.n_cta = (int)(begin + p.n_cta - eq_end);
        r.hist = p.hist + (size_t)(eq_end - begin) * bp->N * blk::block_step_elems(bp->n);
        hook.begin(hook.ctx, 1);
        cudaError_t e2 = blk::launch_block_sweep(bp->n, r, s);
        hook.end(hook.ctx);
        NEGF_CUDA_TRY(e2);
        NEGF_CUDA_TRY(cudaStreamWaitEvent(s, bp->ev_join, 0));
        continue;
      }
      hook.begin(hook.ctx, 1);
      cudaError_t e = blk::launch_block_sweep(bp->n, p, s);
      hook.end(hook.ctx);
      NEGF_CUDA_TRY(e);
      if (eq_end > begin) {
        hook.begin(hook.ctx, 3);
        e = blk::launch_block_combine(bp->n, p, begin, (int)((eq_end - begin) / 2), s);
        hook.end(hook.ctx);
        NEGF_CUDA_TRY(e);
      }
    }
  }
  hook.begin(hook.ctx, 2);
  cudaError_t e = launch_reduce_rows(bp->partial, n_res, bp->C, bp->geq + 2 * bp->gneq, bp->N, 1.0,
                                     bp->scratch, s);
  hook.end(hook.ctx);
  NEGF_CUDA_TRY(e);
  return NEGF_OK;
}

negf_status block_path_copy_sigma(BlockPath* bp, double2* sigma_dev, cudaStream_t s) {
  // table entry = [Sigma | F], n*n each: strided copy of the Sigma halves
  const size_t nn = (size_t)bp->n * bp->n;
  const size_t entries = (size_t)bp->C * ((size_t)bp->K_eq + bp->K_neq) * 2;
  NEGF_CUDA_TRY(cudaMemcpy2DAsync(sigma_dev, nn * sizeof(double2), bp->table, 2 * nn * sizeof(double2),
                                  nn * sizeof(double2), entries, cudaMemcpyDeviceToDevice, s));
  return NEGF_OK;
}

negf_status block_path_check(BlockPath* bp) {
  int host[2] = {0, 0};
  NEGF_CUDA_TRY(cudaMemcpy(host, bp->flags, sizeof(host), cudaMemcpyDeviceToHost));
  bp->last_max_iters = host[0];
  unsigned long long cnt = 0;
  NEGF_CUDA_TRY(cudaMemcpy(&cnt, bp->counters, sizeof(cnt), cudaMemcpyDeviceToHost));
  bp->last_sr_passes = (long long)cnt;
  if (host[1]) {
    NEGF_CUDA_TRY(cudaMemset(bp->flags + 1, 0, sizeof(int)));
    set_error("Sancho-Rubio decimation did not reach sr_tol within sr_maxit = %d iterations for at least "
              "one (channel, energy, lead)", bp->sr_maxit);
    return NEGF_ENOCONV;
  }
  return NEGF_OK;
}

void block_path_plan(BlockPath* bp, negf_plan_info* out) {
  out->history_bytes = bp->hist_bytes;
  out->partial_bytes = bp->partial_bytes;
  out->n_batches = bp->n_launches;
  out->max_sr_iterations = bp->last_max_iters;
  out->sr_passes_total = bp->last_sr_passes;
  // negate + Sancho-Rubio + sweep kernels (n = 17: one for the contour CTAs of a launch, forward + way-back
  // kernel for its real-axis CTAs) + one combine per launch that holds contour CTAs + 2-level reduce
  int sweeps = 0, combines = 0;
  for (long long b = 0; b < bp->total_cta; b += bp->slots) {
    if (bp->n == 17) sweeps += (b < bp->n_eq_cta ? 1 : 0) + (b + bp->slots > bp->n_eq_cta ? 2 : 0);
    else ++sweeps;
    if (b < bp->n_eq_cta) ++combines;
  }
  // overlap plan: two Sancho-Rubio launches and a contour sweep launch of its own
  out->kernel_launches = 1 + 1 + sweeps + combines + 2 + (bp->overlap ? 2 : 0);
}

}  // namespace negf
