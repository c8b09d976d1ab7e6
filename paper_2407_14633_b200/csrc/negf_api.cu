// C-ABI of libnegf_b200 (include/negf.h): handle management, workspace planning, launch sequencing.
// No arithmetic of the method lives here; see scalar_sweep.cu, block_sweep.cu, sancho_rubio.cu,
// reduce.cu, broyden.cu.
#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <string>
#include <vector>

#include "block_path.h"
#include "negf_internal.h"

namespace negf {

static thread_local char g_err[512] = "";

void set_error(const char* fmt, ...) {
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(g_err, sizeof(g_err), fmt, ap);
  va_end(ap);
}

}  // namespace negf

using namespace negf;

namespace {

enum KernelKind { K_SCALAR_SWEEP = 0, K_REDUCE, K_SANCHO, K_BLOCK_SWEEP, K_BLOCK_COMBINE, K_MISC, K_COUNT };
const char* const kKernelNames[K_COUNT] = {"scalar_sweep", "reduce", "sancho_rubio", "block_sweep",
                                           "block_combine", "misc"};

struct ProfEntry {
  int kind;
  cudaEvent_t a, b;
};

struct Batch {
  int warp_begin, warp_end;
};

// scalar handles with at least this many rings run their contour half-sweeps parallel in N (the
// environment variables NEGF_SEG_MIN_RINGS / NEGF_SEG_LEN override the threshold / the segment length, read at
// negf_create; the tests use them to exercise the path on short devices and to compare with the serial pass)
int seg_min_rings() {
  const char* e = getenv("NEGF_SEG_MIN_RINGS");
  return e ? atoi(e) : 8192;
}

}  // namespace

struct negf_handle {
  negf_config cfg;          // pointers inside are nulled after the copy
  cudaStream_t stream;
  int C, N, n, n_modes, K_eq, K_neq;
  bool scalar;
  // device copies of the configuration
  double2 *z_eq, *w_eq, *z_neq;
  double* w_neq;
  double *bsq_even, *bsq_odd, *mode_w, *mode_w_T;
  // state
  double* U;                // [C][N]
  bool have_potential, results_valid;
  // scalar workspace
  int rwarps_per_channel, cwarps_per_channel, total_warps;
  std::vector<Batch> batches;
  char* hist;
  int64_t hist_bytes, partial_bytes;
  double *partial, *scratch, *T_part;
  double2 *seg_M, *seg_v;   // parallel-in-N contour path (long channels), else nullptr
  int seg_S, seg_L;
  cudaStream_t side;        // contour tasks run beside the real-axis tasks (fork / join by events)
  cudaEvent_t ev_fork, ev_join;
  // results
  double *n_res, *T_res;
  // host staging for negf_solve_host
  double* phi_stage;        // device [C][N]
  // probe ring of the semi-adaptive real-axis path
  int probe_ring;           // -1: off
  double* probe;            // [C][2][n_modes][K_neq]
  // block path
  BlockPath* block;
  // profiling
  bool profile;
  std::vector<ProfEntry> prof_pending;
  std::vector<cudaEvent_t> prof_free;
  int64_t prof_launches[K_COUNT];
  double prof_ms[K_COUNT];
};

namespace {

template <typename T>
cudaError_t upload(T** dst, const void* src, size_t count) {
  *dst = nullptr;
  if (count == 0) return cudaSuccess;
  cudaError_t e = cudaMalloc((void**)dst, sizeof(T) * count);
  if (e != cudaSuccess) return e;
  return cudaMemcpy(*dst, src, sizeof(T) * count, cudaMemcpyHostToDevice);
}

cudaEvent_t prof_event(negf_handle* h) {
  if (!h->prof_free.empty()) {
    cudaEvent_t e = h->prof_free.back();
    h->prof_free.pop_back();
    return e;
  }
  cudaEvent_t e = nullptr;
  cudaEventCreate(&e);
  return e;
}

struct ProfScope {
  negf_handle* h;
  ProfEntry ent;
  ProfScope(negf_handle* hh, int kind) : h(hh) {
    if (!h->profile) return;
    ent.kind = kind;
    ent.a = prof_event(h);
    ent.b = prof_event(h);
    cudaEventRecord(ent.a, h->stream);
  }
  ~ProfScope() {
    if (!h->profile) return;
    cudaEventRecord(ent.b, h->stream);
    h->prof_pending.push_back(ent);
  }
};

void prof_collect(negf_handle* h) {
  for (auto& e : h->prof_pending) {
    float ms = 0.f;
    if (cudaEventElapsedTime(&ms, e.a, e.b) == cudaSuccess) {
      h->prof_ms[e.kind] += ms;
      h->prof_launches[e.kind] += 1;
    }
    h->prof_free.push_back(e.a);
    h->prof_free.push_back(e.b);
  }
  h->prof_pending.clear();
}

// begin/end callbacks handed to the block path (kinds: 0 Sancho-Rubio, 1 sweep, 2 reduce, 3 combine)
void hook_begin(void* ctx, int kind) {
  negf_handle* h = static_cast<negf_handle*>(ctx);
  if (!h->profile) return;
  ProfEntry ent;
  static const int map[4] = {K_SANCHO, K_BLOCK_SWEEP, K_REDUCE, K_BLOCK_COMBINE};
  ent.kind = (kind >= 0 && kind < 4) ? map[kind] : K_MISC;
  ent.a = prof_event(h);
  ent.b = prof_event(h);
  cudaEventRecord(ent.a, h->stream);
  h->prof_pending.push_back(ent);
}
void hook_end(void* ctx) {
  negf_handle* h = static_cast<negf_handle*>(ctx);
  if (!h->profile) return;
  cudaEventRecord(h->prof_pending.back().b, h->stream);
}
ProfHook prof_hook(negf_handle* h) { return ProfHook{h, hook_begin, hook_end}; }

negf_status plan_scalar(negf_handle* h) {
  const int64_t N = h->N;
  h->rwarps_per_channel = (h->n_modes * h->K_neq + 31) / 32;
  h->cwarps_per_channel = 2 * ((h->n_modes * h->K_eq + 31) / 32);   // (group, direction) pairs
  const int wpc = h->cwarps_per_channel + 2 * h->rwarps_per_channel;
  const int64_t total = (int64_t)h->C * wpc;
  if (total <= 0 || total > (int64_t)1 << 30) {
    set_error("negf_create: no energy points, or too many tasks");
    return NEGF_EINVAL;
  }
  h->total_warps = (int)total;
  int64_t budget = h->cfg.workspace_bytes > 0 ? h->cfg.workspace_bytes : ((int64_t)64 << 30);
  const int64_t cbytes = N * 32 * 16, rbytes = N * 32 * 8;
  if (budget < 4 * cbytes) budget = 4 * cbytes;
  h->batches.clear();
  int64_t acc = 0, maxacc = 0;
  int begin = 0;
  for (int w = 0; w < h->total_warps; ++w) {
    const int64_t b = (w % wpc) < h->cwarps_per_channel ? cbytes : rbytes;
    const bool second_of_pair = (w % wpc) < h->cwarps_per_channel && ((w % wpc) & 1);
    if (acc + b > budget && !second_of_pair) {
      h->batches.push_back({begin, w});
      maxacc = std::max(maxacc, acc);
      begin = w;
      acc = 0;
    }
    acc += b;
  }
  h->batches.push_back({begin, h->total_warps});
  maxacc = std::max(maxacc, acc);
  h->hist_bytes = maxacc;
  h->partial_bytes = (int64_t)h->total_warps * N * 8;
  NEGF_CUDA_TRY(cudaMalloc((void**)&h->hist, (size_t)h->hist_bytes));
  NEGF_CUDA_TRY(cudaMalloc((void**)&h->partial, (size_t)h->partial_bytes));
  NEGF_CUDA_TRY(cudaStreamCreateWithFlags(&h->side, cudaStreamNonBlocking));
  NEGF_CUDA_TRY(cudaEventCreateWithFlags(&h->ev_fork, cudaEventDisableTiming));
  NEGF_CUDA_TRY(cudaEventCreateWithFlags(&h->ev_join, cudaEventDisableTiming));
  // Long channels: the contour half-sweeps are cut into segments of >= 256 steps and run parallel in N
  // (scalar_sweep.cu).  Workspace: 6 complex per (task, segment).
  h->seg_M = h->seg_v = nullptr;
  h->seg_S = h->seg_L = 0;
  if (N >= seg_min_rings() && N >= 3 && h->cwarps_per_channel > 0) {
    const char* le = getenv("NEGF_SEG_LEN");             // test hook: segment length
    h->seg_L = le ? std::max(1, atoi(le)) : (int)std::max<int64_t>(256, (N - 1 + 1023) / 1024);
    h->seg_S = (int)((N - 1 + h->seg_L - 1) / h->seg_L);
    int max_cw = 0;                                       // most contour warps in one batch
    for (const Batch& b : h->batches) {
      int cw = 0;
      for (int w = b.warp_begin; w < b.warp_end; ++w) cw += (w % wpc) < h->cwarps_per_channel;
      max_cw = std::max(max_cw, cw);
    }
    const size_t per = (size_t)max_cw * h->seg_S * 32;
    NEGF_CUDA_TRY(cudaMalloc((void**)&h->seg_M, sizeof(double2) * 4 * per));
    NEGF_CUDA_TRY(cudaMalloc((void**)&h->seg_v, sizeof(double2) * 2 * per));
  }
  const int nslice = (wpc + 63) / 64;
  NEGF_CUDA_TRY(cudaMalloc((void**)&h->scratch, sizeof(double) * (size_t)h->C * nslice * N));
  NEGF_CUDA_TRY(cudaMalloc((void**)&h->T_part,
                           sizeof(double) * std::max<size_t>(1, (size_t)h->C * h->n_modes * h->K_neq)));
  return NEGF_OK;
}

negf_status run_sweeps(negf_handle* h) {
  if (!h->have_potential) {
    set_error("no potential set: call negf_set_potential first");
    return NEGF_ESTATE;
  }
  if (h->results_valid) return NEGF_OK;
  if (h->scalar) {
    ScalarLaunch p;
    p.C = h->C; p.N = h->N; p.n_modes = h->n_modes; p.K_eq = h->K_eq; p.K_neq = h->K_neq;
    p.rwarps_per_channel = h->rwarps_per_channel;
    p.cwarps_per_channel = h->cwarps_per_channel;
    p.U = h->U; p.bsq_even = h->bsq_even; p.bsq_odd = h->bsq_odd;
    p.mode_w = h->mode_w; p.mode_w_T = h->mode_w_T;
    p.z_neq = h->z_neq; p.w_neq = h->w_neq; p.z_eq = h->z_eq; p.w_eq = h->w_eq;
    p.mu_s = h->cfg.mu_s; p.mu_d = h->cfg.mu_d; p.kT = h->cfg.kT;
    p.hist_r = reinterpret_cast<double*>(h->hist);
    p.hist_c = reinterpret_cast<double2*>(h->hist);
    p.partial = h->partial; p.T_part = h->T_part;
    p.side = h->side; p.ev_fork = h->ev_fork; p.ev_join = h->ev_join;
    p.probe_ring = h->probe_ring; p.probe = h->probe_ring >= 0 ? h->probe : nullptr;
    p.seg_M = h->seg_M; p.seg_v = h->seg_v; p.seg_S = h->seg_S; p.seg_L = h->seg_L;
    for (const Batch& b : h->batches) {
      p.warp_begin = b.warp_begin;
      p.warp_end = b.warp_end;
      ProfScope ps(h, K_SCALAR_SWEEP);
      NEGF_CUDA_TRY(launch_scalar_sweep(p, h->stream));
    }
    {
      ProfScope ps(h, K_REDUCE);
      const int wpc = h->cwarps_per_channel + 2 * h->rwarps_per_channel;
      NEGF_CUDA_TRY(launch_reduce_rows(h->partial, h->n_res, h->C, wpc, h->N, 1.0, h->scratch,
                                       h->stream));
      NEGF_CUDA_TRY(launch_reduce_modes(h->T_part, h->T_res, h->C, h->n_modes, h->K_neq, h->stream));
    }
  } else {
    negf_status st = block_path_run(h->block, h->U, h->n_res, h->T_res, h->probe_ring,
                                    h->probe_ring >= 0 ? h->probe : nullptr, h->stream, prof_hook(h));
    if (st != NEGF_OK) return st;
  }
  h->results_valid = true;
  return NEGF_OK;
}

}  // namespace

extern "C" const char* negf_last_error(void) { return negf::g_err; }
extern "C" const char* negf_version(void) { return "negf_b200 0.1 (sm_100a)"; }

extern "C" negf_status negf_destroy(negf_handle* h) {
  if (!h) return NEGF_OK;
  cudaStreamSynchronize(h->stream);
  prof_collect(h);
  for (auto e : h->prof_free) cudaEventDestroy(e);
  cudaFree(h->z_eq); cudaFree(h->w_eq); cudaFree(h->z_neq); cudaFree(h->w_neq);
  cudaFree(h->bsq_even); cudaFree(h->bsq_odd); cudaFree(h->mode_w); cudaFree(h->mode_w_T);
  cudaFree(h->U); cudaFree(h->hist); cudaFree(h->partial); cudaFree(h->scratch);
  cudaFree(h->seg_M); cudaFree(h->seg_v);
  cudaFree(h->T_part); cudaFree(h->n_res); cudaFree(h->T_res); cudaFree(h->phi_stage); cudaFree(h->probe);
  if (h->block) block_path_destroy(h->block);
  if (h->side) cudaStreamDestroy(h->side);
  if (h->ev_fork) cudaEventDestroy(h->ev_fork);
  if (h->ev_join) cudaEventDestroy(h->ev_join);
  delete h;
  return NEGF_OK;
}

extern "C" negf_status negf_create(const negf_config* cfg, void* cuda_stream, negf_handle** out) {
  if (!out) { set_error("negf_create: out is null"); return NEGF_EINVAL; }
  *out = nullptr;
  if (!cfg) { set_error("negf_create: cfg is null"); return NEGF_EINVAL; }
  if (cfg->n_channels < 1 || cfg->n_rings < 2 || cfg->block < 1 || cfg->block > 32) {
    set_error("negf_create: need n_channels >= 1, n_rings >= 2, 1 <= block <= 32");
    return NEGF_EINVAL;
  }
  if (!(cfg->kT > 0.0) || !(cfg->deg > 0.0)) { set_error("negf_create: need kT > 0 and deg > 0"); return NEGF_EINVAL; }
  if (cfg->reserved != 0 || cfg->workspace_bytes < 0 || !(cfg->pivot_theta >= 0.0)) {
    set_error("negf_create: need reserved == 0, workspace_bytes >= 0 and pivot_theta >= 0");
    return NEGF_EINVAL;
  }
  if (cfg->n_eq < 0 || cfg->n_neq < 0 || cfg->n_eq + cfg->n_neq < 1) {
    set_error("negf_create: need n_eq >= 0, n_neq >= 0 and at least one energy point");
    return NEGF_EINVAL;
  }
  if (!cfg->coup_even || !cfg->coup_odd || (cfg->n_eq > 0 && (!cfg->z_eq || !cfg->w_eq)) ||
      (cfg->n_neq > 0 && (!cfg->z_neq || !cfg->w_neq))) {
    set_error("negf_create: null array in config");
    return NEGF_EINVAL;
  }
  const bool scalar = cfg->block == 1;
  if (scalar && (cfg->lead_kind != 0 || cfg->n_modes < 1 || !cfg->mode_weight)) {
    set_error("negf_create: block == 1 needs lead_kind 0, n_modes >= 1 and mode_weight");
    return NEGF_EINVAL;
  }
  if (!scalar && (cfg->lead_kind != 1 || cfg->n_modes != 1)) {
    set_error("negf_create: block > 1 needs lead_kind 1 (Sancho-Rubio) and n_modes == 1");
    return NEGF_EINVAL;
  }
  if (!scalar && (cfg->sr_maxit < 1 || !(cfg->sr_tol > 0.0))) {
    set_error("negf_create: lead_kind 1 needs sr_maxit >= 1 and sr_tol > 0");
    return NEGF_EINVAL;
  }
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) {
    cudaGetLastError();
    set_error("negf_create: no CUDA device (this library has no CPU fallback)");
    return NEGF_ECUDA;
  }
  negf_handle* h = new (std::nothrow) negf_handle();
  if (!h) { set_error("negf_create: out of host memory"); return NEGF_ENOMEM; }
  h->cfg = *cfg;
  h->stream = static_cast<cudaStream_t>(cuda_stream);
  h->C = cfg->n_channels; h->N = cfg->n_rings; h->n = cfg->block;
  h->n_modes = scalar ? cfg->n_modes : 1;
  h->K_eq = cfg->n_eq; h->K_neq = cfg->n_neq;
  h->scalar = scalar;
  h->profile = cfg->profile != 0;
  h->probe_ring = -1;

  auto fail = [&](negf_status st) { negf_destroy(h); return st; };
  cudaError_t e = cudaSuccess;
  auto chk = [&](cudaError_t r) { if (e == cudaSuccess) e = r; };
  chk(upload(&h->z_eq, cfg->z_eq, h->K_eq));
  chk(upload(&h->w_eq, cfg->w_eq, h->K_eq));
  chk(upload(&h->z_neq, cfg->z_neq, h->K_neq));
  chk(upload(&h->w_neq, cfg->w_neq, h->K_neq));
  chk(cudaMalloc((void**)&h->U, sizeof(double) * (size_t)h->C * h->N));
  chk(cudaMalloc((void**)&h->phi_stage, sizeof(double) * (size_t)h->C * h->N));
  chk(cudaMalloc((void**)&h->n_res, sizeof(double) * (size_t)h->C * h->N));
  chk(cudaMalloc((void**)&h->T_res, sizeof(double) * std::max<size_t>(1, (size_t)h->C * h->K_neq)));
  if (scalar) {
    std::vector<double> be(h->n_modes), bo(h->n_modes), mw(h->n_modes), mwT(h->n_modes);
    for (int j = 0; j < h->n_modes; ++j) {
      be[j] = cfg->coup_even[j].re * cfg->coup_even[j].re + cfg->coup_even[j].im * cfg->coup_even[j].im;
      bo[j] = cfg->coup_odd[j].re * cfg->coup_odd[j].re + cfg->coup_odd[j].im * cfg->coup_odd[j].im;
      mw[j] = cfg->deg * cfg->mode_weight[j];
      mwT[j] = cfg->mode_weight[j];
    }
    chk(upload(&h->bsq_even, be.data(), h->n_modes));
    chk(upload(&h->bsq_odd, bo.data(), h->n_modes));
    chk(upload(&h->mode_w, mw.data(), h->n_modes));
    chk(upload(&h->mode_w_T, mwT.data(), h->n_modes));
  }
  if (e != cudaSuccess) {
    set_error("negf_create: device allocation/copy failed: %s", cudaGetErrorString(e));
    return fail(e == cudaErrorMemoryAllocation ? NEGF_ENOMEM : NEGF_ECUDA);
  }
  negf_status st;
  if (scalar) {
    st = plan_scalar(h);
  } else {
    st = block_path_create(cfg, h->z_eq, h->w_eq, h->z_neq, h->w_neq, &h->block);
  }
  if (st != NEGF_OK) return fail(st);
  h->cfg.coup_even = h->cfg.coup_odd = nullptr;
  h->cfg.mode_weight = nullptr;
  h->cfg.z_eq = h->cfg.w_eq = h->cfg.z_neq = nullptr;
  h->cfg.w_neq = nullptr;
  *out = h;
  return NEGF_OK;
}

extern "C" negf_status negf_set_potential(negf_handle* h, const double* phi_dev) {
  if (!h || !phi_dev) { set_error("negf_set_potential: null argument"); return NEGF_EINVAL; }
  if (!h->scalar) {
    negf_status st = block_path_before_potential(h->block, h->stream);
    if (st != NEGF_OK) return st;
  }
  {
    ProfScope ps(h, K_MISC);
    NEGF_CUDA_TRY(launch_negate(phi_dev, h->U, (int64_t)h->C * h->N, h->stream));   // U = -e phi
  }
  h->have_potential = true;
  h->results_valid = false;
  if (!h->scalar) {
    negf_status st = block_path_self_energy(h->block, h->U, h->stream, prof_hook(h));
    if (st != NEGF_OK) return st;
  }
  return NEGF_OK;
}

extern "C" negf_status negf_charge(negf_handle* h, double* n_dev) {
  if (!h || !n_dev) { set_error("negf_charge: null argument"); return NEGF_EINVAL; }
  negf_status st = run_sweeps(h);
  if (st != NEGF_OK) return st;
  NEGF_CUDA_TRY(cudaMemcpyAsync(n_dev, h->n_res, sizeof(double) * (size_t)h->C * h->N,
                                cudaMemcpyDeviceToDevice, h->stream));
  return NEGF_OK;
}

extern "C" negf_status negf_transmission(negf_handle* h, double* T_dev) {
  if (!h || !T_dev) { set_error("negf_transmission: null argument"); return NEGF_EINVAL; }
  negf_status st = run_sweeps(h);
  if (st != NEGF_OK) return st;
  if (h->K_neq > 0)
    NEGF_CUDA_TRY(cudaMemcpyAsync(T_dev, h->T_res, sizeof(double) * (size_t)h->C * h->K_neq,
                                  cudaMemcpyDeviceToDevice, h->stream));
  return NEGF_OK;
}

extern "C" negf_status negf_self_energy(negf_handle* h, negf_c64* sigma_dev) {
  if (!h || !sigma_dev) { set_error("negf_self_energy: null argument"); return NEGF_EINVAL; }
  if (h->scalar) {
    set_error("negf_self_energy: scalar handles evaluate the closed form inside the sweep kernel");
    return NEGF_EINVAL;
  }
  if (!h->have_potential) { set_error("no potential set: call negf_set_potential first"); return NEGF_ESTATE; }
  return block_path_copy_sigma(h->block, reinterpret_cast<double2*>(sigma_dev), h->stream);
}

extern "C" negf_status negf_current(negf_handle* h, double* current_dev, double* conductance_dev) {
  if (!h) { set_error("negf_current: null handle"); return NEGF_EINVAL; }
  negf_status st = run_sweeps(h);
  if (st != NEGF_OK) return st;
  ProfScope ps(h, K_MISC);
  NEGF_CUDA_TRY(launch_landauer(h->T_res, h->z_neq, h->w_neq, h->C, h->K_neq, h->cfg.mu_s, h->cfg.mu_d,
                                h->cfg.kT, current_dev, conductance_dev, h->stream));
  return NEGF_OK;
}

extern "C" negf_status negf_set_probe(negf_handle* h, int32_t ring) {
  if (!h) { set_error("negf_set_probe: null handle"); return NEGF_EINVAL; }
  if (ring >= h->N) { set_error("negf_set_probe: ring %d outside [0, %d)", ring, h->N); return NEGF_EINVAL; }
  if (ring >= 0 && h->K_neq < 1) { set_error("negf_set_probe: the handle has no real-axis points"); return NEGF_EINVAL; }
  if (ring >= 0 && !h->probe) {
    const size_t cnt = (size_t)h->C * 2 * h->n_modes * h->K_neq;
    NEGF_CUDA_TRY(cudaMalloc((void**)&h->probe, sizeof(double) * cnt));
    NEGF_CUDA_TRY(cudaMemsetAsync(h->probe, 0, sizeof(double) * cnt, h->stream));
  }
  h->probe_ring = ring < 0 ? -1 : ring;
  h->results_valid = false;
  return NEGF_OK;
}

extern "C" negf_status negf_integrand_peak(negf_handle* h, double* integrand_dev, int32_t* k_peak_dev,
                                           double* E_peak_dev) {
  if (!h) { set_error("negf_integrand_peak: null handle"); return NEGF_EINVAL; }
  if (h->probe_ring < 0) { set_error("negf_integrand_peak: no probe ring set (negf_set_probe)"); return NEGF_ESTATE; }
  negf_status st = run_sweeps(h);
  if (st != NEGF_OK) return st;
  ProfScope ps(h, K_MISC);
  NEGF_CUDA_TRY(launch_integrand_peak(h->probe, h->C, h->n_modes, h->K_neq, h->z_neq, h->w_neq, h->cfg.deg,
                                      integrand_dev, k_peak_dev, E_peak_dev, h->stream));
  return NEGF_OK;
}

extern "C" negf_status negf_sync(negf_handle* h) {
  if (!h) { set_error("negf_sync: null handle"); return NEGF_EINVAL; }
  NEGF_CUDA_TRY(cudaStreamSynchronize(h->stream));
  if (h->block) return block_path_check(h->block);
  return NEGF_OK;
}

extern "C" negf_status negf_solve_host(negf_handle* h, const double* phi_host, double* n_host,
                                       double* T_host) {
  if (!h || !phi_host || !n_host) { set_error("negf_solve_host: null argument"); return NEGF_EINVAL; }
  const size_t bytes = sizeof(double) * (size_t)h->C * h->N;
  NEGF_CUDA_TRY(cudaMemcpyAsync(h->phi_stage, phi_host, bytes, cudaMemcpyHostToDevice, h->stream));
  negf_status st = negf_set_potential(h, h->phi_stage);
  if (st != NEGF_OK) return st;
  st = run_sweeps(h);
  if (st != NEGF_OK) return st;
  NEGF_CUDA_TRY(cudaMemcpyAsync(n_host, h->n_res, bytes, cudaMemcpyDeviceToHost, h->stream));
  if (T_host && h->K_neq > 0)
    NEGF_CUDA_TRY(cudaMemcpyAsync(T_host, h->T_res, sizeof(double) * (size_t)h->C * h->K_neq,
                                  cudaMemcpyDeviceToHost, h->stream));
  return negf_sync(h);
}

extern "C" negf_status negf_kernel_stats(negf_handle* h, negf_kernel_stat* out, int32_t* count,
                                         int32_t reset) {
  if (!h || !count) { set_error("negf_kernel_stats: null argument"); return NEGF_EINVAL; }
  NEGF_CUDA_TRY(cudaStreamSynchronize(h->stream));
  prof_collect(h);
  const int cap = *count;
  int nout = 0;
  for (int k = 0; k < K_COUNT && out && nout < cap; ++k) {
    std::memset(&out[nout], 0, sizeof(negf_kernel_stat));
    std::strncpy(out[nout].name, kKernelNames[k], sizeof(out[nout].name) - 1);
    out[nout].launches = h->prof_launches[k];
    out[nout].total_ms = h->prof_ms[k];
    ++nout;
  }
  *count = out ? nout : K_COUNT;
  if (reset) {
    for (int k = 0; k < K_COUNT; ++k) { h->prof_launches[k] = 0; h->prof_ms[k] = 0.0; }
  }
  return NEGF_OK;
}

extern "C" negf_status negf_get_plan(negf_handle* h, negf_plan_info* out) {
  if (!h || !out) { set_error("negf_get_plan: null argument"); return NEGF_EINVAL; }
  std::memset(out, 0, sizeof(*out));
  out->sweeps_per_charge = h->C * h->n_modes * (h->K_eq + h->K_neq);
  if (h->scalar) {
    out->history_bytes = h->hist_bytes;
    out->partial_bytes = h->partial_bytes;
    out->n_batches = (int32_t)h->batches.size();
    // negate + per batch (real-axis sweep [+ contour sweep + contour combine]) + 2-level row reduce + mode reduce
    int launches = 1 + 3;
    const int wpc = h->cwarps_per_channel + 2 * h->rwarps_per_channel;
    for (const Batch& b : h->batches) {
      bool has_c = false, has_r = false;
      for (int w = b.warp_begin; w < b.warp_end && !(has_c && has_r); ++w)
        ((w % wpc) < h->cwarps_per_channel ? has_c : has_r) = true;
      launches += (has_r ? 1 : 0) + (has_c ? (h->seg_M ? 4 : 2) : 0);
    }
    out->kernel_launches = launches;
  } else {
    block_path_plan(h->block, out);
  }
  return NEGF_OK;
}
