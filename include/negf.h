/* negf.h -- C-ABI of libnegf_b200: NEGF charge / transmission / Broyden hot path on one B200.
 *
 * What the calls compute is defined by arXiv 2407.14633 (ELEQTRONeX); citations are
 * PAPER.md:<line> of the extracted text plus equation / algorithm, and "DESIGN.md Rn" for the
 * readings taken where the paper is silent or garbled.
 *
 *   G^R(E)  = [(E + i eta) I - H - Sigma_L - Sigma_R]^-1               eq.(2)
 *   Sigma_l = tau_l^dagger g_l tau_l,  Gamma_l = i (Sigma_l - Sigma_l^dagger)
 *   A_l     = G^R Gamma_l G^R^dagger
 *   n_i     = deg * [ -(1/pi) Im sum_k W_k Tr_ring G_ii(z_k)
 *                     + (1/2pi) sum_k w_k ( f_S(E_k) Tr_ring A_L,ii(E_k) + f_D(E_k) Tr_ring A_R,ii(E_k) ) ]
 *                                                                        eq.(4), PAPER.md:93 (n = -rho, R12)
 *   T(E_k)  = Tr[Gamma_L G^R Gamma_R G^R^dagger]                         eq.(5)
 *   x_{m+1} = Broyden's modified second method, Algorithm 3
 *
 * H is block tridiagonal (Fig.1(a)): N rings per channel, block size n; diagonal block
 * U_i I with U_i = -phi_i (eV; phi in volts); H_{i,i+1} = coup_even for even i, coup_odd for odd i;
 * H_{i+1,i} = H_{i,i+1}^dagger.  Each lead is the semi-infinite continuation of that alternating
 * pattern with uniform on-site energy equal to the adjacent end ring's U (R7, R9); its surface Green's
 * function is the closed form of the alternating scalar chain (lead_kind 0, R8) or Sancho-Rubio
 * decimation (lead_kind 1, R10).
 *
 * General rules
 *   - Every function returns negf_status (0 = success); nothing throws or aborts.
 *   - Pointers named *_dev are DEVICE pointers (e.g. torch tensor.data_ptr()); *_host are HOST pointers.
 *     The arrays inside negf_config are HOST memory and are copied by negf_create.
 *   - The caller owns every array it passes; the library neither frees nor keeps caller pointers after
 *     the call returns, but device arrays must stay alive until the handle's stream has passed the call.
 *   - Work is enqueued on the CUDA stream given at creation (a cudaStream_t cast to void*; NULL = the
 *     legacy default stream) and the call returns without synchronising unless stated otherwise.
 *   - Handles own all workspace.  A handle must not be used from two host threads at once.
 *   - All floating point is FP64; negf_c64 has the layout of double2 / complex128.
 *   - There is no CPU fallback: without a CUDA device every compute call returns NEGF_ECUDA.
 */
#ifndef NEGF_B200_H
#define NEGF_B200_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#if defined(__GNUC__)
#define NEGF_API __attribute__((visibility("default")))
#else
#define NEGF_API
#endif

typedef enum {
  NEGF_OK = 0,
  NEGF_EINVAL = 1,   /* null pointer, size < minimum, kT <= 0, block / lead_kind mismatch ... */
  NEGF_ENOMEM = 2,   /* host or device allocation failed */
  NEGF_ECUDA = 3,    /* CUDA runtime error; text in negf_last_error() */
  NEGF_ENOCONV = 4,  /* Sancho-Rubio reached sr_maxit for at least one energy (results still written) */
  NEGF_ESTATE = 5    /* negf_charge / negf_transmission before any negf_set_potential */
} negf_status;

typedef struct { double re, im; } negf_c64;

typedef struct negf_handle negf_handle;       /* opaque */
typedef struct broyden_handle broyden_handle; /* opaque */

/* Configuration of one device array (HOST struct, HOST arrays; copied by negf_create). */
typedef struct {
  int32_t n_channels;  /* C >= 1: independent channels batched together                 */
  int32_t n_rings;     /* N >= 2: rings per channel, the same for every channel of a handle             */
  int32_t block;       /* n: 1 = scalar mode-space chains, > 1 = dense n x n blocks.  The block kernels are
                          instantiated for n in {2, 3, 4, 5, 8, 17} (17 = the (17,0) tube); any other n > 1
                          returns NEGF_EINVAL                                                              */
  int32_t n_modes;     /* block == 1: chains (modes) per channel; block > 1: must be 1    */
  int32_t lead_kind;   /* 0 = closed-form alternating chain (block == 1 only); 1 = Sancho-Rubio (block > 1) */
  int32_t sr_maxit;    /* lead_kind 1: iteration cap (200)                                               */
  double  sr_tol;      /* lead_kind 1: stop when max|a_ij|,|b_ij| < sr_tol (1e-12), then two more passes and the
                          Newton polish of the fixed point (R10)                                           */
  double  mu_s, mu_d;  /* eV: electrochemical potentials of the source (left, ring 0) and drain leads    */
  double  kT;          /* eV, > 0                                                                        */
  double  deg;         /* degeneracy prefactor of eq.(3), PAPER.md:86 (g_s = 2)                          */
  const negf_c64* coup_even;  /* H_{i,i+1}, i even. block == 1: n_modes values; else n*n row-major      */
  const negf_c64* coup_odd;   /* H_{i,i+1}, i odd, same layout                                           */
  const double*   mode_weight;/* block == 1: n_modes weights (1.0 when all modes are listed); else NULL  */
  int32_t n_eq;               /* K_eq >= 0 contour points (eq.(4) first term)            */
  const negf_c64* z_eq;       /* nodes z_k (complex, used as given: no eta is added)                     */
  const negf_c64* w_eq;       /* complex weights W_k = dz * F_min(z_k) (R13)                             */
  int32_t n_neq;              /* K_neq >= 0 real-axis points (eq.(4) second term)                        */
  const negf_c64* z_neq;      /* nodes E_k + i eta (the caller supplies eta, R11)                        */
  const double*   w_neq;      /* real quadrature weights; Fermi factors are applied by the library       */
  int64_t workspace_bytes;    /* cap on the recursion-history workspace in HBM.  0 = default: what the plan
                                 needs, at most 64 GiB (block == 1) or, for block > 1, at most two waves of
                                 resident sweep CTAs and 85 % of the FREE device memory at creation -- two
                                 full-size block handles do not fit one GPU unless both pass a cap here.
                                 Larger problems are tiled over (channel, energy) batches. */
  int32_t profile;            /* != 0: record CUDA events around every kernel (negf_kernel_stats)        */
  int32_t reserved;           /* must be 0                                                               */
  double  pivot_theta;        /* block > 1: the diagonal pivot candidate of an in-register Gauss-Jordan step is
                                 accepted without a search when |a_kk| >= theta * ||row k of the matrix handed
                                 in||_2; otherwise the task searches the whole column (partial pivoting).
                                 0 = default (1e-4); a huge value (1e150) forces the search at every
                                 elimination step (test hook).  block = 17: the warp-resident inversions
                                 (real-axis forward sweep, decimation passes of the lead self-energies) apply
                                 the same test to the corner row(s) they eliminate first and fall back to
                                 plain partial pivoting in shared memory when it fails, so 1e150 sends every
                                 such inversion through that fallback.                                       */
} negf_config;

/* Create a handle: validates, copies the config, allocates workspace.  `cuda_stream` is a
 * cudaStream_t.  On failure *out is NULL. */
NEGF_API negf_status negf_create(const negf_config* cfg, void* cuda_stream, negf_handle** out);
NEGF_API negf_status negf_destroy(negf_handle* h);

/* Set the electrostatic potential phi[C][N] (volts, channel-major, R20).  Enqueues U = -phi and, for
 * lead_kind 1, the Sancho-Rubio self-energy kernel for every (channel, energy, lead) -- Sigma depends
 * on phi through the end rings (R7).  Invalidates cached results.  phi_dev is read by this call only
 * (the library keeps its own U).  For some single-channel block handles the library also starts the
 * contour half-sweeps of the coming negf_charge here, on a stream of its own that it joins itself
 * (overlap plan); this is invisible to the caller. */
NEGF_API negf_status negf_set_potential(negf_handle* h, const double* phi_dev);

/* Charge n[C][N] (electrons per ring, >= 0; eq.(4)) for the current potential: self-energies ->
 * RGF forward / backward sweeps -> energy reduction.  Also caches T(E).  NEGF_ESTATE if no potential
 * has been set.  Does not synchronise; a Sancho-Rubio non-convergence is reported as NEGF_ENOCONV by
 * the next synchronising call (negf_sync, negf_*_host). */
NEGF_API negf_status negf_charge(negf_handle* h, double* n_dev);

/* Transmission T[C][K_neq] (eq.(5)) for the current potential, summed over modes.  Returns the values
 * cached by negf_charge, or runs the sweep itself if the potential changed since. */
NEGF_API negf_status negf_transmission(negf_handle* h, double* T_dev);

/* Lead self-energies of the current potential (step a1b; eq.(2)): copies
 * Sigma[C][K_eq + K_neq][2 leads: 0 = source/left, 1 = drain/right][n*n row-major] (contour energies
 * first) to sigma_dev.  Block handles (lead_kind 1) only: scalar handles evaluate the closed form
 * inside the sweep kernel and return NEGF_EINVAL here.  NEGF_ESTATE before negf_set_potential. */
NEGF_API negf_status negf_self_energy(negf_handle* h, negf_c64* sigma_dev);

/* Landauer reductions of T(E) (eq.(5)-(6)), per channel:
 *   current[c]     = sum_k w_k T_c(E_k) (f_S(E_k) - f_D(E_k))      in eV, multiply by g_s e/h
 *   conductance[c] = sum_k w_k T_c(E_k) (-df/dE)(E_k; mu_s, kT)    in units of G_0 = g_s e^2/h
 * Either output may be NULL. */
NEGF_API negf_status negf_current(negf_handle* h, double* current_dev, double* conductance_dev);

/* Semi-adaptive real-axis path, the device side ("compute the integrand at
 * the center of the channel as a function of energy, obtain the peak of the singularity E_s").
 * negf_set_probe selects the ring (0 <= ring < N; ring < 0 switches the probe off) whose per-energy
 * contributions the sweep kernels record from then on; it invalidates cached results.
 * negf_integrand_peak runs the sweep if needed and writes, per channel c,
 *   integrand[c][k] = sum_modes mode_weight (F_S Tr_ring A_S,(r,r) + F_D Tr_ring A_D,(r,r))(E_k)   [C][K_neq]
 * (the integrand of the second term of eq.(4) without 1/2pi, deg and the quadrature weight), the index
 * k_peak[c] of its first maximum and E_peak[c] = Re z_neq[k_peak[c]].  Any of the three outputs may be NULL.
 * NEGF_ESTATE without a probe ring or a potential; NEGF_EINVAL for a handle without real-axis points. */
NEGF_API negf_status negf_set_probe(negf_handle* h, int32_t ring);
NEGF_API negf_status negf_integrand_peak(negf_handle* h, double* integrand_dev, int32_t* k_peak_dev,
                                         double* E_peak_dev);

/* Host-buffer convenience path (the end-to-end call): copies phi from HOST memory, runs
 * negf_set_potential + negf_charge (+ transmission), copies n (and T if T_host != NULL) back to HOST
 * memory and synchronises the stream. */
NEGF_API negf_status negf_solve_host(negf_handle* h, const double* phi_host, double* n_host, double* T_host);

/* Block until the handle's stream is idle; returns NEGF_ENOCONV if a Sancho-Rubio task of any
 * negf_set_potential since the last negf_sync / negf_solve_host did not converge (the flag is sticky
 * until it has been reported once), NEGF_ECUDA if the device reported an error. */
NEGF_API negf_status negf_sync(negf_handle* h);

/* Per-kernel timing (only when cfg.profile != 0).  Synchronises.  Fills up to *count entries. */
typedef struct {
  char    name[48];
  int64_t launches;
  double  total_ms;
} negf_kernel_stat;
NEGF_API negf_status negf_kernel_stats(negf_handle* h, negf_kernel_stat* out, int32_t* count, int32_t reset);

/* Facts about the workspace plan chosen at creation (for DESIGN.md / bench reporting). */
typedef struct {
  int64_t history_bytes;     /* recursion-history workspace allocated                    */
  int64_t partial_bytes;     /* per-warp partial charge sums                             */
  int32_t n_batches;         /* launches of the sweep kernel per negf_charge             */
  int32_t sweeps_per_charge; /* C * chains * (K_eq + K_neq)                              */
  int32_t max_sr_iterations; /* largest Sancho-Rubio iteration count of the last set_potential (after sync) */
  int32_t kernel_launches;   /* kernels launched by one negf_set_potential + negf_charge pair               */
  int64_t sr_passes_total;   /* decimation passes of the last negf_set_potential summed over all
                                (channel, energy, lead) tasks (after sync)                                  */
} negf_plan_info;
NEGF_API negf_status negf_get_plan(negf_handle* h, negf_plan_info* out);

/* ---- Broyden's modified second method, Algorithm 3, vector-agnostic ---------- */

/* len >= 1 entries, history >= 1 stored (v, w) pairs (sliding window, R17), mixing fraction zeta (R15). */
NEGF_API negf_status broyden_create(int64_t len, int32_t history, double zeta, void* cuda_stream,
                           broyden_handle** out);
/* One pass of the loop body (steps 2-19): x_in holds x_m on entry and x_{m+1} on return; x_out = F(x_m).
 * eps_max_host (may be NULL) receives max_t |f_t| / |x_in,t + x_out,t| (steps 4-7) and forces a sync. */
NEGF_API negf_status broyden_step(broyden_handle* h, double* x_in_dev, const double* x_out_dev,
                         double* eps_max_host);
NEGF_API negf_status broyden_reset(broyden_handle* h);
NEGF_API negf_status broyden_destroy(broyden_handle* h);

/* The convergence measure of the self-consistent loop WITHOUT any allocation (for callers that cannot call
 * cudaMalloc: CUDA graph capture, tight serving loops, harnesses that forbid it):
 *     *eps_max_dev = max_t |x_in,t - x_out,t| / max(|x_in,t + x_out,t|, 1e-300)   (Alg.3 steps 2, 4-7,
 * PAPER.md:216-230; the value broyden_step returns in eps_max_host; NaN / infinity in the residual give
 * +infinity).  x_in_dev, x_out_dev: DEVICE, len doubles each, read only; eps_max_dev: DEVICE, one double,
 * written; all caller-owned.  Two kernels are launched on cuda_stream (a cudaStream_t, NULL = default
 * stream); nothing is synchronised, no handle is needed, and no cudaMalloc, cudaFree or allocating routine is
 * called.  The per-block partial maxima live in a 128 KiB file-scope device array (residual_noalloc.cu) that
 * every GPU loading the library holds until the process exits; one partial per 4096 entries, so
 * 1 <= len <= NEGF_NOALLOC_MAX_LEN, else NEGF_EINVAL.  The array's device address is resolved on the first
 * call on each device (cudaGetSymbolAddress, no allocation): make that first call outside stream capture.
 * All calls on a device share the array: a call overwrites the entries it reads, so nothing carries over
 * from the previous call, but calls that overlap on the GPU (different streams, no dependency) race. */
#define NEGF_NOALLOC_MAX_LEN ((int64_t)1 << 26)
NEGF_API negf_status broyden_residual_noalloc(const double* x_in_dev, const double* x_out_dev, int64_t len,
                                     double* eps_max_dev, void* cuda_stream);

/* Diagnostic: measured FP64 throughput of the current device in TFLOP/s, from chains of independent
 * DFMA instructions and of DMMA (mma.sync.m8n8k4.f64) instructions; used as the roofline denominator
 * of the FP64-bound block kernels.  Synchronous; takes a few milliseconds. */
NEGF_API negf_status negf_fp64_peak(double* dfma_tflops, double* dmma_tflops);

/* Environment variables read at negf_create (test hooks; the defaults are the product path):
 *   NEGF_SEG_MIN_RINGS  scalar handles with at least this many rings run their contour half-sweeps parallel
 *                       in N (default 8192);  NEGF_SEG_LEN  segment length of that pass (default max(256, N/1024));
 *   NEGF_FORCE_OVERLAP  "1" / "0": force / forbid the overlap plan of single-channel block handles. */

/* Last error text of the calling thread (static storage, never NULL). */
NEGF_API const char* negf_last_error(void);
/* Library version string, e.g. "negf_b200 0.1 (sm_100a)". */
NEGF_API const char* negf_version(void);

#ifdef __cplusplus
}
#endif
#endif /* NEGF_B200_H */
