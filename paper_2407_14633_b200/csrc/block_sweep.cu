// Block RGF sweep kernels: steps a2, a3, a4 and the first stage of a5 of SURVEY.md 8(a) for dense
// n x n blocks (BASELINE.json configs[2..4]).
//
// Formulation.  With H = -M off the diagonal and K_s the coupling that
// enters ring s of a half-sweep from the ring before it (direction 0: K_s = H_{i-1,i}^dagger, i = s;
// direction 1: K_s = H_{i,i+1}, i = N-1-s), a half-sweep task runs Algorithm 2
//     g_s      = [ (z - U_i) I - Sigma_first [s=0] - Sigma_last [s=N-1] - K_s ytilde_{s-1} ]^-1
//     ytilde_s = g_s K_{s+1}^dagger                      (the paper's ytilde / xtilde, history in HBM)
// away from its first lead, then the column recursion of Algorithm 1 steps 2-3 and 6-8
// back from the last lead k,
//     C_{N-1} = g_{N-1} F_k,   C_s = ytilde_s C_{s+1}    (C_s = G_(i,k) F_k,  Gamma_k = F_k F_k^dagger)
//     Tr A_k,(i,i) = ||C_s||_F^2,   T = ||F_first^dagger C_0||_F^2   (eq.(5))
// Contour points need Tr G_(i,i) = Tr [alpha_i - x_i - y_i]^-1 (Alg.1 step 1): their two half-sweeps
// store x_i / y_i = K_s ytilde_{s-1} and a second kernel (parallel over rings) inverts and traces.
#include "block_ops.cuh"
#include "block_path.h"
#include "negf_internal.h"

namespace negf {
namespace blk {

constexpr double kPi = 3.14159265358979323846;

struct CtaId {
  bool contour;
  int c, grp, dir;
};
__device__ __forceinline__ CtaId decode_cta(const SweepLaunch& p, long long gid) {
  const long long n_eq_cta = (long long)p.C * p.geq * 2;
  CtaId id;
  id.contour = gid < n_eq_cta;
  const long long r = id.contour ? gid : gid - n_eq_cta;
  const int per = 2 * (id.contour ? p.geq : p.gneq);
  id.c = (int)(r / per);
  const int rem = (int)(r - (long long)id.c * per);
  id.grp = rem >> 1;
  id.dir = rem & 1;
  return id;
}

template <int NB>
__global__ void __launch_bounds__(Geo<NB>::THREADS, 2) block_sweep_kernel(const SweepLaunch p) {
  using G = Geo<NB>;
  extern __shared__ __align__(16) char smem_raw[];
  Smem<NB> sm;
  char* nxt = sm.carve(smem_raw, 1);
  const int tid = threadIdx.x;
  const bool live = tid < G::LIVE;
  const int t = live ? tid / NB : 0;
  const int a = tid % NB;
  const int lane = tid & 31, warp = tid >> 5;
  const int N = p.N;

  const CtaId id = decode_cta(p, p.cta_begin + blockIdx.x);
  const bool contour = id.contour;
  const int dir = id.dir;
  const int K = contour ? p.K_eq : p.K_neq;
  int k = id.grp * G::TPC + t;
  const bool active = live && k < K;
  if (k >= K) k = K - 1;
  const int kk = contour ? k : p.K_eq + k;
  const c64 z = contour ? p.z_eq[k] : p.z_neq[k];
  const size_t K_all = (size_t)p.K_eq + p.K_neq;
  const c64* tabL = p.table + (((size_t)id.c * K_all + kk) * 2 + 0) * 2 * G::MAT;
  const c64* tabR = tabL + 2 * G::MAT;
  const c64* tab_first = dir ? tabR : tabL;
  const c64* tab_last = dir ? tabL : tabR;
  const double* Uc = p.U + (size_t)id.c * N;

  // couplings of this direction, by parity of the bond: [0] even bond, [1] odd bond
  Csr Kpar[2];
  c64* kd[2];                       // their diagonals (used when the coupling is a diagonal matrix)
  bool kdiag[2];
  {
    const int m0 = dir ? CSR_E : CSR_EDAG, m1 = dir ? CSR_O : CSR_ODAG;
    nxt = csr_to_shared(Kpar[0], nxt, p.csr.rowptr + m0 * (NB + 1), p.csr.col + (size_t)m0 * p.csr.nnz_cap,
                        p.csr.val + (size_t)m0 * p.csr.nnz_cap, NB, p.csr.nnz_cap);
    nxt = csr_to_shared(Kpar[1], nxt, p.csr.rowptr + m1 * (NB + 1), p.csr.col + (size_t)m1 * p.csr.nnz_cap,
                        p.csr.val + (size_t)m1 * p.csr.nnz_cap, NB, p.csr.nnz_cap);
    kd[0] = reinterpret_cast<c64*>(nxt);
    kd[1] = kd[0] + NB;
    if (tid < NB) {
      kd[0][tid] = p.csr.diag[m0 * NB + tid];
      kd[1][tid] = p.csr.diag[m1 * NB + tid];
    }
    kdiag[0] = (p.csr.diag_mask >> m0) & 1;
    kdiag[1] = (p.csr.diag_mask >> m1) & 1;
  }
  __syncthreads();

  c64* mat_t = sm.mat + (size_t)t * G::MAT;
  c64* hb = p.hist + (size_t)blockIdx.x * N * G::STEP_ELEMS + tid;   // + (s * NB + b) * THREADS

  // ------------------------------------------------------------------ connected Green's functions
  // Loop invariant at the top of step s > 0: d = row a of ytilde_{s-1} in registers; if the coupling
  // entering step s is not diagonal, ytilde_{s-1} is also in the task's exchange matrix.
  c64 d[NB];
  c64* hp = hb;
  for (int s = 0; s < N; ++s, hp += G::STEP_ELEMS) {
    const int i = dir ? N - 1 - s : s;
    if (s == 0) {
#pragma unroll
      for (int b = 0; b < NB; ++b) {
        const c64 sg = tab_first[a * NB + b];
        d[b] = make_double2(-sg.x, -sg.y);
      }
    } else {
      const int par = dir ? (i & 1) : ((i - 1) & 1);
      if (kdiag[par]) {
        const c64 ka = kd[par][a];                                 // (K ytilde)_ab = K_aa ytilde_ab
#pragma unroll
        for (int b = 0; b < NB; ++b) d[b] = cmul(ka, d[b]);
      } else {
        sparse_left<NB>(d, Kpar[par], mat_t, a);                   // K_s ytilde_{s-1}
      }
      if (contour) {
#pragma unroll
        for (int b = 0; b < NB; ++b) hp[(size_t)b * G::THREADS] = d[b];
        if (s == N - 1) break;
      }
#pragma unroll
      for (int b = 0; b < NB; ++b) d[b] = make_double2(-d[b].x, -d[b].y);
    }
    if (!contour && s == N - 1) {
#pragma unroll
      for (int b = 0; b < NB; ++b) {
        const c64 sg = tab_last[a * NB + b];
        d[b].x -= sg.x;
        d[b].y -= sg.y;
      }
    }
    const double zu = z.x - Uc[i];
#pragma unroll
    for (int b = 0; b < NB; ++b)
      if (b == a) { d[b].x += zu; d[b].y += z.y; }
    const bool permuted = gj_invert<NB>(d, sm, t, a, live, p.theta2);
    int parn = 0;
    bool next_diag = false;
    if (s < N - 1) {
      const int inext = dir ? i - 1 : i + 1;
      parn = dir ? (inext & 1) : ((inext - 1) & 1);
      next_diag = kdiag[parn];
    }
    if (s == N - 1 || next_diag) {
      if (permuted) {                                              // rare: undo the implicit row order
        store_inverse<NB>(d, mat_t, sm, t, a, live, true);
        __syncthreads();
#pragma unroll
        for (int b = 0; b < NB; ++b) d[b] = mat_t[a * NB + b];
      }
      if (s < N - 1) {
        const c64* kdn = kd[parn];                                 // ytilde_ab = g_ab conj(K_bb)
#pragma unroll
        for (int b = 0; b < NB; ++b) d[b] = cmul(d[b], cconj(kdn[b]));
      }                                                            // last ring: G_(k,k) itself
      if (!contour) {
#pragma unroll
        for (int b = 0; b < NB; ++b) hp[(size_t)b * G::THREADS] = d[b];
      }
      __syncthreads();                                             // separates consecutive gj_invert calls
    } else {
      store_inverse<NB>(d, mat_t, sm, t, a, live, permuted);
      __syncthreads();
      sparse_right_dagger<NB>(d, Kpar[parn], mat_t + a * NB);      // ytilde_s = g_s K_{s+1}^dagger
      if (!contour) {
#pragma unroll
        for (int b = 0; b < NB; ++b) hp[(size_t)b * G::THREADS] = d[b];
      }
      if (live) {                                                  // only this thread reads row a above
#pragma unroll
        for (int b = 0; b < NB; ++b) mat_t[a * NB + b] = d[b];
      }
      __syncthreads();
    }
  }
  if (contour) return;

  // ------------------------------------------------------------------ column recursion back
  const int R = p.geq + 2 * p.gneq;
  double* prow_out = p.partial + ((size_t)id.c * R + p.geq + 2 * id.grp + dir) * N;
  const double f_last = fermi(z.x, dir ? p.mu_s : p.mu_d, p.kT);
  const double wt = active ? p.deg * p.w_neq[k] * (1.0 / (2.0 * kPi)) * f_last : 0.0;
  {
    const c64* F_last = tab_last + G::MAT;
    if (live) {
#pragma unroll
      for (int b = 0; b < NB; ++b) mat_t[a * NB + b] = F_last[a * NB + b];
    }
  }
  c64 A[NB];
#pragma unroll
  for (int kq = 0; kq < NB; ++kq) A[kq] = hb[((size_t)(N - 1) * NB + kq) * G::THREADS];
  __syncthreads();
  c64 cc[NB];
  for (int s = N - 1; s >= 0; --s) {
    const int i = dir ? N - 1 - s : s;
    const c64* hnext = hb + (size_t)(s > 0 ? s - 1 : 0) * NB * G::THREADS;
#pragma unroll
    for (int b = 0; b < NB; ++b) cc[b] = make_double2(0.0, 0.0);
#pragma unroll
    for (int kq = 0; kq < NB; ++kq) {
      const c64 av = A[kq];
      A[kq] = hnext[(size_t)kq * G::THREADS];                     // prefetch ring s-1 of the history
#pragma unroll
      for (int b = 0; b < NB; ++b) cfma(cc[b], av, mat_t[kq * NB + b]);
    }
    double v = 0.0;
#pragma unroll
    for (int b = 0; b < NB; ++b) v += cabs2(cc[b]);
    v = live ? wt * v : 0.0;
    v = warp_sum(v);
    if (lane == 0) sm.red[(s & 1) * G::NWARPS + warp] = v;
    __syncthreads();
    if (tid == 0) {
      double tot = 0.0;
#pragma unroll
      for (int w = 0; w < G::NWARPS; ++w) tot += sm.red[(s & 1) * G::NWARPS + w];
      prow_out[i] = tot;
    }
    if (s > 0) {
      if (live) {
#pragma unroll
        for (int b = 0; b < NB; ++b) mat_t[a * NB + b] = cc[b];
      }
      __syncthreads();
    }
  }
  // ------------------------------------------------------------------ transmission (direction 0)
  if (dir == 0) {
    const c64* F_first = tab_first + G::MAT;
    if (live) {
#pragma unroll
      for (int b = 0; b < NB; ++b) mat_t[a * NB + b] = cc[b];      // C_0 = G_(0,N-1) F_R
    }
    __syncthreads();
#pragma unroll
    for (int b = 0; b < NB; ++b) cc[b] = make_double2(0.0, 0.0);
    for (int c2 = 0; c2 < NB; ++c2) {
      const c64 f = cconj(F_first[c2 * NB + a]);
#pragma unroll
      for (int b = 0; b < NB; ++b) cfma(cc[b], f, mat_t[c2 * NB + b]);
    }
    double v = 0.0;
#pragma unroll
    for (int b = 0; b < NB; ++b) v += cabs2(cc[b]);
    if (live) sm.mag[t * NB + a] = v;
    __syncthreads();
    if (a == 0 && active) {
      double tot = 0.0;
      for (int r = 0; r < NB; ++r) tot += sm.mag[t * NB + r];
      p.T[(size_t)id.c * p.K_neq + k] = tot;
    }
  }
}

// Contour combine: G_(i,i) = [alpha_i - x_i - y_i]^-1 (Alg.1 step 1) and the first term
// of eq.(4): -(deg/pi) Im[W_k Tr G_(i,i)].  grid = (ring chunks, pairs of contour sweep CTAs).
template <int NB>
__global__ void __launch_bounds__(Geo<NB>::THREADS, 2)
block_combine_kernel(const SweepLaunch p, long long pair_cta_begin, int rings_per_cta) {
  using G = Geo<NB>;
  extern __shared__ __align__(16) char smem_raw[];
  Smem<NB> sm;
  sm.carve(smem_raw, 1);
  const int tid = threadIdx.x;
  const bool live = tid < G::LIVE;
  const int t = live ? tid / NB : 0;
  const int a = tid % NB;
  const int lane = tid & 31, warp = tid >> 5;
  const int N = p.N;
  const long long gid = pair_cta_begin + 2 * (long long)blockIdx.y;
  const CtaId id = decode_cta(p, gid);
  const size_t slotL = (size_t)(gid - p.cta_begin);
  int k = id.grp * G::TPC + t;
  const bool active = live && k < p.K_eq;
  if (k >= p.K_eq) k = p.K_eq - 1;
  const c64 z = p.z_eq[k];
  const c64 W = p.w_eq[k];
  const double wc = active ? -p.deg / kPi : 0.0;
  const size_t K_all = (size_t)p.K_eq + p.K_neq;
  const c64* tabL = p.table + (((size_t)id.c * K_all + k) * 2 + 0) * 2 * G::MAT;
  const c64* tabR = tabL + 2 * G::MAT;
  const double* Uc = p.U + (size_t)id.c * N;
  const c64* hL = p.hist + slotL * N * G::STEP_ELEMS + tid;
  const c64* hR = p.hist + (slotL + 1) * N * G::STEP_ELEMS + tid;
  c64* mat_t = sm.mat + (size_t)t * G::MAT;
  const int R = p.geq + 2 * p.gneq;
  double* prow_out = p.partial + ((size_t)id.c * R + id.grp) * N;

  const int i0 = blockIdx.x * rings_per_cta;
  const int i1 = min(N, i0 + rings_per_cta);
  for (int i = i0; i < i1; ++i) {
    c64 d[NB];
#pragma unroll
    for (int b = 0; b < NB; ++b) {
      const c64 yl = (i == 0) ? tabL[a * NB + b] : hL[((size_t)i * NB + b) * G::THREADS];
      const c64 xr = (i == N - 1) ? tabR[a * NB + b] : hR[((size_t)(N - 1 - i) * NB + b) * G::THREADS];
      d[b] = make_double2(-yl.x - xr.x, -yl.y - xr.y);
    }
    const double zu = z.x - Uc[i];
#pragma unroll
    for (int b = 0; b < NB; ++b)
      if (b == a) { d[b].x += zu; d[b].y += z.y; }
    const bool permuted = gj_invert<NB>(d, sm, t, a, live, p.theta2);
    c64 gaa = make_double2(0.0, 0.0);
    if (!permuted) {
#pragma unroll
      for (int b = 0; b < NB; ++b)
        if (b == a) gaa = d[b];
    } else {
      store_inverse<NB>(d, mat_t, sm, t, a, live, true);
      __syncthreads();
      gaa = mat_t[a * NB + a];
    }
    double v = live ? wc * (W.x * gaa.y + W.y * gaa.x) : 0.0;
    v = warp_sum(v);
    const int par = (i - i0) & 1;
    if (lane == 0) sm.red[par * G::NWARPS + warp] = v;
    __syncthreads();
    if (tid == 0) {
      double tot = 0.0;
#pragma unroll
      for (int w = 0; w < G::NWARPS; ++w) tot += sm.red[par * G::NWARPS + w];
      prow_out[i] = tot;
    }
  }
}

// ---------------------------------------------------------------------------------- host side

template <int NB>
static size_t sweep_smem_t(int nnz_cap) {
  return Smem<NB>::bytes(1) + 2 * csr_shared_bytes(NB, nnz_cap) + 2 * NB * sizeof(c64) + 32;
}

template <int NB>
static cudaError_t launch_sweep_t(const SweepLaunch& p, cudaStream_t s) {
  using G = Geo<NB>;
  const size_t smem = sweep_smem_t<NB>(p.csr.nnz_cap);
  cudaError_t e = cudaFuncSetAttribute(block_sweep_kernel<NB>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e != cudaSuccess) return e;
  block_sweep_kernel<NB><<<p.n_cta, G::THREADS, smem, s>>>(p);
  return cudaGetLastError();
}

template <int NB>
static cudaError_t launch_combine_t(const SweepLaunch& p, long long pair_cta_begin, int n_pairs, cudaStream_t s) {
  using G = Geo<NB>;
  const size_t smem = Smem<NB>::bytes(1);
  cudaError_t e = cudaFuncSetAttribute(block_combine_kernel<NB>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e != cudaSuccess) return e;
  const int rings_per_cta = 8;
  for (int done = 0; done < n_pairs; done += 65535) {
    const int np = n_pairs - done < 65535 ? n_pairs - done : 65535;
    dim3 grid((p.N + rings_per_cta - 1) / rings_per_cta, np);
    block_combine_kernel<NB><<<grid, G::THREADS, smem, s>>>(p, pair_cta_begin + 2LL * done, rings_per_cta);
    e = cudaGetLastError();
    if (e != cudaSuccess) return e;
  }
  return cudaSuccess;
}

template <int NB>
static int ctas_per_sm_t(int nnz_cap) {
  int nb = 0;
  const size_t smem = sweep_smem_t<NB>(nnz_cap);
  if (cudaFuncSetAttribute(block_sweep_kernel<NB>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) !=
      cudaSuccess)
    return 0;
  if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, block_sweep_kernel<NB>, Geo<NB>::THREADS, smem) !=
      cudaSuccess)
    return 0;
  return nb;
}

cudaError_t launch_block_sweep(int nb, const SweepLaunch& p, cudaStream_t s) {
  switch (nb) {
#define NEGF_CASE(NB_) case NB_: return launch_sweep_t<NB_>(p, s);
    NEGF_BLOCK_SIZES(NEGF_CASE)
#undef NEGF_CASE
    default: return cudaErrorInvalidValue;
  }
}
cudaError_t launch_block_combine(int nb, const SweepLaunch& p, long long pair_cta_begin, int n_pairs,
                                 cudaStream_t s) {
  switch (nb) {
#define NEGF_CASE(NB_) case NB_: return launch_combine_t<NB_>(p, pair_cta_begin, n_pairs, s);
    NEGF_BLOCK_SIZES(NEGF_CASE)
#undef NEGF_CASE
    default: return cudaErrorInvalidValue;
  }
}
int block_tasks_per_cta(int nb) {
  switch (nb) {
#define NEGF_CASE(NB_) case NB_: return Geo<NB_>::TPC;
    NEGF_BLOCK_SIZES(NEGF_CASE)
#undef NEGF_CASE
    default: return 0;
  }
}
int block_threads(int nb) {
  switch (nb) {
#define NEGF_CASE(NB_) case NB_: return Geo<NB_>::THREADS;
    NEGF_BLOCK_SIZES(NEGF_CASE)
#undef NEGF_CASE
    default: return 0;
  }
}
size_t block_sweep_smem(int nb, int nnz_cap) {
  switch (nb) {
#define NEGF_CASE(NB_) case NB_: return sweep_smem_t<NB_>(nnz_cap);
    NEGF_BLOCK_SIZES(NEGF_CASE)
#undef NEGF_CASE
    default: return 0;
  }
}
int block_sweep_ctas_per_sm(int nb, int nnz_cap) {
  switch (nb) {
#define NEGF_CASE(NB_) case NB_: return ctas_per_sm_t<NB_>(nnz_cap);
    NEGF_BLOCK_SIZES(NEGF_CASE)
#undef NEGF_CASE
    default: return 0;
  }
}
bool block_size_supported(int nb) { return block_tasks_per_cta(nb) > 0; }

}  // namespace blk
}  // namespace negf
