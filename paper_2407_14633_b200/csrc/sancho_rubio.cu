// Lead self-energies of the block path by Sancho-Rubio decimation (step a1b of SURVEY.md 8(a);
// PAPER.md:117 "decimation technique [33,34]"; readings R7, R9, R10) and the factor F of
// Gamma = i (Sigma - Sigma^dagger) = F F^dagger that the sweep kernel propagates.
//
// The lead is a semi-infinite stack of rings r0 (surface), r1, r2, ... with uniform on-site energy
// U and alternating hoppings V0 = H_{r0,r1}, V1 = H_{r1,r2}, V0, ...  Because every on-site block is
// U I, the odd rings are eliminated in closed form first (w = 1/(z - U)):
//     eps_s = U + w V0 V0^dagger,   eps = U + w (V1^dagger V1 + V0 V0^dagger),
//     a = w V0 V1,                  b = w V1^dagger V0^dagger,
// which leaves an n x n chain (not the 2n x 2n principal layer) for the decimation loop
//     g = (z - eps)^-1;  eps_s += a g b;  eps += a g b + b g a;  a <- a g a;  b <- b g b
// until max|a_ij|, |b_ij| < sr_tol, plus two more passes (quadratic convergence: the fixed point is
// then exact to rounding, so the result does not depend on the route taken to it).
// g_surf = (z - eps_s)^-1,  Sigma = L g_surf R  with (L, R) = (tau^dagger, tau).
#include "block_ops.cuh"
#include "block_path.h"
#include "negf_internal.h"

namespace negf {
namespace blk {

template <int NB>
__global__ void __launch_bounds__(Geo<NB>::THREADS, 1) sancho_rubio_kernel(const SrLaunch p) {
  using G = Geo<NB>;
  extern __shared__ __align__(16) char smem_raw[];
  Smem<NB> sm;
  sm.carve(smem_raw, 3);
  const int tid = threadIdx.x;
  const bool live = tid < G::LIVE;
  const int t = live ? tid / NB : 0;
  const int a = tid % NB;
  c64* bufG = sm.mat + (size_t)t * G::MAT;
  c64* bufA = sm.mat + ((size_t)G::TPC + t) * G::MAT;
  c64* bufB = sm.mat + ((size_t)2 * G::TPC + t) * G::MAT;

  const int K_all = p.K_eq + p.K_neq;
  const long long n_task = (long long)p.C * K_all * 2;
  long long task = (long long)blockIdx.x * G::TPC + t;
  const bool active = live && task < n_task;
  if (task >= n_task) task = n_task - 1;
  const int lead = (int)(task & 1);
  const long long ck = task >> 1;
  const int c = (int)(ck / K_all);
  const int kk = (int)(ck - (long long)c * K_all);
  const c64 z = kk < p.K_eq ? p.z_eq[kk] : p.z_neq[kk - p.K_eq];
  const double U = p.U[(size_t)c * p.N + (lead ? p.N - 1 : 0)];
  const c64 w = crcp(make_double2(z.x - U, z.y));
  const c64* lm = p.lead_mats + (size_t)lead * 6 * G::MAT;   // P00, PE, PA, PB, L, R (row-major)

  c64 eps_s[NB], eps[NB];
#pragma unroll
  for (int b = 0; b < NB; ++b) {
    eps_s[b] = cmul(w, lm[0 * G::MAT + a * NB + b]);
    eps[b] = cmul(w, lm[1 * G::MAT + a * NB + b]);
    if (b == a) { eps_s[b].x += U; eps[b].x += U; }
    if (live) {
      bufA[a * NB + b] = cmul(w, lm[2 * G::MAT + a * NB + b]);
      bufB[a * NB + b] = cmul(w, lm[3 * G::MAT + a * NB + b]);
    }
  }
  int remaining = -1;       // -1: criterion not met yet; >= 0: passes still to do after it was met
  int iters = 0;
  bool frozen = false;
  __syncthreads();

  for (int it = 0; it < p.maxit + 2; ++it) {
    c64 d[NB];
#pragma unroll
    for (int b = 0; b < NB; ++b) d[b] = make_double2((b == a ? z.x : 0.0) - eps[b].x, (b == a ? z.y : 0.0) - eps[b].y);
    const bool permuted = gj_invert<NB>(d, sm, t, a, live, p.theta2);
    store_inverse<NB>(d, bufG, sm, t, a, live, permuted);
    __syncthreads();
    c64 ag[NB], bg[NB];
    {
      c64 row[NB];
#pragma unroll
      for (int k = 0; k < NB; ++k) row[k] = bufA[a * NB + k];
      gemm_row<NB>(ag, row, bufG);
#pragma unroll
      for (int k = 0; k < NB; ++k) row[k] = bufB[a * NB + k];
      gemm_row<NB>(bg, row, bufG);
    }
    __syncthreads();                       // bufG is free from here on
    double rowmax = 0.0;
    c64 nb_[NB];
    {
      c64 tmp[NB];
      gemm_row<NB>(tmp, ag, bufB);         // a g b
      if (!frozen) {
#pragma unroll
        for (int b = 0; b < NB; ++b) {
          eps_s[b].x += tmp[b].x; eps_s[b].y += tmp[b].y;
          eps[b].x += tmp[b].x;   eps[b].y += tmp[b].y;
        }
      }
      gemm_row<NB>(tmp, bg, bufA);         // b g a
      if (!frozen) {
#pragma unroll
        for (int b = 0; b < NB; ++b) { eps[b].x += tmp[b].x; eps[b].y += tmp[b].y; }
      }
      gemm_row<NB>(tmp, ag, bufA);         // a g a -> new a, parked in bufG
#pragma unroll
      for (int b = 0; b < NB; ++b) {
        if (frozen) tmp[b] = make_double2(0.0, 0.0);
        rowmax = fmax(rowmax, fmax(fabs(tmp[b].x), fabs(tmp[b].y)));
        if (live) bufG[a * NB + b] = tmp[b];
      }
      gemm_row<NB>(nb_, bg, bufB);         // b g b -> new b
#pragma unroll
      for (int b = 0; b < NB; ++b) {
        if (frozen) nb_[b] = make_double2(0.0, 0.0);
        rowmax = fmax(rowmax, fmax(fabs(nb_[b].x), fabs(nb_[b].y)));
      }
    }
    if (live) sm.mag[t * NB + a] = rowmax;
    __syncthreads();                       // everyone is done reading bufA / bufB
#pragma unroll
    for (int b = 0; b < NB; ++b) {
      if (live) {
        bufB[a * NB + b] = nb_[b];
        bufA[a * NB + b] = bufG[a * NB + b];   // own row only
      }
    }
    double tmax = 0.0;
#pragma unroll
    for (int i = 0; i < NB; ++i) tmax = fmax(tmax, sm.mag[t * NB + i]);
    if (!frozen) {
      ++iters;
      if (remaining < 0) {
        if (tmax < p.tol) remaining = 2;
      } else {
        --remaining;
      }
      if (remaining == 0) frozen = true;
    }
    if (__syncthreads_and(frozen || !live)) break;
  }
  if (active && a == 0) {
    atomicMax(p.max_iters, iters);
    if (!frozen) atomicExch(p.noconv_flag, 1);
  }

  // ---- surface Green's function and Sigma = L g R
  c64 srow[NB];
  {
    c64 d[NB];
#pragma unroll
    for (int b = 0; b < NB; ++b)
      d[b] = make_double2((b == a ? z.x : 0.0) - eps_s[b].x, (b == a ? z.y : 0.0) - eps_s[b].y);
    const bool permuted = gj_invert<NB>(d, sm, t, a, live, p.theta2);
    store_inverse<NB>(d, bufG, sm, t, a, live, permuted);
#pragma unroll
    for (int b = 0; b < NB; ++b)
      if (live) bufA[a * NB + b] = lm[5 * G::MAT + a * NB + b];     // R
    __syncthreads();
    c64 grow[NB], t1[NB];
#pragma unroll
    for (int k = 0; k < NB; ++k) grow[k] = bufG[a * NB + k];
    gemm_row<NB>(t1, grow, bufA);                                    // g R
#pragma unroll
    for (int b = 0; b < NB; ++b)
      if (live) bufB[a * NB + b] = t1[b];
    __syncthreads();
#pragma unroll
    for (int k = 0; k < NB; ++k) grow[k] = lm[4 * G::MAT + a * NB + k];   // L row
    gemm_row<NB>(srow, grow, bufB);                                  // L g R
  }
  c64* out = p.table + (size_t)task * 2 * G::MAT;
#pragma unroll
  for (int b = 0; b < NB; ++b) {
    if (active) out[a * NB + b] = srow[b];
    if (live) bufG[a * NB + b] = srow[b];
  }
  __syncthreads();

  // ---- Gamma = i (Sigma - Sigma^dagger) and its pivoted Cholesky factor, Gamma = F F^dagger
  c64 S[NB], F[NB];
#pragma unroll
  for (int b = 0; b < NB; ++b) {
    const c64 sba = bufG[b * NB + a];
    S[b] = make_double2(-(srow[b].y + sba.y), srow[b].x - sba.x);
    F[b] = make_double2(0.0, 0.0);
  }
  bool usedc = false;
#pragma unroll
  for (int j = 0; j < NB; ++j) {
    double diag = 0.0;
#pragma unroll
    for (int b = 0; b < NB; ++b)
      if (b == a) diag = S[b].x;
    if (live) sm.mag[t * NB + a] = usedc ? -1.0 : diag;
    __syncthreads();
    int piv = 0;
    double dmax = sm.mag[t * NB];
#pragma unroll
    for (int i = 1; i < NB; ++i) {
      const double v = sm.mag[t * NB + i];
      if (v > dmax) { dmax = v; piv = i; }
    }
    c64* prow = sm.prow + ((size_t)(j & 1) * G::TPC + t) * NB;
    if (a == piv && live) {
#pragma unroll
      for (int b = 0; b < NB; ++b) prow[b] = S[b];
    }
    __syncthreads();
    if (dmax > 0.0) {
      const double rs = 1.0 / sqrt(dmax);
      c64 la;
      if (a == piv) {
        la = make_double2(dmax * rs, 0.0);
        usedc = true;
      } else if (usedc) {
        la = make_double2(0.0, 0.0);
      } else {
        const c64 cp = prow[a];
        la = make_double2(cp.x * rs, -cp.y * rs);         // S[a][piv] / sqrt(d) = conj(S[piv][a]) / sqrt(d)
        const c64 f = make_double2(la.x * rs, la.y * rs);
#pragma unroll
        for (int b = 0; b < NB; ++b) cfms(S[b], f, prow[b]);   // S[a][b] -= L_a conj(L_b)
      }
      F[j] = la;
    }
  }
#pragma unroll
  for (int b = 0; b < NB; ++b)
    if (active) out[G::MAT + a * NB + b] = F[b];
}

template <int NB>
static cudaError_t launch_sr_t(const SrLaunch& p, cudaStream_t s) {
  using G = Geo<NB>;
  const size_t smem = Smem<NB>::bytes(3);
  static bool attr_set = false;
  if (!attr_set) {
    cudaError_t e = cudaFuncSetAttribute(sancho_rubio_kernel<NB>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         (int)smem);
    if (e != cudaSuccess) return e;
    attr_set = true;
  }
  const long long n_task = (long long)p.C * (p.K_eq + p.K_neq) * 2;
  const int blocks = (int)((n_task + G::TPC - 1) / G::TPC);
  sancho_rubio_kernel<NB><<<blocks, G::THREADS, smem, s>>>(p);
  return cudaGetLastError();
}

cudaError_t launch_sancho_rubio(int nb, const SrLaunch& p, cudaStream_t s) {
  switch (nb) {
#define NEGF_CASE(NB_) case NB_: return launch_sr_t<NB_>(p, s);
    NEGF_BLOCK_SIZES(NEGF_CASE)
#undef NEGF_CASE
    default: return cudaErrorInvalidValue;
  }
}

}  // namespace blk
}  // namespace negf
