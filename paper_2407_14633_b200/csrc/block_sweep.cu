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
#include "block_ops17.cuh"
#include "block_ops2.cuh"
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

// y[q][b] = - sum_{c in nz(K_rid)} K[rid][c] * X[c][b] for the thread's two rows (X in shared memory)
template <int NB>
__device__ __forceinline__ void sparse_left2(c64 (&y)[2][NB], const CsrS K, unsigned X, int a, bool valid1) {
  constexpr int TPT = Geo2<NB>::TPT;
#pragma unroll
  for (int q = 0; q < 2; ++q) {
#pragma unroll
    for (int b = 0; b < NB; ++b) y[q][b] = make_double2(0.0, 0.0);
    if (q == 1 && !valid1) continue;
    const int rid = a + q * TPT;
    const int e0 = lds_i32(K.rowptr + 4 * rid), e1 = lds_i32(K.rowptr + 4 * rid + 4);
#pragma unroll 1
    for (int e = e0; e < e1; ++e) {
      const c64 v = lds_c64(K.val + 16 * e);
      const unsigned xr = X + (unsigned)lds_i32(K.col + 4 * e) * (NB * 16);
#pragma unroll
      for (int b = 0; b < NB; ++b) cfms(y[q][b], v, lds_c64(xr + 16 * b));
    }
  }
}

// y[q][b] = sum_{d in nz(K_b)} X[rid][d] * conj(K[b][d])   (rows of X K^dagger from the thread's own rows
// of X in shared memory)
template <int NB>
__device__ __forceinline__ void sparse_right_dagger2(c64 (&y)[2][NB], const CsrS K, unsigned X, int a,
                                                     bool valid1) {
  constexpr int TPT = Geo2<NB>::TPT;
  const unsigned x0 = X + a * (NB * 16);
  const unsigned x1 = X + (valid1 ? a + TPT : a) * (NB * 16);
#pragma unroll
  for (int b = 0; b < NB; ++b) {
    c64 acc0 = make_double2(0.0, 0.0), acc1 = make_double2(0.0, 0.0);
    const int e0 = lds_i32(K.rowptr + 4 * b), e1 = lds_i32(K.rowptr + 4 * b + 4);
#pragma unroll 1
    for (int e = e0; e < e1; ++e) {
      const c64 kv = cconj(lds_c64(K.val + 16 * e));
      const unsigned cidx = 16u * (unsigned)lds_i32(K.col + 4 * e);
      cfma(acc0, lds_c64(x0 + cidx), kv);
      cfma(acc1, lds_c64(x1 + cidx), kv);
    }
    y[0][b] = acc0;
    y[1][b] = valid1 ? acc1 : make_double2(0.0, 0.0);
  }
}

template <int NB>
__global__ void __launch_bounds__(Geo2<NB>::THREADS, (NB >= 16 ? 4 : 1)) block_sweep_kernel(const SweepLaunch p) {
  using G = Geo2<NB>;
  constexpr int TPT = G::TPT;
  extern __shared__ __align__(16) char smem_raw[];
  Smem2<NB> sm;
  char* nxt = sm.carve(smem_raw);
  const int tid = threadIdx.x;
  const bool live = tid < G::LIVE;
  const int t = live ? tid / TPT : 0;
  const int a = tid % TPT;
  const bool valid1 = a + TPT < NB;
  const int rid1 = valid1 ? a + TPT : a;            // clamped row index for address computations
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
  // Long-lived pointers are re-derived where they are used (ring 0, ring N-1, the history stores): the
  // elimination loop needs every register it can get for the matrix rows and the pivot-row loads.
  const size_t tab_off = (((size_t)id.c * K_all + kk) * 2 + 0) * 2 * G::MAT;
#define NEGF_TAB_FIRST (p.table + tab_off + (dir ? 2 * G::MAT : 0))
#define NEGF_TAB_LAST (p.table + tab_off + (dir ? 0 : 2 * G::MAT))

  // couplings of this direction, by parity of the bond: [0] even bond, [1] odd bond
  Csr Kgen[2];
  CsrS Kpar[2];
  c64* kd[2];                       // their diagonals (used when the coupling is a diagonal matrix)
  bool kdiag[2];
  {
    const int m0 = dir ? CSR_E : CSR_EDAG, m1 = dir ? CSR_O : CSR_ODAG;
    nxt = csr_to_shared(Kgen[0], nxt, p.csr.rowptr + m0 * (NB + 1), p.csr.col + (size_t)m0 * p.csr.nnz_cap,
                        p.csr.val + (size_t)m0 * p.csr.nnz_cap, NB, p.csr.nnz_cap);
    nxt = csr_to_shared(Kgen[1], nxt, p.csr.rowptr + m1 * (NB + 1), p.csr.col + (size_t)m1 * p.csr.nnz_cap,
                        p.csr.val + (size_t)m1 * p.csr.nnz_cap, NB, p.csr.nnz_cap);
    Kpar[0] = csr_shared(Kgen[0]);
    Kpar[1] = csr_shared(Kgen[1]);
    kd[0] = reinterpret_cast<c64*>(nxt);
    kd[1] = kd[0] + NB;
    for (int i = tid; i < NB; i += G::THREADS) {
      kd[0][i] = p.csr.diag[m0 * NB + i];
      kd[1][i] = p.csr.diag[m1 * NB + i];
    }
    kdiag[0] = (p.csr.diag_mask >> m0) & 1;
    kdiag[1] = (p.csr.diag_mask >> m1) & 1;
  }
  __syncthreads();

  c64* mat_t = sm.mat + (size_t)t * G::MAT;
  const unsigned mat_s = smem_addr(mat_t);
  c64* hb = p.hist + (size_t)blockIdx.x * N * G::STEP_ELEMS + tid;   // + ((s*2 + q)*NB + b) * THREADS
  constexpr size_t HQ = (size_t)NB * G::THREADS;                     // offset of the second row slot

  // ------------------------------------------------------------------ connected Green's functions
  // Loop invariant at the top of step s > 0: d = the thread's rows of ytilde_{s-1}; if the coupling
  // entering step s is not diagonal, ytilde_{s-1} is also in the task's exchange matrix.
  c64 d[2][NB];
  // n = 17, real-axis CTAs: ytilde_s goes out row-major (row stride 18: rows start on 32-byte sectors)
  // with 32-byte stores, one full sector per lane and instruction; block_back.cu reads it back as
  // DMMA fragments.  (16-byte stores at row-strided addresses cost 2.4x the L2 write sectors.)
  auto store_row17 = [&](c64* dst, const c64 (&row)[NB]) {
#pragma unroll
    for (int j = 0; j < 8; ++j)
      asm volatile("st.global.v4.f64 [%0], {%1, %2, %3, %4};" ::"l"(dst + 2 * j), "d"(row[2 * j].x),
                   "d"(row[2 * j].y), "d"(row[2 * j + 1].x), "d"(row[2 * j + 1].y)
                   : "memory");
    // the 17th element together with the padding element 17: a full 32-byte sector, so that L2 does not
    // have to fetch the other half from DRAM (the 16-byte tail store cost 9.2 GB of reads per config-4 launch)
    asm volatile("st.global.v4.f64 [%0], {%1, %2, %3, %4};" ::"l"(dst + 16), "d"(row[NB - 1].x), "d"(row[NB - 1].y),
                 "d"(0.0), "d"(0.0)
                 : "memory");
  };
  auto store_history = [&](const c64 (&y)[2][NB], int s) {
    if (!live) return;
    c64* hp = hb + (size_t)s * G::STEP_ELEMS;
    if constexpr (NB == 17) {
      c64* hrec = hp - tid + (size_t)t * kHistRec17;
      store_row17(hrec + a * kHistLd17, y[0]);
      if (valid1) store_row17(hrec + rid1 * kHistLd17, y[1]);
    } else {
#pragma unroll
      for (int b = 0; b < NB; ++b) {
        hp[(size_t)b * G::THREADS] = y[0][b];
        if (valid1) hp[HQ + (size_t)b * G::THREADS] = y[1][b];
      }
    }
  };
  for (int s = 0; s < N; ++s) {
    const int i = dir ? N - 1 - s : s;
    if (s == 0) {
#pragma unroll
      for (int b = 0; b < NB; ++b) {
        const c64 s0 = NEGF_TAB_FIRST[a * NB + b], s1 = NEGF_TAB_FIRST[rid1 * NB + b];
        d[0][b] = make_double2(-s0.x, -s0.y);
        d[1][b] = valid1 ? make_double2(-s1.x, -s1.y) : make_double2(0.0, 0.0);
      }
    } else {
      const int par = dir ? (i & 1) : ((i - 1) & 1);
      // d := -K_s ytilde_{s-1} (the sign is folded into the product)
      if (kdiag[par]) {
        const c64 k0 = kd[par][a], k1 = kd[par][rid1];             // (K ytilde)_ab = K_aa ytilde_ab
        const c64 n0 = make_double2(-k0.x, -k0.y), n1 = make_double2(-k1.x, -k1.y);
#pragma unroll
        for (int b = 0; b < NB; ++b) {
          d[0][b] = cmul(n0, d[0][b]);
          d[1][b] = cmul(n1, d[1][b]);
        }
      } else {
        sparse_left2<NB>(d, Kpar[par], mat_s, a, valid1);          // -K_s ytilde_{s-1}
      }
      if (contour) {
        if (live) {                                                // the combine kernel reads +K ytilde
          c64* hp = hb + (size_t)s * G::STEP_ELEMS;
#pragma unroll
          for (int b = 0; b < NB; ++b) {
            hp[(size_t)b * G::THREADS] = make_double2(-d[0][b].x, -d[0][b].y);
            if (valid1) hp[HQ + (size_t)b * G::THREADS] = make_double2(-d[1][b].x, -d[1][b].y);
          }
        }
        if (s == N - 1) break;
      }
    }
    if (!contour && s == N - 1) {
#pragma unroll
      for (int b = 0; b < NB; ++b) {
        const c64 s0 = NEGF_TAB_LAST[a * NB + b], s1 = NEGF_TAB_LAST[rid1 * NB + b];
        d[0][b].x -= s0.x;
        d[0][b].y -= s0.y;
        if (valid1) { d[1][b].x -= s1.x; d[1][b].y -= s1.y; }
      }
    }
    const double zu = z.x - p.U[(size_t)id.c * N + i];
#pragma unroll
    for (int b = 0; b < NB; ++b) {
      if (b == a) { d[0][b].x += zu; d[0][b].y += z.y; }
      if (b == a + TPT) { d[1][b].x += zu; d[1][b].y += z.y; }
    }
    const bool permuted = gj_invert2<NB>(d, sm, t, a, live, p.theta2);
    int parn = 0;
    bool next_diag = false;
    if (s < N - 1) {
      const int inext = dir ? i - 1 : i + 1;
      parn = dir ? (inext & 1) : ((inext - 1) & 1);
      next_diag = kdiag[parn];
    }
    if (s == N - 1 || next_diag) {
      if (permuted) {                                              // rare: undo the implicit row order
        store_inverse2<NB>(d, mat_t, sm, t, a, live, true);
        __syncthreads();
#pragma unroll
        for (int b = 0; b < NB; ++b) {
          d[0][b] = mat_t[a * NB + b];
          d[1][b] = valid1 ? mat_t[rid1 * NB + b] : make_double2(0.0, 0.0);
        }
      }
      if (s < N - 1) {
        const c64* kdn = kd[parn];                                 // ytilde_ab = g_ab conj(K_bb)
#pragma unroll
        for (int b = 0; b < NB; ++b) {
          const c64 kb = cconj(kdn[b]);
          d[0][b] = cmul(d[0][b], kb);
          d[1][b] = cmul(d[1][b], kb);
        }
      }                                                            // last ring: G_(k,k) itself
      if (!contour) store_history(d, s);
      __syncthreads();                                             // separates consecutive gj_invert2 calls
    } else {
      store_inverse2<NB>(d, mat_t, sm, t, a, live, permuted);
      __syncthreads();
      sparse_right_dagger2<NB>(d, Kpar[parn], mat_s, a, valid1);   // ytilde_s = g_s K_{s+1}^dagger
      if (!contour) store_history(d, s);
      if (live) {                                                  // only this thread reads its rows above
#pragma unroll
        for (int b = 0; b < NB; ++b) {
          mat_t[a * NB + b] = d[0][b];
          if (valid1) mat_t[rid1 * NB + b] = d[1][b];
        }
      }
      __syncthreads();
    }
  }
  if (contour) return;
  if constexpr (NB == 17) return;   // the way back runs on the tensor cores: block_back.cu

  // ------------------------------------------------------------------ column recursion back
  const int R = p.geq + 2 * p.gneq;
  double* prow_out = p.partial + ((size_t)id.c * R + p.geq + 2 * id.grp + dir) * N;
  const double f_last = fermi(z.x, dir ? p.mu_s : p.mu_d, p.kT);
  const double wt = active ? p.deg * p.w_neq[k] * (1.0 / (2.0 * kPi)) * f_last : 0.0;
  {
    const c64* F_last = NEGF_TAB_LAST + G::MAT;
    if (live) {
#pragma unroll
      for (int b = 0; b < NB; ++b) {
        mat_t[a * NB + b] = F_last[a * NB + b];
        if (valid1) mat_t[rid1 * NB + b] = F_last[rid1 * NB + b];
      }
    }
  }
  // The thread's two rows of ytilde_s stream through registers one column at a time.  Three register
  // pairs P[0..2] hold columns 3g, 3g+1, 3g+2 of the current group; each is refilled, right after its
  // use, with the column three slots ahead (a ring is padded to NG*3 slots so that the slot -> register
  // assignment is static; the loop over groups is not unrolled: instruction-cache footprint).
  constexpr int NG = (NB + 2) / 3;
  const c64* pf = hb + (size_t)(N - 1) * G::STEP_ELEMS;   // prefetch cursor: ring pf_ring, slot pf_kq
  int pf_ring = N - 1, pf_kq = 0;
  c64 P[3][2];
  auto fetch = [&](c64 (&dst)[2]) {
    if (pf_kq < NB) {
      dst[0] = pf[0];
      dst[1] = valid1 ? pf[HQ] : make_double2(0.0, 0.0);
    }
    pf += G::THREADS;
    if (++pf_kq == 3 * NG) {
      pf_kq = 0;
      pf -= (size_t)3 * NG * G::THREADS;
      if (pf_ring > 0) { --pf_ring; pf -= G::STEP_ELEMS; }
    }
  };
  fetch(P[0]);
  fetch(P[1]);
  fetch(P[2]);
  __syncthreads();
  c64 cc[2][NB];
  for (int s = N - 1; s >= 0; --s) {
    const int i = dir ? N - 1 - s : s;
#pragma unroll
    for (int b = 0; b < NB; ++b) cc[0][b] = cc[1][b] = make_double2(0.0, 0.0);
#pragma unroll 1
    for (int g = 0; g < NG; ++g) {
#pragma unroll
      for (int u = 0; u < 3; ++u) {
        const int kq = 3 * g + u;
        const c64 av0 = P[u][0], av1 = P[u][1];
        fetch(P[u]);
        if (kq < NB) {
          const c64* brow = mat_t + kq * NB;
          c64 bv[NB];
#pragma unroll
          for (int b = 0; b < NB; ++b) bv[b] = brow[b];
#pragma unroll
          for (int b = 0; b < NB; ++b) {
            cfma(cc[0][b], av0, bv[b]);
            cfma(cc[1][b], av1, bv[b]);
          }
        }
      }
    }
    double v = 0.0;
#pragma unroll
    for (int b = 0; b < NB; ++b) v += cabs2(cc[0][b]) + cabs2(cc[1][b]);
    v = live ? wt * v : 0.0;
    if (p.probe && i == p.probe_ring) {                            // per-task value (CTA-uniform branch)
      if (live) sm.mag[t * NB + a] = v;
      __syncthreads();
      if (a == 0 && active) {
        double tot = 0.0;
        for (int r = 0; r < TPT; ++r) tot += sm.mag[t * NB + r];
        p.probe[((size_t)id.c * 2 + dir) * p.K_neq + k] = tot;
      }
    }
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
        for (int b = 0; b < NB; ++b) {
          mat_t[a * NB + b] = cc[0][b];
          if (valid1) mat_t[rid1 * NB + b] = cc[1][b];
        }
      }
      __syncthreads();
    }
  }
  // ------------------------------------------------------------------ transmission (direction 0)
  if (dir == 0) {
    const c64* F_first = NEGF_TAB_FIRST + G::MAT;
    if (live) {
#pragma unroll
      for (int b = 0; b < NB; ++b) {                               // C_0 = G_(0,N-1) F_R
        mat_t[a * NB + b] = cc[0][b];
        if (valid1) mat_t[rid1 * NB + b] = cc[1][b];
      }
    }
    __syncthreads();
#pragma unroll
    for (int b = 0; b < NB; ++b) cc[0][b] = cc[1][b] = make_double2(0.0, 0.0);
    for (int c2 = 0; c2 < NB; ++c2) {                              // rows of F_first^dagger C_0
      const c64 f0 = cconj(F_first[c2 * NB + a]);
      const c64 f1 = valid1 ? cconj(F_first[c2 * NB + rid1]) : make_double2(0.0, 0.0);
#pragma unroll
      for (int b = 0; b < NB; ++b) {
        const c64 bv = mat_t[c2 * NB + b];
        cfma(cc[0][b], f0, bv);
        cfma(cc[1][b], f1, bv);
      }
    }
    double v = 0.0;
#pragma unroll
    for (int b = 0; b < NB; ++b) v += cabs2(cc[0][b]) + cabs2(cc[1][b]);
    if (live) sm.mag[t * NB + a] = v;
    __syncthreads();
    if (a == 0 && active) {
      double tot = 0.0;
      for (int r = 0; r < TPT; ++r) tot += sm.mag[t * NB + r];
      p.T[(size_t)id.c * p.K_neq + k] = tot;
    }
  }
}

#undef NEGF_TAB_FIRST
#undef NEGF_TAB_LAST

// Contour combine: G_(i,i) = [alpha_i - x_i - y_i]^-1 (Alg.1 step 1) and the first term
// of eq.(4): -(deg/pi) Im[W_k Tr G_(i,i)].  grid = (ring chunks, pairs of contour sweep CTAs).
template <int NB>
__global__ void __launch_bounds__(Geo2<NB>::THREADS, (NB >= 16 ? 4 : 1))
block_combine_kernel(const SweepLaunch p, long long pair_cta_begin, int rings_per_cta) {
  using G = Geo2<NB>;
  constexpr int TPT = G::TPT;
  extern __shared__ __align__(16) char smem_raw[];
  Smem2<NB> sm;
  sm.carve(smem_raw);
  const int tid = threadIdx.x;
  const bool live = tid < G::LIVE;
  const int t = live ? tid / TPT : 0;
  const int a = tid % TPT;
  const bool valid1 = a + TPT < NB;
  const int rid1 = valid1 ? a + TPT : a;
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
  constexpr size_t HQ = (size_t)NB * G::THREADS;
  c64* mat_t = sm.mat + (size_t)t * G::MAT;
  const int R = p.geq + 2 * p.gneq;
  double* prow_out = p.partial + ((size_t)id.c * R + id.grp) * N;

  const int i0 = blockIdx.x * rings_per_cta;
  const int i1 = min(N, i0 + rings_per_cta);
  for (int i = i0; i < i1; ++i) {
    c64 d[2][NB];
    const c64* pl = hL + (size_t)i * G::STEP_ELEMS;
    const c64* pr = hR + (size_t)(N - 1 - i) * G::STEP_ELEMS;
#pragma unroll
    for (int b = 0; b < NB; ++b) {
      const c64 yl0 = (i == 0) ? tabL[a * NB + b] : pl[(size_t)b * G::THREADS];
      const c64 xr0 = (i == N - 1) ? tabR[a * NB + b] : pr[(size_t)b * G::THREADS];
      d[0][b] = make_double2(-yl0.x - xr0.x, -yl0.y - xr0.y);
      if (valid1) {
        const c64 yl1 = (i == 0) ? tabL[rid1 * NB + b] : pl[HQ + (size_t)b * G::THREADS];
        const c64 xr1 = (i == N - 1) ? tabR[rid1 * NB + b] : pr[HQ + (size_t)b * G::THREADS];
        d[1][b] = make_double2(-yl1.x - xr1.x, -yl1.y - xr1.y);
      } else {
        d[1][b] = make_double2(0.0, 0.0);
      }
    }
    const double zu = z.x - Uc[i];
#pragma unroll
    for (int b = 0; b < NB; ++b) {
      if (b == a) { d[0][b].x += zu; d[0][b].y += z.y; }
      if (b == a + TPT) { d[1][b].x += zu; d[1][b].y += z.y; }
    }
    const bool permuted = gj_invert2<NB>(d, sm, t, a, live, p.theta2);
    c64 gaa = make_double2(0.0, 0.0);
    if (!permuted) {
#pragma unroll
      for (int b = 0; b < NB; ++b) {
        if (b == a) { gaa.x += d[0][b].x; gaa.y += d[0][b].y; }
        if (b == a + TPT) { gaa.x += d[1][b].x; gaa.y += d[1][b].y; }
      }
    } else {
      store_inverse2<NB>(d, mat_t, sm, t, a, live, true);
      __syncthreads();
      gaa = mat_t[a * NB + a];
      if (valid1) { gaa.x += mat_t[rid1 * NB + rid1].x; gaa.y += mat_t[rid1 * NB + rid1].y; }
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
  return Smem2<NB>::bytes() + 2 * csr_shared_bytes(NB, nnz_cap) + 2 * NB * sizeof(c64) + 32;
}

template <int NB>
static cudaError_t launch_sweep_t(const SweepLaunch& p, cudaStream_t s) {
  using G = Geo2<NB>;
  const size_t smem = sweep_smem_t<NB>(p.csr.nnz_cap);
  cudaError_t e = cudaFuncSetAttribute(block_sweep_kernel<NB>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e != cudaSuccess) return e;
  block_sweep_kernel<NB><<<p.n_cta, G::THREADS, smem, s>>>(p);
  return cudaGetLastError();
}

template <int NB>
static cudaError_t launch_combine_t(const SweepLaunch& p, long long pair_cta_begin, int n_pairs, cudaStream_t s) {
  using G = Geo2<NB>;
  const size_t smem = Smem2<NB>::bytes();
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
  if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, block_sweep_kernel<NB>, Geo2<NB>::THREADS, smem) !=
      cudaSuccess)
    return 0;
  return nb;
}

cudaError_t launch_block_sweep(int nb, const SweepLaunch& p, cudaStream_t s) {
  if (nb == 17) {
    // contour CTAs of the range: this file's kernel; real-axis CTAs: block_fwd17.cu, then block_back.cu
    const long long eq_end = p.cta_begin + p.n_cta < p.n_eq_cta ? p.cta_begin + p.n_cta : p.n_eq_cta;
    if (eq_end > p.cta_begin) {
      SweepLaunch q = p;
      q.n_cta = (int)(eq_end - p.cta_begin);
      cudaError_t e = launch_sweep_t<17>(q, s);
      if (e != cudaSuccess) return e;
    }
    cudaError_t e = launch_block_fwd17(p, s);
    return e != cudaSuccess ? e : launch_block_back17(p, s);
  }
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
#define NEGF_CASE(NB_) case NB_: return Geo2<NB_>::TPC;
    NEGF_BLOCK_SIZES(NEGF_CASE)
#undef NEGF_CASE
    default: return 0;
  }
}
int block_tasks_per_cta_real(int nb) { return nb == 17 ? kTpc17 : block_tasks_per_cta(nb); }
int block_threads(int nb) {
  switch (nb) {
#define NEGF_CASE(NB_) case NB_: return Geo2<NB_>::THREADS;
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
int block_sweep_ctas_per_sm(int nb, int nnz_cap, int row_nnz_max) {
  if (nb == 17) {                      // both forward kernels must fit; the real-axis one carries the load
    const int a = ctas_per_sm_t<17>(nnz_cap), b = block_fwd17_ctas_per_sm(row_nnz_max);
    return a < 1 ? a : b;
  }
  switch (nb) {
#define NEGF_CASE(NB_) case NB_: return ctas_per_sm_t<NB_>(nnz_cap);
    NEGF_BLOCK_SIZES(NEGF_CASE)
#undef NEGF_CASE
    default: return 0;
  }
}
long long block_step_elems(int nb) {
  switch (nb) {
#define NEGF_CASE(NB_) case NB_: return Geo2<NB_>::STEP_ELEMS;
    NEGF_BLOCK_SIZES(NEGF_CASE)
#undef NEGF_CASE
    default: return 0;
  }
}
bool block_size_supported(int nb) { return block_tasks_per_cta(nb) > 0; }

}  // namespace blk
}  // namespace negf
