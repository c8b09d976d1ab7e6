// Lead self-energies of the block path by Sancho-Rubio decimation (step a1b of SURVEY.md 8(a);
// PAPER.md:117 "decimation technique [33,34]"; readings R7, R9, R10) and the factor F of
// Gamma = i (Sigma - Sigma^dagger) = F F^dagger that the sweep kernel propagates.
//
// The lead is a semi-infinite stack of rings r0 (surface), r1, r2, ... with uniform on-site energy
// U and alternating hoppings V0 = H_{r0,r1}, V1 = H_{r1,r2}, V0, ...  Its principal layer is the
// two-ring cell (r0, r1):  H00 = [[U, V0], [V0^+, U]],  H01 = [[0, 0], [V1, 0]].  Cells must hold an
// even number of rings: segments with an odd number of rings of a bipartite chain carry zero modes
// at z = U, so any decimation that isolates them (e.g. eliminating every other ring first) is
// singular in the middle of the energy window.
//
// Because H01 has a single non-zero n x n block, the decimation matrices keep that shape for ever,
//     a = |1> X <0|,  b = |0> Y <1|,   X = V1, Y = V1^+ initially,
// and with g = (z - eps)^-1 (2n x 2n, four n x n blocks g00 g01 g10 g11) one pass is
//     eps_11 += X g00 Y;  eps_s,11 += X g00 Y (= eps_11);  eps_00 += Y g11 X;  X <- X g01 X;  Y <- Y g10 Y,
// the off-diagonal blocks of eps staying V0, V0^+.  So the only 2n x 2n operation is the inversion;
// the eight products are n x n.  Loop until max|X_ij|, |Y_ij| < sr_tol, plus two more passes.
//
// Thread geometry: 2n threads per task, thread (h, a) owns row h n + a of the 2n x 2n matrix during
// the inversion (block_ops.cuh gj_invert<2n>) and row a of the n x n blocks of half h otherwise.
//
// The raw decimation is conditioning-limited (it inverts isolated 2^k-cell segments whose poles lie
// on the real axis, eta away from z): 1e-13 typical, 1e-8 next to such a pole.  It is therefore
// polished with Newton steps on the surface block X = g_surf,00, the only part the next cell sees:
//     G(X) = [z - H00 - |1> V1 X V1^+ <1|]^-1,   F(X) = G00 - X = 0,
//     dG00 = P dX Q,  P = G01 V1,  Q = V1^+ G10,   D - P D Q = G00 - X  summed by doubling
//     (D += P D Q;  P <- P^2;  Q <- Q^2),
// until the fixed-point residual is at rounding level (at most kNewtonMax passes).
#include <math_constants.h>

#include "block_ops.cuh"
#include "block_ops34.cuh"
#include "cgemm17.cuh"
#include "block_path.h"
#include "negf_internal.h"

namespace negf {
namespace blk {

constexpr int kNewtonMax = 4;
constexpr int kDoublingMax = 64;   // 2^64 terms of the Neumann series: beyond any 1/eta

// c[b] = sum_k arow[k] * X[k * LD + b]
template <int NB, int LD>
__device__ __forceinline__ void gemm_row_ld(c64 (&c)[NB], const c64 (&arow)[NB], const c64* X) {
#pragma unroll
  for (int b = 0; b < NB; ++b) c[b] = make_double2(0.0, 0.0);
#pragma unroll
  for (int k = 0; k < NB; ++k) {
    const c64 av = arow[k];
#pragma unroll
    for (int b = 0; b < NB; ++b) cfma(c[b], av, X[k * LD + b]);
  }
}
template <int NB>
__device__ __forceinline__ void row_from(c64 (&r)[NB], const c64* src) {
#pragma unroll
  for (int b = 0; b < NB; ++b) r[b] = src[b];
}
template <int NB>
__device__ __forceinline__ void row_to(c64* dst, const c64 (&r)[NB], bool pred) {
  if (!pred) return;
#pragma unroll
  for (int b = 0; b < NB; ++b) dst[b] = r[b];
}
template <int NB>
__device__ __forceinline__ double row_absmax(const c64 (&r)[NB]) {
  // fmax drops NaNs, so a row with a NaN or an infinity reports +infinity explicitly: every
  // convergence test downstream then fails instead of passing on garbage
  double m = 0.0;
  bool finite = true;
#pragma unroll
  for (int b = 0; b < NB; ++b) {
    const double v = fmax(fabs(r[b].x), fabs(r[b].y));
    finite = finite && (fabs(r[b].x) < CUDART_INF) && (fabs(r[b].y) < CUDART_INF);
    m = fmax(m, v);
  }
  return finite ? m : CUDART_INF;
}

template <int NB>
__global__ void __launch_bounds__(Geo<2 * NB>::THREADS, 1) sancho_rubio_kernel(const SrLaunch p) {
  constexpr int N2 = 2 * NB;
  using G2 = Geo<N2>;
  constexpr int MATN = NB * NB;
  extern __shared__ __align__(16) char smem_raw[];
  Smem<N2> sm;
  char* nxt = sm.carve(smem_raw, 1);
  const int tid = threadIdx.x;
  const bool live = tid < G2::LIVE;
  const int t = live ? tid / N2 : 0;
  const int r = tid % N2;
  const int h = r / NB;            // 0: rows of ring r0, 1: rows of ring r1
  const int a = r - h * NB;
  const bool live0 = live && h == 0;
  c64* Gt = sm.mat + (size_t)t * G2::MAT;                          // 2n x 2n, leading dimension N2
  c64* Xb = reinterpret_cast<c64*>(nxt) + (size_t)t * 2 * MATN;    // n x n
  c64* Yb = Xb + MATN;                                             // n x n
  c64* mine = h == 0 ? Yb : Xb;    // half 0 carries Y (-> eps_00, new Y), half 1 carries X
  c64* other = h == 0 ? Xb : Yb;
  // n = 17: the 34 x 34 inversions run one warp per task (block_ops34.cuh), on the matrix in shared memory
  int* perm34 = reinterpret_cast<int*>(reinterpret_cast<c64*>(nxt) + (size_t)G2::TPC * 2 * MATN);
  // the thread's row m of the 2n x 2n matrix -> the inverse in Gt; the caller places __syncthreads() after
  // fast: the decimation passes, whose result the Newton polish corrects; the surface Green's function and the
  // polish itself keep gj_invert (pivots in row order): the warp version, which takes rows 32, 33 first, left
  // T(E) of config 4 off by 3.6e-10 at one energy when it was used there too
  auto invert_to_Gt = [&](c64 (&m)[N2], bool fast) {
    if (NB == 17 && fast) {
      __syncthreads();                                             // nobody reads the old Gt any more
      row_to<N2>(Gt + r * N2, m, live);
      __syncthreads();
      const int warp = tid >> 5;
      if (warp < G2::TPC)
        invert34_w32(sm.mat + (size_t)warp * G2::MAT, perm34 + warp * 32, p.theta2, tid & 31);
    } else {
      const bool permuted = gj_invert<N2>(m, sm, t, r, live, p.theta2);
      store_inverse<N2>(m, Gt, sm, t, r, live, permuted);
    }
  };

  const int K_all = p.K_eq + p.K_neq;
  const long long n_task = p.task_end;
  long long task = p.task_begin + (long long)blockIdx.x * G2::TPC + t;
  const bool active = live && task < n_task;
  if (task >= n_task) task = n_task - 1;
  const int lead = (int)(task & 1);
  const long long ck = task >> 1;
  const int c = (int)(ck / K_all);
  const int kk = (int)(ck - (long long)c * K_all);
  const c64 z = kk < p.K_eq ? p.z_eq[kk] : p.z_neq[kk - p.K_eq];
  const double U = p.U[(size_t)c * p.N + (lead ? p.N - 1 : 0)];
  const c64* lm = p.lead_mats + (size_t)lead * kLeadMats * MATN;   // see block_path.h
  const c64* gL = lm + 4 * MATN;
  const c64* gR = lm + 5 * MATN;
  const c64* gV0 = lm + 6 * MATN;
  const c64* gV1 = lm + 7 * MATN;
  const c64* gV0d = lm + 8 * MATN;
  const c64* gV1d = lm + 9 * MATN;
  // this thread's row of the constant off-diagonal block of z - eps: -V0 (half 0) / -V0^+ (half 1)
  const c64* offrow = (h == 0 ? gV0 : gV0d) + a * NB;
  const c64* my_init = (h == 0 ? gV1d : gV1) + a * NB;

  // row r of z - eps:  half 0: [z - eps_00 | -V0],  half 1: [-V0^+ | z - eps_11]
  auto build_row = [&](c64 (&m)[N2], const c64 (&ediag)[NB], const c64 z) {
#pragma unroll
    for (int j = 0; j < NB; ++j) {
      const c64 dg = make_double2((j == a ? z.x : 0.0) - ediag[j].x, (j == a ? z.y : 0.0) - ediag[j].y);
      const c64 of = offrow[j];
      const c64 no = make_double2(-of.x, -of.y);
      m[j] = h == 0 ? dg : no;
      m[NB + j] = h == 0 ? no : dg;
    }
  };

  // Attempt 0 decimates at z itself.  Next to a pole of an isolated 2^k-cell segment the raw result can
  // be off by ~1e-7, enough to push the spectral radius of the Newton operator P (.) Q past 1 for
  // propagating modes (it is 1 - O(eta) at the fixed point), and then the doubling sum below diverges.
  // Such a task (rare) is redone with the decimation at z + i*shift, which is well conditioned, and
  // polished from there at the true z.  The whole CTA repeats; unaffected tasks recompute the same bits.
  bool diverged = false;
  double final_res = 0.0, final_scale = 1.0;
  c64* Pb = Gt;                    // staging inside Gt once the inverse has been consumed
  c64* Qb = Gt + MATN;
  c64* Tb = Gt + 2 * MATN;
  for (int attempt = 0; attempt < 2; ++attempt) {
  const c64 zd = diverged ? make_double2(z.x, z.y + p.shift) : z;
  bool div_now = false;
  // row a of eps_hh.  The surface block eps_s,11 receives the same increments X g00 Y as eps_11 and eps_s,00
  // stays U I, so eps_s needs no storage of its own.
  c64 eh[NB];
#pragma unroll
  for (int b = 0; b < NB; ++b) {
    eh[b] = make_double2(b == a ? U : 0.0, 0.0);
    if (live) mine[a * NB + b] = my_init[b];
  }
  int remaining = -1;  // -1: criterion not met yet; >= 0: passes still to do after it was met
  int iters = 0;
  bool frozen = false;
  __syncthreads();

  for (int it = 0; it < p.maxit + 2; ++it) {
    {
      c64 m[N2];
      build_row(m, eh, zd);
      invert_to_Gt(m, true);
    }
    __syncthreads();
    const int rb = (1 - h) * NB;   // half 0 works on g11 / g10, half 1 on g00 / g01
    c64 res[NB];
    if constexpr (NB == 17) {
      // The eight n x n products of the pass on the tensor cores (cgemm17.cuh), one warp per product, in place
      // in the blocks of Gt: first the four left factors X, Y, then the four right factors.  (As rows of
      // register products they were a quarter of the kernel's stall samples and 200 registers of live rows.)
      const int warp = tid >> 5, lane = tid & 31;
      c64* xy = reinterpret_cast<c64*>(nxt);
#pragma unroll 1
      for (int stage = 0; stage < 2; ++stage) {
#pragma unroll 1
        for (int item = warp; item < 4 * G2::TPC; item += G2::NWARPS) {
          const int tt = item >> 2, w = item & 3;            // w = 0: Y g11 (X), 1: X g00 (Y), 2: Y g10 (Y), 3: X g01 (X)
          c64* Xt = xy + (size_t)tt * 2 * MATN;
          c64* Yt = Xt + MATN;
          c64* blk = sm.mat + (size_t)tt * G2::MAT + (w == 0 ? NB * N2 + NB : w == 1 ? 0 : w == 2 ? NB * N2 : NB);
          if (stage == 0) cgemm17_warp((w & 1) ? Xt : Yt, NB, blk, N2, blk, N2, lane);
          else cgemm17_warp(blk, N2, (w == 0 || w == 3) ? Xt : Yt, NB, blk, N2, lane);
        }
        __syncthreads();
      }
      row_from<NB>(res, Gt + (rb + a) * N2 + rb);            // Y g11 X | X g00 Y
      if (!frozen) {
#pragma unroll
        for (int b = 0; b < NB; ++b) {
          eh[b].x += res[b].x; eh[b].y += res[b].y;
        }
      }
      row_from<NB>(res, Gt + (rb + a) * N2 + (NB - rb));     // Y g10 Y | X g01 X
    } else {
      c64 ar[NB], pq[NB];
      row_from<NB>(ar, mine + a * NB);
      gemm_row_ld<NB, N2>(pq, ar, Gt + rb * N2 + rb);          // Y g11   | X g00
      gemm_row<NB>(res, pq, other);                            // Y g11 X | X g00 Y
      if (!frozen) {
#pragma unroll
        for (int b = 0; b < NB; ++b) {
          eh[b].x += res[b].x; eh[b].y += res[b].y;
        }
      }
      gemm_row_ld<NB, N2>(pq, ar, Gt + rb * N2 + (NB - rb));   // Y g10   | X g01
      gemm_row<NB>(res, pq, mine);                             // Y g10 Y | X g01 X
    }
    if (frozen) {
#pragma unroll
      for (int b = 0; b < NB; ++b) res[b] = make_double2(0.0, 0.0);
    }
    if (live) sm.mag[t * N2 + r] = row_absmax<NB>(res);
    __syncthreads();                                         // all reads of Gt, Xb, Yb done
    row_to<NB>(mine + a * NB, res, live);
    double tmax = 0.0;
#pragma unroll
    for (int i = 0; i < N2; ++i) tmax = fmax(tmax, sm.mag[t * N2 + i]);
    if (!frozen) {
      ++iters;
      if (!(tmax < CUDART_INF)) {            // the decimation broke down (z on a pole of a segment)
        div_now = true;
        frozen = true;
      } else if (remaining < 0) {
        if (tmax < p.tol) remaining = 2;
      } else {
        --remaining;
      }
      if (remaining == 0) frozen = true;
    }
    if (__syncthreads_and(frozen || !live)) break;
  }
  if (active && r == 0) {
    atomicMax(p.max_iters, iters);
    atomicAdd(p.iters_total, (unsigned long long)iters);
    if (!frozen) atomicExch(p.noconv_flag, 1);
  }

  // ---- surface Green's function of the layer: (z - eps_s)^-1, eps_s,00 = U I
  {
    c64 m[N2], ed[NB];
#pragma unroll
    for (int b = 0; b < NB; ++b) ed[b] = h == 0 ? make_double2(b == a ? U : 0.0, 0.0) : eh[b];
    build_row(m, ed, zd);
    invert_to_Gt(m, false);
#pragma unroll
    for (int b = 0; b < NB; ++b)
      if (live) mine[a * NB + b] = my_init[b];               // Xb = V1, Yb = V1^+ again
  }
  __syncthreads();

  // ---- Newton polish of X = g_surf,00 (header).  Gt holds a full inverse whose 00 block is X.
  const int n_pass = attempt ? 2 * kNewtonMax : kNewtonMax;     // CTA-uniform
  for (int pass = 0; pass < n_pass; ++pass) {
    c64 gold[NB];                  // row a of X (half 0)
    {
      c64 m[N2], ed[NB];
      if (h == 0) {
        row_from<NB>(gold, Gt + a * N2);
#pragma unroll
        for (int b = 0; b < NB; ++b) ed[b] = make_double2(b == a ? U : 0.0, 0.0);
      } else {
        c64 ar[NB], w1[NB];
        row_from<NB>(ar, Xb + a * NB);                       // V1 row a
        gemm_row_ld<NB, N2>(w1, ar, Gt);                     // V1 X
        gemm_row<NB>(ed, w1, Yb);                            // V1 X V1^+
#pragma unroll
        for (int b = 0; b < NB; ++b)
          if (b == a) ed[b].x += U;
      }
      build_row(m, ed, z);
      invert_to_Gt(m, false);
    }
    __syncthreads();
    c64 dlt[NB];                   // half 0: residual row, then the Newton correction
    c64 pqrow[NB];                 // half 0: row a of P;  half 1: row a of Q
    if (h == 0) {
      c64 ar[NB];
#pragma unroll
      for (int b = 0; b < NB; ++b) {
        const c64 gn = Gt[a * N2 + b];
        dlt[b] = make_double2(gn.x - gold[b].x, gn.y - gold[b].y);
        ar[b] = Gt[a * N2 + NB + b];                         // G01 row a
      }
      gemm_row<NB>(pqrow, ar, Xb);                           // P = G01 V1
      if (live) {
        sm.mag[t * N2 + a] = row_absmax<NB>(dlt);
        sm.mag[t * N2 + NB + a] = row_absmax<NB>(gold);
      }
    } else {
      c64 ar[NB];
      row_from<NB>(ar, Yb + a * NB);                         // V1^+ row a
      gemm_row_ld<NB, N2>(pqrow, ar, Gt + NB * N2);          // Q = V1^+ G10
#pragma unroll
      for (int b = 0; b < NB; ++b) dlt[b] = make_double2(0.0, 0.0);
    }
    __syncthreads();                                         // reads of Gt done; mag visible
    double tres = 0.0, tg = 0.0;
#pragma unroll
    for (int i = 0; i < NB; ++i) {
      tres = fmax(tres, sm.mag[t * N2 + i]);
      tg = fmax(tg, sm.mag[t * N2 + NB + i]);
    }
    final_res = tres;
    final_scale = tg;
    const bool good = (tres <= 2e-14 * tg) && (tg < CUDART_INF) && !div_now;
    if (__syncthreads_and(good || !live)) break;            // Gt still holds G(X): X = its 00 block
    // stage P and Q inside Gt (the inverse is dead from here)
    row_to<NB>((h == 0 ? Pb : Qb) + a * NB, pqrow, live);
    __syncthreads();
    bool pdone = false;
    if constexpr (NB == 17) {
      // the doubling sum on the tensor cores (cgemm17.cuh): P, Q, T = D Q and D are the four n x n blocks of Gt
      c64* Db = Gt + 3 * MATN;
      row_to<NB>(Db + a * NB, dlt, live0);
      __syncthreads();
      const int warp = tid >> 5, lane = tid & 31;
      for (int it = 0; it < kDoublingMax; ++it) {
#pragma unroll 1
        for (int tt = warp; tt < G2::TPC; tt += G2::NWARPS) {          // T = D Q
          c64* g = sm.mat + (size_t)tt * G2::MAT;
          cgemm17_warp(g + 3 * MATN, NB, g + MATN, NB, g + 2 * MATN, NB, lane);
        }
        __syncthreads();
#pragma unroll 1
        for (int item = warp; item < 2 * G2::TPC; item += G2::NWARPS) {
          c64* g = sm.mat + (size_t)(item >> 1) * G2::MAT;
          if (item & 1) {
            cgemm17_warp(g + MATN, NB, g + MATN, NB, g + MATN, NB, lane);        // Q <- Q^2
          } else {
            cgemm17_warp(g, NB, g + 2 * MATN, NB, g + 2 * MATN, NB, lane);      // T <- P D Q
            cgemm17_warp(g, NB, g, NB, g, NB, lane);                            // P <- P^2
          }
        }
        __syncthreads();
        double rowmax = 0.0;
        if (h == 0) {
          if (!pdone) {
            c64 w[NB];
            row_from<NB>(w, Tb + a * NB);
#pragma unroll
            for (int b = 0; b < NB; ++b) { dlt[b].x += w[b].x; dlt[b].y += w[b].y; }
            row_to<NB>(Db + a * NB, dlt, live);
          }
        } else {
          c64 w[NB];
          row_from<NB>(w, Pb + a * NB);
          rowmax = row_absmax<NB>(w);
          row_from<NB>(w, Qb + a * NB);
          rowmax = fmax(rowmax, row_absmax<NB>(w));
          if (pdone) rowmax = 0.0;
        }
        if (live) sm.mag[t * N2 + r] = rowmax;
        __syncthreads();
        double tmax = 0.0;
#pragma unroll
        for (int i = 0; i < N2; ++i) tmax = fmax(tmax, sm.mag[t * N2 + i]);
        const bool was_done = pdone;
        if (tmax < 1e-4) pdone = true;                         // |P_j| |Q_j| < 1e-8: series summed
        if (!(tmax < 1e6)) { pdone = true; div_now = true; }   // growing powers: spectral radius > 1
        if (pdone && !was_done && h == 1 && live) {            // a finished task adds nothing any more
#pragma unroll
          for (int b = 0; b < NB; ++b) Pb[a * NB + b] = Qb[a * NB + b] = make_double2(0.0, 0.0);
        }
        if (__syncthreads_and(pdone || !live)) break;
      }
    } else {
        for (int it = 0; it < kDoublingMax; ++it) {
        c64 w[NB];
        if (h == 0) {
          gemm_row<NB>(w, dlt, Qb);                            // D Q
          row_to<NB>(Tb + a * NB, w, live);
        } else {
          gemm_row<NB>(w, pqrow, Qb);                          // Q^2
  #pragma unroll
          for (int b = 0; b < NB; ++b) pqrow[b] = pdone ? make_double2(0.0, 0.0) : w[b];
        }
        __syncthreads();
        double rowmax = 0.0;
        c64 p2[NB];
        if (h == 0) {
          gemm_row<NB>(w, pqrow, Tb);                          // P D Q
          if (!pdone) {
  #pragma unroll
            for (int b = 0; b < NB; ++b) { dlt[b].x += w[b].x; dlt[b].y += w[b].y; }
          }
        } else {
          c64 ar[NB];
          row_from<NB>(ar, Pb + a * NB);
          gemm_row<NB>(p2, ar, Pb);                            // P^2 (computed by half 1 to balance the work)
          if (pdone) {
  #pragma unroll
            for (int b = 0; b < NB; ++b) p2[b] = make_double2(0.0, 0.0);
          }
          rowmax = fmax(row_absmax<NB>(p2), row_absmax<NB>(pqrow));
        }
        if (live) sm.mag[t * N2 + r] = rowmax;
        __syncthreads();                                       // reads of Pb, Qb, Tb done
        if (h == 1) {
          row_to<NB>(Pb + a * NB, p2, live);
          row_to<NB>(Qb + a * NB, pqrow, live);
        }
        double tmax = 0.0;
  #pragma unroll
        for (int i = 0; i < N2; ++i) tmax = fmax(tmax, sm.mag[t * N2 + i]);
        if (tmax < 1e-4) pdone = true;                         // |P_j| |Q_j| < 1e-8: series summed
        if (!(tmax < 1e6)) { pdone = true; div_now = true; }   // growing powers: spectral radius > 1
        const bool all_done = __syncthreads_and(pdone || !live);
        if (h == 0) row_from<NB>(pqrow, Pb + a * NB);
        if (all_done) break;
      }
    }
    // X <- X + D, written where the next pass (or the code below) expects the 00 block
    __syncthreads();
    if (live0) {
#pragma unroll
      for (int b = 0; b < NB; ++b)
        Gt[a * N2 + b] = div_now ? gold[b] : make_double2(gold[b].x + dlt[b].x, gold[b].y + dlt[b].y);
    }
    __syncthreads();
  }
  if (attempt == 1 || !__syncthreads_or(div_now && live)) break;
  diverged = div_now;
  }
  if (active && r == 0 && !(final_res <= 1e-9 * final_scale)) atomicExch(p.noconv_flag, 1);

  // ---- Sigma = L g00 R  (rows owned by half 0)
  c64 srow[NB];
  {
    c64 grow[NB], t1[NB];
    row_from<NB>(grow, Gt + a * N2);
    __syncthreads();                                         // everyone has its row of g00
    if (live0) {
#pragma unroll
      for (int b = 0; b < NB; ++b) Yb[a * NB + b] = gR[a * NB + b];
    }
    __syncthreads();
    gemm_row<NB>(t1, grow, Yb);                              // g00 R
    row_to<NB>(Xb + a * NB, t1, live0);
    __syncthreads();
    row_from<NB>(grow, gL + a * NB);
    gemm_row<NB>(srow, grow, Xb);                            // L g00 R
  }
  c64* out = p.table + (size_t)task * 2 * MATN;
#pragma unroll
  for (int b = 0; b < NB; ++b) {
    if (active && h == 0) out[a * NB + b] = srow[b];
    if (live0) Yb[a * NB + b] = srow[b];
  }
  __syncthreads();

  // ---- Gamma = i (Sigma - Sigma^dagger) and its pivoted Cholesky factor, Gamma = F F^dagger
  c64 S[NB], F[NB];
#pragma unroll
  for (int b = 0; b < NB; ++b) {
    const c64 sba = Yb[b * NB + a];
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
    if (live0) sm.mag[t * N2 + a] = usedc ? -1.0 : diag;
    __syncthreads();
    int piv = 0;
    double dmax = sm.mag[t * N2];
#pragma unroll
    for (int i = 1; i < NB; ++i) {
      const double v = sm.mag[t * N2 + i];
      if (v > dmax) { dmax = v; piv = i; }
    }
    c64* prow = sm.prow + ((size_t)(j & 1) * G2::TPC + t) * N2;
    if (a == piv && live0) {
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
    if (active && h == 0) out[MATN + a * NB + b] = F[b];
}

template <int NB>
static size_t sr_smem_t() {
  return Smem<2 * NB>::bytes(1) + sizeof(c64) * (size_t)Geo<2 * NB>::TPC * 2 * NB * NB +
         sizeof(int) * 32 * Geo<2 * NB>::TPC + 32;
}

template <int NB>
static cudaError_t launch_sr_t(const SrLaunch& p, cudaStream_t s) {
  using G2 = Geo<2 * NB>;
  const size_t smem = sr_smem_t<NB>();
  cudaError_t e = cudaFuncSetAttribute(sancho_rubio_kernel<NB>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                       (int)smem);
  if (e != cudaSuccess) return e;
  const long long n_task = p.task_end - p.task_begin;
  if (n_task <= 0) return cudaSuccess;
  const int blocks = (int)((n_task + G2::TPC - 1) / G2::TPC);
  sancho_rubio_kernel<NB><<<blocks, G2::THREADS, smem, s>>>(p);
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
