// Device primitives of the real-axis forward sweep for n = 17 (block_fwd17.cu; DESIGN.md "Block
// kernels"): a 17 x 17 complex inversion held by EIGHT lanes of one warp, four tasks per warp.
//
// Why: with the two-rows-per-thread geometry of block_ops2.cuh a task is 9 threads, tasks straddle
// warps, and every elimination step costs a divergent pivot-row publish (18 STS.128 by 3-4 lanes: 3.5
// shared-memory wavefronts each), a CTA barrier and 17 LDS.128 -- measured on config 3 the publish, the
// barrier and the wait after it are as many stall samples as the elimination itself.  17 = 16 + 1:
// the leading 16 x 16 block A fits 8 lanes x 2 rows exactly, so a task can live inside a warp, the pivot
// row is broadcast with shuffles from its owner's registers (no publish, no barrier, no divergence),
// and the 17th row and column are folded in by a block (Schur) step:
//     M = [[A, b], [c, d]]
//     A' = A - b d^-1 c,   G = A'^-1,   M^-1 = [[G, -G b d^-1], [-d^-1 c G, d^-1 + d^-1 c G b d^-1]],
// i.e. row 16 is the FIRST pivot row.  Its pivot is d when |d|^2 >= theta^2 |row 16|^2, otherwise the
// largest element of the row (the two columns of M are exchanged, and the two rows of M^-1 exchanged
// back).  G is formed by the same Gauss-Jordan scheme as gj_invert2: diagonal candidates accepted by the
// row-norm test, otherwise a column search over the task's unused rows.
//
// Register layout of lane l8 = lane & 7 of a task: R[q][0..16] = row l8 + 8q of M (q = 0, 1; column 16
// is b); S[0], S[1] = M[16][l8], M[16][l8 + 8]; S[2] = d on every lane of the task.
#pragma once
#include "block_ops.cuh"

namespace negf {
namespace blk {

constexpr int kTpc17 = 8;                 // tasks per 64-thread CTA of block_fwd17_kernel (4 per warp)
constexpr unsigned kFullMask = 0xffffffffu;

__device__ __forceinline__ c64 shfl_c(c64 v, int src) {
  return make_double2(__shfl_sync(kFullMask, v.x, src), __shfl_sync(kFullMask, v.y, src));
}
__device__ __forceinline__ c64 shfl_xor_c(c64 v, int m) {
  return make_double2(__shfl_xor_sync(kFullMask, v.x, m), __shfl_xor_sync(kFullMask, v.y, m));
}
__device__ __forceinline__ c64 csel(bool p, c64 a, c64 b) { return p ? a : b; }
__device__ __forceinline__ c64 cadd(c64 a, c64 b) { return make_double2(a.x + b.x, a.y + b.y); }

// sum over the 8 lanes of a task, result on all of them
__device__ __forceinline__ double sum8(double v) {
  v += __shfl_xor_sync(kFullMask, v, 1);
  v += __shfl_xor_sync(kFullMask, v, 2);
  v += __shfl_xor_sync(kFullMask, v, 4);
  return v;
}
__device__ __forceinline__ c64 sum8(c64 v) { return make_double2(sum8(v.x), sum8(v.y)); }

// x[i] on lane l holds a partial of element i (i = 0 .. 7); returns the full sum of element l8 on lane l8
// (recursive halving: 7 exchanged values instead of 24 for a butterfly over all eight).
__device__ __forceinline__ c64 reduce_scatter8(const c64 (&x)[8], int l8) {
  c64 y[4], w[2];
  const bool h4 = l8 & 4, h2 = l8 & 2, h1 = l8 & 1;
#pragma unroll
  for (int i = 0; i < 4; ++i) y[i] = cadd(csel(h4, x[4 + i], x[i]), shfl_xor_c(csel(h4, x[i], x[4 + i]), 4));
#pragma unroll
  for (int i = 0; i < 2; ++i) w[i] = cadd(csel(h2, y[2 + i], y[i]), shfl_xor_c(csel(h2, y[i], y[2 + i]), 2));
  return cadd(csel(h1, w[1], w[0]), shfl_xor_c(csel(h1, w[0], w[1]), 1));
}

// One elimination step of the 16 x 16 Gauss-Jordan inversion: pivot row p of the lane's task, held in
// row slot pq of lane pown.  SLOT = 0 / 1: slot known at compile time (all tasks of the warp took their
// diagonal candidate); SLOT = -1: per-task slot.  Registers rotate by one column per step as in
// gj_phase2 (block_ops2.cuh): the pivot column is register column 0, the new inverse column enters at 15.
template <int SLOT>
__device__ __forceinline__ void gj16_eliminate(c64 (&R)[2][17], c64 pv, int p, int pq, int pown, int l8,
                                               bool (&used)[2], c64 (&dinv)[2]) {
  const c64 inv = crcp(pv);
  const bool piv0 = (l8 == p), piv1 = (l8 + 8 == p);
  c64 f0 = cmul(R[0][0], inv), f1 = cmul(R[1][0], inv);
  if (piv0) { f0 = make_double2(0.0, 0.0); dinv[0] = inv; used[0] = true; }
  if (piv1) { f1 = make_double2(0.0, 0.0); dinv[1] = inv; used[1] = true; }
#pragma unroll
  for (int j = 0; j < 15; ++j) {
    const c64 src = SLOT == 0 ? R[0][j + 1] : SLOT == 1 ? R[1][j + 1] : csel(pq != 0, R[1][j + 1], R[0][j + 1]);
    const c64 pj = shfl_c(src, pown);
    c64 t0 = R[0][j + 1], t1 = R[1][j + 1];
    cfms(t0, f0, pj);
    cfms(t1, f1, pj);
    R[0][j] = t0;
    R[1][j] = t1;
  }
  R[0][15] = make_double2((piv0 ? 1.0 : 0.0) - f0.x, -f0.y);
  R[1][15] = make_double2((piv1 ? 1.0 : 0.0) - f1.x, -f1.y);
}

template <int Q>
__device__ __forceinline__ void gj16_phase(c64 (&R)[2][17], const double (&thr)[2], bool (&used)[2],
                                           c64 (&dinv)[2], int l8, int base, unsigned long long& perm,
                                           bool& any_search) {
#pragma unroll 1
  for (int kk = 0; kk < 8; ++kk) {
    const int k = 8 * Q + kk;
    const int own = base + kk;
    c64 pv = shfl_c(R[Q][0], own);                    // the diagonal candidate of every task
    const double m = cabs2(pv);
    const bool mine = (l8 == kk);
    const bool ok = !used[Q] && (m >= thr[Q]) && (m > 0.0);
    const unsigned bal = __ballot_sync(kFullMask, ok || !mine);
    if (bal == kFullMask) {
      gj16_eliminate<Q>(R, pv, k, Q, own, l8, used, dinv);
      perm |= (unsigned long long)k << (4 * k);
    } else {
      // rare: the tasks whose candidate was rejected search column k over their unused rows
      any_search = true;
      const bool rejected = !((bal >> own) & 1u);
      const double c0 = used[0] ? -1.0 : cabs2(R[0][0]);
      const double c1 = used[1] ? -1.0 : cabs2(R[1][0]);
      double best = c0;
      int bi = l8;
      if (c1 > best) { best = c1; bi = l8 + 8; }
#pragma unroll
      for (int mk = 1; mk < 8; mk <<= 1) {
        const double ob = __shfl_xor_sync(kFullMask, best, mk);
        const int oi = __shfl_xor_sync(kFullMask, bi, mk);
        if (ob > best || (ob == best && oi < bi)) { best = ob; bi = oi; }
      }
      const int p = rejected ? bi : k;
      const int pq = p >> 3, pown = base + (p & 7);
      pv = shfl_c(csel(pq != 0, R[1][0], R[0][0]), pown);
      gj16_eliminate<-1>(R, pv, p, pq, pown, l8, used, dinv);
      perm |= (unsigned long long)p << (4 * k);
    }
  }
}

// In-place inversion of the task's 17 x 17 matrix (layout in the header).  `scratch` is the task's own
// shared-memory matrix (17 rows, leading dimension ld >= 17), used only on the rare paths: a column search
// reordered the pivots, or row 16 needed a pivot other than d.  Warp-synchronous: all 32 lanes call it.
__device__ __forceinline__ void invert17_w8(c64 (&R)[2][17], c64 (&S)[3], double theta2, int l8, int base,
                                            c64* scratch, int ld) {
  double thr[2];
#pragma unroll
  for (int q = 0; q < 2; ++q) {
    double m = 0.0;
#pragma unroll
    for (int j = 0; j < 17; ++j) m = fma(R[q][j].x, R[q][j].x, fma(R[q][j].y, R[q][j].y, m));
    thr[q] = m * theta2;
  }
  // ---- first pivot: row 16.  d = M[16][16] if it passes the row-norm test, else the largest element of
  // the row (columns js and 16 of M are exchanged, rows js and 16 of the inverse are exchanged back below)
  const double c0 = cabs2(S[0]), c1 = cabs2(S[1]), md = cabs2(S[2]);
  const double n16 = sum8(c0 + c1) + md;
  const bool first = (md >= theta2 * n16) && (md > 0.0);
  const bool any_swap = !__all_sync(kFullMask, first);
  int js = 16;
  if (any_swap) {
    double best = c0;
    int bj = l8;
    if (c1 > best) { best = c1; bj = l8 + 8; }
#pragma unroll
    for (int mk = 1; mk < 8; mk <<= 1) {
      const double ob = __shfl_xor_sync(kFullMask, best, mk);
      const int oj = __shfl_xor_sync(kFullMask, bj, mk);
      if (ob > best || (ob == best && oj < bj)) { best = ob; bj = oj; }
    }
    const c64 newd = shfl_c(csel(bj >= 8, S[1], S[0]), base + (bj & 7));
    if (!first) {
      js = bj;
      // columns js <-> 16 of the lane's rows, through its own rows of the scratch matrix (a register
      // array indexed by js would be demoted to local memory)
#pragma unroll
      for (int q = 0; q < 2; ++q) {
        c64* mine = scratch + (l8 + 8 * q) * ld;
        mine[16] = R[q][16];
#pragma unroll
        for (int j = 0; j < 16; ++j) mine[j] = R[q][j];
        R[q][16] = mine[js];
        mine[js] = mine[16];
#pragma unroll
        for (int j = 0; j < 16; ++j) R[q][j] = mine[j];
      }
      if (l8 == (js & 7)) {
        if (js >= 8) S[1] = S[2]; else S[0] = S[2];
      }
      S[2] = newd;
    }
    __syncwarp();
  }
  const c64 dinv16 = crcp(S[2]);
  {
    const c64 g0 = cmul(R[0][16], dinv16), g1 = cmul(R[1][16], dinv16);   // A' = A - b d^-1 c
#pragma unroll
    for (int j = 0; j < 16; ++j) {
      const c64 cj = shfl_c(S[j >> 3], base + (j & 7));
      cfms(R[0][j], g0, cj);
      cfms(R[1][j], g1, cj);
    }
  }
  // ---- G = A'^-1
  bool used[2] = {false, false};
  c64 dinv[2] = {make_double2(1.0, 0.0), make_double2(1.0, 0.0)};
  unsigned long long perm = 0;
  bool any_search = false;
  gj16_phase<0>(R, thr, used, dinv, l8, base, perm, any_search);
  gj16_phase<1>(R, thr, used, dinv, l8, base, perm, any_search);
#pragma unroll
  for (int q = 0; q < 2; ++q)
#pragma unroll
    for (int j = 0; j < 16; ++j) R[q][j] = cmul(R[q][j], dinv[q]);
  if (any_search) {
    // lane holds, in R[q], row perm^-1(l8 + 8q) of G with register column j being column perm[j]
#pragma unroll
    for (int q = 0; q < 2; ++q) {
      const int rid = l8 + 8 * q;
      int row = 0;
#pragma unroll
      for (int k = 0; k < 16; ++k)
        if ((int)((perm >> (4 * k)) & 15u) == rid) row = k;
#pragma unroll
      for (int j = 0; j < 16; ++j) scratch[row * ld + (int)((perm >> (4 * j)) & 15u)] = R[q][j];
    }
    __syncwarp();
#pragma unroll
    for (int q = 0; q < 2; ++q)
#pragma unroll
      for (int j = 0; j < 16; ++j) R[q][j] = scratch[(l8 + 8 * q) * ld + j];
    __syncwarp();
  }
  // ---- border:  u = G b,  v = c G,  t = c u;  column -u d^-1, row -d^-1 v, corner d^-1 + d^-1 t d^-1
  c64 u0 = make_double2(0.0, 0.0), u1 = make_double2(0.0, 0.0);
#pragma unroll
  for (int j = 0; j < 16; ++j) {
    const c64 bj = shfl_c(R[j >> 3][16], base + (j & 7));
    cfma(u0, R[0][j], bj);
    cfma(u1, R[1][j], bj);
  }
  c64 v[2];
#pragma unroll
  for (int h = 0; h < 2; ++h) {
    c64 vp[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) {
      vp[i] = cmul(S[0], R[0][8 * h + i]);
      cfma(vp[i], S[1], R[1][8 * h + i]);
    }
    v[h] = reduce_scatter8(vp, l8);
  }
  c64 tp = cmul(S[0], u0);
  cfma(tp, S[1], u1);
  const c64 t = sum8(tp);
  const c64 nd = make_double2(-dinv16.x, -dinv16.y);
  R[0][16] = cmul(u0, nd);
  R[1][16] = cmul(u1, nd);
  S[0] = cmul(nd, v[0]);
  S[1] = cmul(nd, v[1]);
  c64 corner = cmul(cmul(dinv16, t), dinv16);
  S[2] = make_double2(corner.x + dinv16.x, corner.y + dinv16.y);
  if (any_swap) {
    // inverse of (M with columns js, 16 exchanged) -> exchange rows js and 16, through the scratch matrix
    // (rare path: registers and shuffles are kept for the common one)
    const bool own0 = !first && l8 == js, own1 = !first && l8 + 8 == js;
    c64* rowj = scratch;             // old row js
    c64* row16 = scratch + ld;       // old row 16
    if (own0 || own1) {
#pragma unroll
      for (int j = 0; j < 17; ++j) rowj[j] = own0 ? R[0][j] : R[1][j];
    }
    row16[l8] = S[0];
    row16[l8 + 8] = S[1];
    if (l8 == 0) row16[16] = S[2];
    __syncwarp();
    if (own0) {
#pragma unroll
      for (int j = 0; j < 17; ++j) R[0][j] = row16[j];
    }
    if (own1) {
#pragma unroll
      for (int j = 0; j < 17; ++j) R[1][j] = row16[j];
    }
    if (!first) {
      S[0] = rowj[l8];
      S[1] = rowj[l8 + 8];
      S[2] = rowj[16];
    }
    __syncwarp();
  }
}

}  // namespace blk
}  // namespace negf
