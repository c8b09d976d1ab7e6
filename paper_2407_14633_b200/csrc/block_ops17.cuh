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
//     M = [[A, b], [c, d]],   A' = A - b d^-1 c,   G = A'^-1,
//     M^-1 = [[G, -G b d^-1], [-d^-1 c G, d^-1 + d^-1 c G b d^-1]],
// i.e. row 16 is the FIRST pivot row, with pivot d.  When |d|^2 < theta^2 |row 16|^2 for a task (rare) its warp
// takes a slow path instead: plain partial pivoting in shared memory (invert17_slow).  G is formed by the Gauss-Jordan scheme of gj_invert2 -- diagonal candidates accepted by the
// row-norm test, otherwise a column search over the task's unused rows -- with -b d^-1 carried along as a
// right-hand side, which leaves column 16 of the inverse in place.  Row 16 of the inverse, -d^-1 c G, is
// formed from the shared-memory copy of G by a rolled loop (invert17_border): code size matters here, the
// instruction cache behind a scheduler holds 32 KB and the sweep's ring body is about that long.
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
__device__ __forceinline__ c64 csel(bool p, c64 a, c64 b) { return p ? a : b; }

// sum over the 8 lanes of a task, result on all of them
__device__ __forceinline__ double sum8(double v) {
  v += __shfl_xor_sync(kFullMask, v, 1);
  v += __shfl_xor_sync(kFullMask, v, 2);
  v += __shfl_xor_sync(kFullMask, v, 4);
  return v;
}
// arg-max over the 8 lanes of a task (ties: the smaller index), result on all of them
__device__ __forceinline__ int argmax8(double best, int bi) {
#pragma unroll
  for (int mk = 1; mk < 8; mk <<= 1) {
    const double ob = __shfl_xor_sync(kFullMask, best, mk);
    const int oi = __shfl_xor_sync(kFullMask, bi, mk);
    if (ob > best || (ob == best && oi < bi)) { best = ob; bi = oi; }
  }
  return bi;
}

// Per-task bookkeeping of the column searches, in shared memory so that the common path carries no registers
// for it: pivot row chosen for column k (identity unless a search happened).
struct Rare17 {
  int perm[16];
  int pad[4];
};

// One elimination step of the 16 x 16 Gauss-Jordan inversion: pivot row p of the lane's task, held in
// row slot pq of lane pown.  SLOT = 0 / 1: slot known at compile time (all tasks of the warp took their
// diagonal candidate); SLOT = -1: per-task slot.  Registers rotate by one column per step as in
// gj_phase2 (block_ops2.cuh): the pivot column is register column 0, the new inverse column enters at 15;
// column 16, the right-hand side, does not rotate.
template <int SLOT>
__device__ __forceinline__ void gj16_eliminate(c64 (&R)[2][17], c64 pv, int p, int pq, int pown, int l8,
                                               bool (&used)[2], c64 (&dinv)[2]) {
  const c64 inv = crcp(pv);
  const bool piv0 = (l8 == p), piv1 = (l8 + 8 == p);
  c64 f0 = cmul(R[0][0], inv), f1 = cmul(R[1][0], inv);
  if (piv0) { f0 = make_double2(0.0, 0.0); dinv[0] = inv; used[0] = true; }
  if (piv1) { f1 = make_double2(0.0, 0.0); dinv[1] = inv; used[1] = true; }
  // the pivot row arrives by shuffle, kDepth elements ahead of their use (issued back to back with their
  // uses, every element would expose the shuffle latency: 25 % of the kernel's stall samples)
  constexpr int kDepth = 3;
  c64 pj[16];
#pragma unroll
  for (int j = 0; j < kDepth; ++j) {
    const c64 src = SLOT == 0 ? R[0][j + 1] : SLOT == 1 ? R[1][j + 1] : csel(pq != 0, R[1][j + 1], R[0][j + 1]);
    pj[j] = shfl_c(src, pown);
  }
#pragma unroll
  for (int j = 0; j < 16; ++j) {
    if (j + kDepth < 16) {
      const int jn = j + kDepth;
      const c64 src = SLOT == 0 ? R[0][jn + 1] : SLOT == 1 ? R[1][jn + 1] : csel(pq != 0, R[1][jn + 1], R[0][jn + 1]);
      pj[jn] = shfl_c(src, pown);
    }
    c64 t0 = R[0][j + 1], t1 = R[1][j + 1];
    cfms(t0, f0, pj[j]);
    cfms(t1, f1, pj[j]);
    if (j < 15) {
      R[0][j] = t0;
      R[1][j] = t1;
    } else {
      R[0][16] = t0;
      R[1][16] = t1;
    }
  }
  R[0][15] = make_double2((piv0 ? 1.0 : 0.0) - f0.x, -f0.y);
  R[1][15] = make_double2((piv1 ? 1.0 : 0.0) - f1.x, -f1.y);
}

template <int Q>
__device__ __forceinline__ void gj16_phase(c64 (&R)[2][17], const double (&thr)[2], bool (&used)[2],
                                           c64 (&dinv)[2], int l8, int base, Rare17* rare, bool& any_search) {
#pragma unroll 1
  for (int kk = 0; kk < 8; ++kk) {
    const int k = 8 * Q + kk;
    const int own = base + kk;
    c64 pv = shfl_c(R[Q][0], own);                    // the diagonal candidate of every task
    const double m = cabs2(pv);
    const bool ok = !used[Q] && (m >= thr[Q]) && (m > 0.0);
    const unsigned bal = __ballot_sync(kFullMask, ok || l8 != kk);
    if (bal == kFullMask) {
      gj16_eliminate<Q>(R, pv, k, Q, own, l8, used, dinv);
    } else {
      // rare: the tasks whose candidate was rejected search column k over their unused rows
      any_search = true;
      const bool rejected = !((bal >> own) & 1u);
      const double c0 = used[0] ? -1.0 : cabs2(R[0][0]);
      const double c1 = used[1] ? -1.0 : cabs2(R[1][0]);
      const int bi = argmax8(c1 > c0 ? c1 : c0, c1 > c0 ? l8 + 8 : l8);
      const int p = rejected ? bi : k;
      __syncwarp();
      if (rejected && l8 == 0) rare->perm[k] = p;
      const int pq = p >> 3, pown = base + (p & 7);
      pv = shfl_c(csel(pq != 0, R[1][0], R[0][0]), pown);
      gj16_eliminate<-1>(R, pv, p, pq, pown, l8, used, dinv);
    }
  }
}

// Whether d = M[16][16] is acceptable as the first pivot: |d|^2 >= theta^2 |row 16|^2 (per task).
__device__ __forceinline__ bool invert17_first_ok(const c64 (&S)[3], double theta2) {
  const double md = cabs2(S[2]);
  const double n16 = sum8(cabs2(S[0]) + cabs2(S[1])) + md;
  return (md >= theta2 * n16) && (md > 0.0);
}

// First part of the inversion of the task's 17 x 17 matrix (layout in the header), d being an acceptable
// first pivot.  On return R[q][0..15] are the lane's rows of G and R[q][16] its elements of -G b d^-1 (column
// 16 of the inverse); c has moved to row 16 of `scratch`; the return value is d^-1.  `scratch` is the task's
// own 17 x 17 shared-memory matrix (row-major, leading dimension 17); rows 0..15 are used only when a column
// search reordered the pivots.  Warp-synchronous: all 32 lanes call it together.
__device__ __forceinline__ c64 invert17_core(c64 (&R)[2][17], c64 (&S)[3], double theta2, int l8, int base,
                                             c64* scratch, Rare17* rare) {
  constexpr int LD = 17;
  double thr[2];
#pragma unroll
  for (int q = 0; q < 2; ++q) {
    double m = 0.0;                      // row scale: squared 2-norm
#pragma unroll
    for (int j = 0; j < 17; ++j) m = fma(R[q][j].x, R[q][j].x, fma(R[q][j].y, R[q][j].y, m));
    thr[q] = m * theta2;
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
    R[0][16] = make_double2(-g0.x, -g0.y);                                 // -b d^-1 rides along as column 16
    R[1][16] = make_double2(-g1.x, -g1.y);
  }
  scratch[16 * LD + l8] = S[0];            // c waits in row 16 of the shared-memory matrix (invert17_border):
  scratch[16 * LD + l8 + 8] = S[1];        // no registers for it during the elimination
  // ---- G = A'^-1 and G (-b d^-1)
  rare->perm[l8] = l8;
  rare->perm[l8 + 8] = l8 + 8;
  bool used[2] = {false, false};
  c64 dinv[2] = {make_double2(1.0, 0.0), make_double2(1.0, 0.0)};
  bool any_search = false;
  gj16_phase<0>(R, thr, used, dinv, l8, base, rare, any_search);
  gj16_phase<1>(R, thr, used, dinv, l8, base, rare, any_search);
#pragma unroll
  for (int q = 0; q < 2; ++q)
#pragma unroll
    for (int j = 0; j < 17; ++j) R[q][j] = cmul(R[q][j], dinv[q]);
  if (any_search) {
    // the lane holds, in R[q], row perm^-1(l8 + 8q) of G, register column j being column perm[j]
    __syncwarp();
#pragma unroll
    for (int q = 0; q < 2; ++q) {
      int row = 0;
      for (int k = 0; k < 16; ++k)
        if (rare->perm[k] == l8 + 8 * q) row = k;
#pragma unroll
      for (int j = 0; j < 16; ++j) scratch[row * LD + rare->perm[j]] = R[q][j];
      scratch[row * LD + 16] = R[q][16];
    }
    __syncwarp();
#pragma unroll
    for (int q = 0; q < 2; ++q)
#pragma unroll
      for (int j = 0; j < 17; ++j) R[q][j] = scratch[(l8 + 8 * q) * LD + j];
    __syncwarp();
  }
  return dinv16;
}

// Second part: row 16 of the inverse and the corner, from the task's shared-memory matrix `m` holding G and
// -G b d^-1 in rows 0..15 (columns 0..15 and 16) and c in row 16 (columns 0..15):
//     S[0], S[1] := elements l8, l8 + 8 of -d^-1 c G;   S[2] := d^-1 + d^-1 c G b d^-1.
// A rolled loop on purpose (header).  The caller places __syncwarp() before and after.
__device__ __forceinline__ void invert17_border(c64 (&S)[3], c64 dinv16, unsigned m, int l8) {
  c64 v0 = make_double2(0.0, 0.0), v1 = v0, t = v0;
  unsigned row = m + 16u * l8, crow = m + 16u * (16 * 17);
#pragma unroll 2
  for (int r = 0; r < 16; ++r) {
    const c64 cr = lds_c64(crow);
    cfma(v0, cr, lds_c64(row));
    cfma(v1, cr, lds_c64(row + 16 * 8));
    cfma(t, cr, lds_c64(row + 16u * (16 - l8)));
    row += 16 * 17;
    crow += 16;
  }
  const c64 nd = make_double2(-dinv16.x, -dinv16.y);
  S[0] = cmul(nd, v0);
  S[1] = cmul(nd, v1);
  const c64 corner = cmul(nd, t);                         // t = -c G b d^-1
  S[2] = make_double2(dinv16.x + corner.x, dinv16.y + corner.y);
}

// Slow path, taken by a whole warp when d is not acceptable as first pivot for one of its tasks (rare): plain
// Gauss-Jordan inversion with partial pivoting of the task's matrix `m` (17 x 17, row-major, leading dimension
// 17) in shared memory, in place, by the task's eight lanes.  Not inlined: it must not cost the fast path
// registers.  Warp-synchronous.
static __device__ __noinline__ void invert17_slow(c64* m, int l8) {
  constexpr int LD = 17;
  int piv[17];
  for (int k = 0; k < 17; ++k) {
    // pivot search in column k over the rows k .. 16
    double best = -1.0;
    int bi = k;
    for (int i = k + l8; i < 17; i += 8) {
      const double v = cabs2(m[i * LD + k]);
      if (v > best) { best = v; bi = i; }
    }
    const int p = argmax8(best, bi);
    piv[k] = p;
    __syncwarp();
    if (p != k) {
      for (int j = l8; j < 17; j += 8) {
        const c64 a = m[k * LD + j];
        m[k * LD + j] = m[p * LD + j];
        m[p * LD + j] = a;
      }
    }
    __syncwarp();
    const c64 inv = crcp(m[k * LD + k]);
    __syncwarp();
    for (int j = l8; j < 17; j += 8) m[k * LD + j] = j == k ? inv : cmul(m[k * LD + j], inv);
    __syncwarp();
    for (int i = l8; i < 17; i += 8) {
      if (i == k) continue;
      const c64 f = m[i * LD + k];
      for (int j = 0; j < 17; ++j) {
        const c64 pk = m[k * LD + j];
        c64 t = j == k ? make_double2(0.0, 0.0) : m[i * LD + j];
        cfms(t, f, pk);
        m[i * LD + j] = t;
      }
    }
    __syncwarp();
  }
  for (int k = 16; k >= 0; --k) {            // the row exchanges become column exchanges of the inverse
    const int p = piv[k];
    if (p != k) {
      for (int i = l8; i < 17; i += 8) {
        const c64 a = m[i * LD + k];
        m[i * LD + k] = m[i * LD + p];
        m[i * LD + p] = a;
      }
    }
    __syncwarp();
  }
}

}  // namespace blk
}  // namespace negf
