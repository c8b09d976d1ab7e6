// 34 x 34 complex inversion by ONE WARP, for the Sancho-Rubio decimation of n = 17 (sancho_rubio.cu): the
// principal layer of the lead is two rings, so every decimation pass and every Newton pass inverts a
// 34 x 34 matrix.  With one row per thread and 34 threads per task (block_ops.cuh gj_invert<34>) an
// inversion is 34 CTA barriers and a pivot-row publish through shared memory per step; tasks straddle warps.
// Here, as in block_ops17.cuh: 34 = 32 + 2, lane l holds row l of the leading 32 x 32 block A and its two
// elements of the border columns B; the pivot row reaches the other lanes by shuffle; rows 32, 33 are the
// FIRST pivot rows (block step with the 2 x 2 corner D):
//     M = [[A, B], [C, D]],   A' = A - B D^-1 C,   G = A'^-1,
//     M^-1 = [[G, -G B D^-1], [-D^-1 C G, D^-1 + D^-1 C G B D^-1]],
// with -B D^-1 carried through the Gauss-Jordan elimination as two right-hand-side columns.  Pivoting as in
// gj_invert: the diagonal candidate is accepted when |a_kk|^2 >= theta^2 |row k|^2, otherwise the whole
// column is searched over the unused rows (the permutation is undone through shared memory); when the corner
// pivots fail the same test (rare) the warp falls back to plain partial pivoting in shared memory.
// The matrix lives in shared memory (34 x 34, row-major) before and after; one task per warp, so every
// decision is warp-uniform.
#pragma once
#include "block_ops.cuh"

namespace negf {
namespace blk {

constexpr int kLd34 = 34;
constexpr unsigned kMask34 = 0xffffffffu;

__device__ __forceinline__ c64 shfl34(c64 v, int src) {
  return make_double2(__shfl_sync(kMask34, v.x, src), __shfl_sync(kMask34, v.y, src));
}
__device__ __forceinline__ double warp_sum34(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(kMask34, v, o);
  return v;
}
__device__ __forceinline__ c64 warp_sum34(c64 v) { return make_double2(warp_sum34(v.x), warp_sum34(v.y)); }
// arg-max over the warp (ties: the smaller index), result on all lanes
__device__ __forceinline__ int argmax34(double best, int bi) {
#pragma unroll
  for (int mk = 1; mk < 32; mk <<= 1) {
    const double ob = __shfl_xor_sync(kMask34, best, mk);
    const int oi = __shfl_xor_sync(kMask34, bi, mk);
    if (ob > best || (ob == best && oi < bi)) { best = ob; bi = oi; }
  }
  return bi;
}

// Plain Gauss-Jordan inversion with partial pivoting of the 34 x 34 matrix m in shared memory, in place, by
// one warp (rare path; not inlined: it must not cost the fast path registers).
static __device__ __noinline__ void invert34_slow(c64* m, int lane) {
  constexpr int N = 34, LD = kLd34;
  int piv[N];
  for (int k = 0; k < N; ++k) {
    double best = -1.0;
    int bi = k;
    for (int i = k + lane; i < N; i += 32) {
      const double v = cabs2(m[i * LD + k]);
      if (v > best) { best = v; bi = i; }
    }
    const int p = argmax34(best, bi);
    piv[k] = p;
    __syncwarp();
    if (p != k) {
      for (int j = lane; j < N; j += 32) {
        const c64 a = m[k * LD + j];
        m[k * LD + j] = m[p * LD + j];
        m[p * LD + j] = a;
      }
    }
    __syncwarp();
    const c64 inv = crcp(m[k * LD + k]);
    __syncwarp();
    for (int j = lane; j < N; j += 32) m[k * LD + j] = j == k ? inv : cmul(m[k * LD + j], inv);
    __syncwarp();
    for (int i = lane; i < N; i += 32) {
      if (i == k) continue;
      const c64 f = m[i * LD + k];
      for (int j = 0; j < N; ++j) {
        const c64 pk = m[k * LD + j];
        c64 t = j == k ? make_double2(0.0, 0.0) : m[i * LD + j];
        cfms(t, f, pk);
        m[i * LD + j] = t;
      }
    }
    __syncwarp();
  }
  for (int k = N - 1; k >= 0; --k) {           // the row exchanges become column exchanges of the inverse
    const int p = piv[k];
    if (p != k) {
      for (int i = lane; i < N; i += 32) {
        const c64 a = m[i * LD + k];
        m[i * LD + k] = m[i * LD + p];
        m[i * LD + p] = a;
      }
    }
    __syncwarp();
  }
}

// In-place inversion of the 34 x 34 matrix m (shared memory, row-major, leading dimension 34) by one warp.
// perm: 32 ints of shared memory owned by the warp.  All 32 lanes call it; the caller synchronises before
// (m complete) and after (other threads read m).
static __device__ __noinline__ void invert34_w32(c64* m, int* perm, double theta2, int lane) {
  constexpr int LD = kLd34;
  c64 R[32], Rb[2];
#pragma unroll
  for (int j = 0; j < 32; ++j) R[j] = m[lane * LD + j];
  Rb[0] = m[lane * LD + 32];
  Rb[1] = m[lane * LD + 33];
  double thr = fma(Rb[0].x, Rb[0].x, fma(Rb[0].y, Rb[0].y, fma(Rb[1].x, Rb[1].x, Rb[1].y * Rb[1].y)));
#pragma unroll
  for (int j = 0; j < 32; ++j) thr = fma(R[j].x, R[j].x, fma(R[j].y, R[j].y, thr));
  thr *= theta2;                           // row scale: squared 2-norm of the row as handed in
  // ---- first pivots: rows 32 and 33 (2 x 2 corner D), accepted by the same row-norm test
  {
    const c64 C0 = m[32 * LD + lane], C1 = m[33 * LD + lane];
    const c64 D00 = m[32 * LD + 32], D01 = m[32 * LD + 33], D10 = m[33 * LD + 32], D11 = m[33 * LD + 33];
    const double n32 = warp_sum34(cabs2(C0)) + cabs2(D00) + cabs2(D01);
    const double n33 = warp_sum34(cabs2(C1)) + cabs2(D10) + cabs2(D11);
    const double m00 = cabs2(D00);
    bool ok = (m00 >= theta2 * n32) && (m00 > 0.0);
    const c64 f = cmul(D10, crcp(D00));
    c64 s11 = D11;                         // second pivot, after the elimination with row 32
    cfms(s11, f, D01);
    const double m11 = cabs2(s11);
    ok = ok && (m11 >= theta2 * n33) && (m11 > 0.0);
    if (!ok) {
      __syncwarp();
      invert34_slow(m, lane);
      return;
    }
    const c64 idet = crcp(cmul(D00, s11));
    const c64 E00 = cmul(D11, idet), E11 = cmul(D00, idet);
    const c64 nidet = make_double2(-idet.x, -idet.y);
    const c64 E01 = cmul(D01, nidet), E10 = cmul(D10, nidet);
    c64 g0 = cmul(Rb[0], E00), g1 = cmul(Rb[0], E01);          // B D^-1 (this lane's row)
    cfma(g0, Rb[1], E10);
    cfma(g1, Rb[1], E11);
#pragma unroll
    for (int j = 0; j < 32; ++j) {                             // A' = A - B D^-1 C
      cfms(R[j], g0, shfl34(C0, j));
      cfms(R[j], g1, shfl34(C1, j));
    }
    Rb[0] = make_double2(-g0.x, -g0.y);                        // -B D^-1 rides along as two right-hand sides
    Rb[1] = make_double2(-g1.x, -g1.y);
    __syncwarp();                                              // every lane has read D
    if (lane == 0) {                                           // D^-1 waits in the corner
      m[32 * LD + 32] = E00;
      m[32 * LD + 33] = E01;
      m[33 * LD + 32] = E10;
      m[33 * LD + 33] = E11;
    }
  }
  // ---- G = A'^-1 and G (-B D^-1): Gauss-Jordan, pivot row by shuffle, registers rotated by one column per
  // step (the pivot column is register column 0, the new inverse column enters at column 31)
  perm[lane] = lane;
  bool used = false, any_search = false;
  c64 dinv = make_double2(1.0, 0.0);
#pragma unroll 2
  for (int k = 0; k < 32; ++k) {
    const double mm = cabs2(R[0]);
    const int cand_ok = (!used && (mm >= thr) && (mm > 0.0)) ? 1 : 0;
    int p = k;
    if (!__shfl_sync(kMask34, cand_ok, k)) {                   // rare: search column k over the unused rows
      any_search = true;
      p = argmax34(used ? -1.0 : mm, lane);
      __syncwarp();
      if (lane == 0) perm[k] = p;
    }
    const c64 inv = crcp(shfl34(R[0], p));
    const bool piv = (lane == p);
    c64 f = cmul(R[0], inv);
    if (piv) { f = make_double2(0.0, 0.0); dinv = inv; used = true; }
#pragma unroll
    for (int j = 0; j < 31; ++j) {
      const c64 pj = shfl34(R[j + 1], p);
      c64 t0 = R[j + 1];
      cfms(t0, f, pj);
      R[j] = t0;
    }
    R[31] = make_double2((piv ? 1.0 : 0.0) - f.x, -f.y);
    cfms(Rb[0], f, shfl34(Rb[0], p));
    cfms(Rb[1], f, shfl34(Rb[1], p));
  }
#pragma unroll
  for (int j = 0; j < 32; ++j) R[j] = cmul(R[j], dinv);
  Rb[0] = cmul(Rb[0], dinv);
  Rb[1] = cmul(Rb[1], dinv);
  // ---- G and G (-B D^-1) to shared memory (rows 0..31); the lane holds row `row` of them
  int row = lane;
  if (!any_search) {
#pragma unroll
    for (int j = 0; j < 32; ++j) m[lane * LD + j] = R[j];
  } else {
    __syncwarp();
    for (int k = 0; k < 32; ++k)
      if (perm[k] == lane) row = k;
#pragma unroll
    for (int j = 0; j < 32; ++j) m[row * LD + perm[j]] = R[j];
  }
  m[row * LD + 32] = Rb[0];
  m[row * LD + 33] = Rb[1];
  // ---- border: T = C (G B') by warp sums, V = C G by a rolled loop over the rows of G
  const c64 c0r = m[32 * LD + row], c1r = m[33 * LD + row];
  const c64 T00 = warp_sum34(cmul(c0r, Rb[0])), T01 = warp_sum34(cmul(c0r, Rb[1]));
  const c64 T10 = warp_sum34(cmul(c1r, Rb[0])), T11 = warp_sum34(cmul(c1r, Rb[1]));
  __syncwarp();
  c64 V0 = make_double2(0.0, 0.0), V1 = V0;
#pragma unroll 4
  for (int r = 0; r < 32; ++r) {
    const c64 g = m[r * LD + lane];
    cfma(V0, m[32 * LD + r], g);
    cfma(V1, m[33 * LD + r], g);
  }
  const c64 E00 = m[32 * LD + 32], E01 = m[32 * LD + 33], E10 = m[33 * LD + 32], E11 = m[33 * LD + 33];
  __syncwarp();                                                // every lane has read C and D^-1
  c64 W0 = cmul(E00, V0), W1 = cmul(E10, V0);                  // rows 32, 33 of the inverse: -D^-1 C G
  cfma(W0, E01, V1);
  cfma(W1, E11, V1);
  m[32 * LD + lane] = make_double2(-W0.x, -W0.y);
  m[33 * LD + lane] = make_double2(-W1.x, -W1.y);
  if (lane == 0) {                                             // corner: D^-1 - D^-1 T  (T = -C G B D^-1)
    c64 K00 = E00, K01 = E01, K10 = E10, K11 = E11;
    cfms(K00, E00, T00); cfms(K00, E01, T10);
    cfms(K01, E00, T01); cfms(K01, E01, T11);
    cfms(K10, E10, T00); cfms(K10, E11, T10);
    cfms(K11, E10, T01); cfms(K11, E11, T11);
    m[32 * LD + 32] = K00;
    m[32 * LD + 33] = K01;
    m[33 * LD + 32] = K10;
    m[33 * LD + 33] = K11;
  }
  __syncwarp();
}

}  // namespace blk
}  // namespace negf
