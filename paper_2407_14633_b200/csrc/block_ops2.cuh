// Device primitives of the block RGF sweep with TWO matrix rows per thread (DESIGN.md "Block
// kernels").  Why two: every operand of the elimination / product inner loops is a 16-byte complex
// read from shared memory, and the shared-memory return path delivers 128 B/clk/SM, i.e. one warp-wide
// LDS.128 per 4 clk, while the FP64 pipe retires the 4 DFMAs of one complex multiply-add per warp in
// 2 clk.  With one row per thread each operand feeds one multiply-add, so the kernel is bound by
// shared-memory bandwidth at < 50 % of the FP64 peak (measured: 59 % LSU, 28 % FP64); with two rows
// per thread each operand feeds two.
//
// Geometry: thread `a` (0 .. TPT-1, TPT = ceil(n/2)) of a task owns rows a and a + TPT of the task's
// n x n complex matrix in registers (the second row of the last thread is a zero dummy when n is odd);
// TPT consecutive threads form a task, TPC tasks share a CTA and advance in lock step.  Tasks straddle
// warp boundaries, so rows are exchanged through shared memory and CTA barriers.
#pragma once
#include "block_ops.cuh"

namespace negf {
namespace blk {

template <int NB>
struct Geo2 {
  static constexpr int TPT = (NB + 1) / 2;                           // threads per task
  static constexpr int TPC = (63 / TPT) > 32 ? 32 : (63 / TPT);      // tasks per CTA (2 warps at n = 17)
  static constexpr int LIVE = TPC * TPT;
  static constexpr int THREADS = (LIVE + 31) / 32 * 32;
  static constexpr int NWARPS = THREADS / 32;
  static constexpr int MAT = NB * NB;
  static constexpr int PROW = NB + 1;                                // pivot row + reciprocal pivot
  // one ring step of recursion history of one CTA: [slot q][column b][thread] complex; for n = 17 the
  // real-axis CTAs (block_fwd17.cu) store, in the same space, row-major matrices of kHistRec17 elements
  // (n = 17: 8 records of 306, the 8 tasks of a block_fwd17 CTA; the contour CTAs use the first 2176)
  static constexpr long long STEP_ELEMS = NB == 17 ? 8LL * 306 : 2LL * NB * THREADS;
  static_assert(STEP_ELEMS >= 2LL * NB * THREADS, "the contour layout must fit the step");
};

template <int NB>
struct Smem2 {
  c64* mat;      // [TPC][NB*NB]    one exchange matrix per task
  c64* prow;     // [2][TPC][NB+1]  published pivot rows (double buffered by elimination step)
  double* mag;   // [TPC][NB]       pivot-search magnitudes
  double* red;   // [2][NWARPS]     block reduction scratch
  int* pk;       // [2][TPC]        pivot row of the current elimination step
  int* perm;     // [TPC][NB]       pivot row chosen for column k
  int* ok;       // [TPC]           1 if the diagonal candidate was accepted this step

  static constexpr size_t bytes() {
    using G = Geo2<NB>;
    return sizeof(c64) * ((size_t)G::TPC * G::MAT + 2 * G::TPC * G::PROW) +
           sizeof(double) * (G::TPC * NB + 2 * G::NWARPS) + sizeof(int) * (2 * G::TPC + G::TPC * NB + G::TPC) + 64;
  }
  __device__ char* carve(char* base) {
    using G = Geo2<NB>;
    mat = reinterpret_cast<c64*>(base);
    prow = mat + (size_t)G::TPC * G::MAT;
    mag = reinterpret_cast<double*>(prow + 2 * G::TPC * G::PROW);
    red = mag + G::TPC * NB;
    pk = reinterpret_cast<int*>(red + 2 * G::NWARPS);
    perm = pk + 2 * G::TPC;
    ok = perm + G::TPC * NB;
    char* end = reinterpret_cast<char*>(ok + G::TPC);
    return reinterpret_cast<char*>((reinterpret_cast<uintptr_t>(end) + 15) & ~uintptr_t(15));
  }
};

// The elimination steps k = kbeg .. kend-1 of gj_invert2; the diagonal pivot candidate of step k lives
// in row slot Q = k / TPT of thread a = k - Q*TPT (both slots are tested at run time: ONE loop for all
// steps -- compiled as one loop per slot the register allocator kept a single pivot-row load in
// flight and exposed every load's latency).  The loop is NOT unrolled: after every step the thread's
// registers are rotated by one column (the rotation is folded into the destination registers of the
// elimination FMAs, it costs no instruction), so the pivot column is always register column 0 and the
// new inverse column enters at register column NB-1.  After all NB steps the columns are back in
// their original order.  (A fully unrolled elimination is ~140 KB of code per inversion; with two
// warps per scheduler the kernel then stalls on instruction fetch.)
template <int NB>
__device__ __forceinline__ void gj_phase2(c64 (&r)[2][NB], const Smem2<NB>& sm, int t, int a, bool live,
                                          const double (&thr)[2], bool (&used)[2], c64 (&dinv)[2], int kbeg,
                                          int kend, bool& any_search) {
  using G = Geo2<NB>;
  constexpr int TPT = G::TPT;
  const bool valid1 = a + TPT < NB;
#pragma unroll 1
  for (int k = kbeg; k < kend; ++k) {
    const int buf = k & 1;
    c64* prow = sm.prow + ((size_t)buf * G::TPC + t) * G::PROW;
    int bad = 0;
#pragma unroll
    for (int Q = 0; Q < 2; ++Q) {
      if (a + Q * TPT == k) {
        const double m = cabs2(r[Q][0]);
        const bool accept = !used[Q] && (m >= thr[Q]) && (m > 0.0);
        if (accept) {
          const double rm = 1.0 / m;
          dinv[Q] = make_double2(r[Q][0].x * rm, -r[Q][0].y * rm);
          r[Q][0] = make_double2(1.0, 0.0);
          used[Q] = true;
          if (live) {
#pragma unroll
            for (int j = 0; j < NB; ++j) prow[j] = r[Q][j];
            prow[NB] = dinv[Q];
            sm.pk[buf * G::TPC + t] = k;
            sm.perm[t * NB + k] = k;
          }
        }
        if (live) sm.ok[t] = accept ? 1 : 0;
        bad = (live && !accept) ? 1 : 0;
      }
    }
    int p = k;
    if (__syncthreads_or(bad)) {
      // rare path: every task whose candidate was rejected searches column k over its unused rows
      any_search = true;
      const bool need = sm.ok[t] == 0;
      if (need && live) {
        sm.mag[t * NB + a] = used[0] ? -1.0 : cabs2(r[0][0]);
        if (valid1) sm.mag[t * NB + a + TPT] = used[1] ? -1.0 : cabs2(r[1][0]);
      }
      __syncthreads();
      if (need) {
        int best = 0;
        double bm = sm.mag[t * NB];
        for (int i = 1; i < NB; ++i) {
          const double v = sm.mag[t * NB + i];
          if (v > bm) { bm = v; best = i; }
        }
#pragma unroll
        for (int q = 0; q < 2; ++q) {
          if (a + q * TPT == best) {
            const double rm = 1.0 / cabs2(r[q][0]);
            dinv[q] = make_double2(r[q][0].x * rm, -r[q][0].y * rm);
            r[q][0] = make_double2(1.0, 0.0);
            used[q] = true;
            if (live) {
#pragma unroll
              for (int j = 0; j < NB; ++j) prow[j] = r[q][j];
              prow[NB] = dinv[q];
              sm.pk[buf * G::TPC + t] = best;
              sm.perm[t * NB + k] = best;
            }
          }
        }
      }
      __syncthreads();
      p = sm.pk[buf * G::TPC + t];
    }
    {
      const c64 inv = prow[NB];
      const bool piv0 = (a == p), piv1 = (a + TPT == p);
      c64 f0 = cmul(r[0][0], inv), f1 = cmul(r[1][0], inv);
      if (piv0) f0 = make_double2(0.0, 0.0);
      if (piv1) f1 = make_double2(0.0, 0.0);
      // (hoisting or batching these loads in the source does not change the generated code: at 255
      // registers the allocator keeps a single pivot-row element in flight, and each load's latency is
      // exposed -- profiles/r01_final.md)
#pragma unroll
      for (int j = 0; j + 1 < NB; ++j) {
        const c64 pj = prow[j + 1];
        c64 t0 = r[0][j + 1], t1 = r[1][j + 1];
        cfms(t0, f0, pj);
        cfms(t1, f1, pj);
        r[0][j] = t0;
        r[1][j] = t1;
      }
      // the pivot column leaves, the new inverse column enters: 1 for the pivot row, -f for the others
      r[0][NB - 1] = make_double2((piv0 ? 1.0 : 0.0) - f0.x, -f0.y);
      r[1][NB - 1] = make_double2((piv1 ? 1.0 : 0.0) - f1.x, -f1.y);
    }
  }
}

// In-place Gauss-Jordan inversion, two rows per thread: r[q] is row a + q*TPT.  Same scheme as
// gj_invert (block_ops.cuh): the pivot row is published raw with a 1 in the pivot column plus the
// reciprocal pivot, every other row forms its own multiplier, all rows are scaled once at the end.
// The diagonal candidate a_kk is accepted when |a_kk|^2 >= theta2 * sum_j |a_kj(0)|^2, else the task
// searches column k over its unused rows.  On return thread a holds, in r[q], row perm^-1(a + q*TPT)
// of the inverse with register column j being inverse column perm[j]; the return value says
// (CTA-uniform) whether any task left the diagonal order (perm != identity possible).
template <int NB>
__device__ __forceinline__ bool gj_invert2(c64 (&r)[2][NB], const Smem2<NB>& sm, int t, int a, bool live,
                                           double theta2) {
  using G = Geo2<NB>;
  constexpr int TPT = G::TPT;
  const bool valid1 = a + TPT < NB;
  double thr[2];
  bool used[2] = {false, !valid1};
  c64 dinv[2];
#pragma unroll
  for (int q = 0; q < 2; ++q) {
    double m = 0.0;                      // row scale: squared 2-norm (cheaper than a NaN-aware max)
#pragma unroll
    for (int j = 0; j < NB; ++j) m = fma(r[q][j].x, r[q][j].x, fma(r[q][j].y, r[q][j].y, m));
    thr[q] = m * theta2;
    dinv[q] = make_double2(1.0, 0.0);
  }
  bool any_search = false;
  gj_phase2<NB>(r, sm, t, a, live, thr, used, dinv, 0, NB, any_search);
#pragma unroll
  for (int q = 0; q < 2; ++q)
#pragma unroll
    for (int j = 0; j < NB; ++j) r[q][j] = cmul(r[q][j], dinv[q]);
  return any_search;
}

// Write the inverse left in registers by gj_invert2 to the task's exchange matrix in logical
// (row, column) order.  Needs a barrier before anyone reads other rows.
template <int NB>
__device__ __forceinline__ void store_inverse2(const c64 (&r)[2][NB], c64* mat_t, const Smem2<NB>& sm, int t,
                                               int a, bool live, bool permuted) {
  constexpr int TPT = Geo2<NB>::TPT;
  if (!live) return;
#pragma unroll
  for (int q = 0; q < 2; ++q) {
    const int rid = a + q * TPT;
    if (rid >= NB) continue;
    if (!permuted) {
#pragma unroll
      for (int j = 0; j < NB; ++j) mat_t[rid * NB + j] = r[q][j];
    } else {
      const int* perm = sm.perm + t * NB;
      int row = 0;
      for (int k = 0; k < NB; ++k)
        if (perm[k] == rid) row = k;
#pragma unroll
      for (int j = 0; j < NB; ++j) mat_t[row * NB + perm[j]] = r[q][j];
    }
  }
}

}  // namespace blk
}  // namespace negf
