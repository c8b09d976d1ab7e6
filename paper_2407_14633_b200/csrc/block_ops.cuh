// Device primitives shared by the block (n x n, real-space) kernels: complex helpers, the one-row-per-
// thread geometry and Gauss-Jordan inversion used by sancho_rubio.cu (2n x 2n matrices), CSR tables
// in shared memory, block reductions.  The sweep kernels use the two-rows-per-thread geometry of
// block_ops2.cuh.
//
// One-row geometry: one thread owns one ROW of its task's matrix in registers; NB consecutive threads
// form a task; TPC tasks share a CTA and advance in lock step.  Tasks straddle warp boundaries, so
// rows are exchanged through shared memory and CTA barriers, never through shuffles.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace negf {
namespace blk {

typedef double2 c64;

__device__ __forceinline__ c64 cmul(c64 a, c64 b) {
  return make_double2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x);
}
__device__ __forceinline__ c64 cconj(c64 a) { return make_double2(a.x, -a.y); }
// acc += a * b
__device__ __forceinline__ void cfma(c64& acc, c64 a, c64 b) {
  acc.x = fma(a.x, b.x, acc.x);
  acc.x = fma(-a.y, b.y, acc.x);
  acc.y = fma(a.x, b.y, acc.y);
  acc.y = fma(a.y, b.x, acc.y);
}
// acc -= a * b
__device__ __forceinline__ void cfms(c64& acc, c64 a, c64 b) {
  acc.x = fma(-a.x, b.x, acc.x);
  acc.x = fma(a.y, b.y, acc.x);
  acc.y = fma(-a.x, b.y, acc.y);
  acc.y = fma(-a.y, b.x, acc.y);
}
__device__ __forceinline__ double cabs2(c64 a) { return fma(a.x, a.x, a.y * a.y); }
__device__ __forceinline__ c64 crcp(c64 d) {
  const double r = 1.0 / cabs2(d);
  return make_double2(d.x * r, -d.y * r);
}

template <int NB>
struct Geo {
  static constexpr int TPC = (255 / NB) > 32 ? 32 : (255 / NB);   // tasks per CTA
  static constexpr int LIVE = TPC * NB;                            // threads that own a row
  static constexpr int THREADS = (LIVE + 31) / 32 * 32;            // CTA size (ghosts pad the last warp)
  static constexpr int NWARPS = THREADS / 32;
  static constexpr int MAT = NB * NB;
  // one ring step of recursion history of one CTA: [column b][thread] complex, 16-byte coalesced
  static constexpr int64_t STEP_ELEMS = (int64_t)NB * THREADS;
};

// Sparse matrix in CSR form, read-only in shared memory.
struct Csr {
  const int* rowptr;   // [NB + 1]
  const int* col;      // [nnz]
  const c64* val;      // [nnz]
};

// Shared-memory working set of one CTA (carved from dynamic shared memory).
template <int NB>
struct Smem {
  c64* mat;      // [TPC][NB*NB]   one exchange matrix per task
  c64* prow;     // [2][TPC][NB+1] published pivot rows + inverse pivot (double buffered by elimination step)
  double* mag;   // [TPC][NB]      pivot-search magnitudes / small per-task reductions
  int* pk;       // [2][TPC]       pivot row of the current elimination step
  int* perm;     // [TPC][NB]      pivot row chosen for column k
  int* ok;       // [TPC]          1 if the diagonal candidate was accepted this step
  double* red;   // [2][NWARPS]    block reduction scratch

  static constexpr size_t bytes(int nmat = 1) {
    using G = Geo<NB>;
    return sizeof(c64) * ((size_t)nmat * G::TPC * G::MAT + 2 * G::TPC * (NB + 1)) +
           sizeof(double) * (G::TPC * NB + 2 * G::NWARPS) + sizeof(int) * (2 * G::TPC + G::TPC * NB + G::TPC) + 64;
  }
  // returns the first byte after the carved region (16-byte aligned)
  __device__ char* carve(char* base, int nmat = 1) {
    using G = Geo<NB>;
    mat = reinterpret_cast<c64*>(base);
    prow = mat + (size_t)nmat * G::TPC * G::MAT;
    mag = reinterpret_cast<double*>(prow + 2 * G::TPC * (NB + 1));
    red = mag + G::TPC * NB;
    pk = reinterpret_cast<int*>(red + 2 * G::NWARPS);
    perm = pk + 2 * G::TPC;
    ok = perm + G::TPC * NB;
    char* end = reinterpret_cast<char*>(ok + G::TPC);
    return reinterpret_cast<char*>((reinterpret_cast<uintptr_t>(end) + 15) & ~uintptr_t(15));
  }
};

// Default threshold of the diagonal-candidate test in gj_invert: the candidate pivot a_kk is accepted
// when |a_kk|^2 >= theta2 * sum_j |a_kj(0)|^2 (row k of the matrix as handed in); otherwise the task
// falls back to a full column search over its unused rows (partial pivoting).
// theta = 1e-4 (round 2; 1e-3 in round 1): on config 3 the search is then taken by 3 % of the inversions
// instead of 13 % (-1.9 % forward time) and the results against the oracle are unchanged (T(E) 1.1e-13);
// an emulation of the rule on 24 000 matrices of config 3 against an extended-precision inverse shows the
// same forward error as LAPACK for theta = 1e-4 ... 1e-2.
constexpr double kTheta2Default = 1e-8;

// In-place Gauss-Jordan inversion of the task's matrix, rows in registers (r = row `a`).
// The pivot row is NOT normalised during the elimination (that would be a divergent n-element
// scaling by one thread per step): its owner publishes the raw row with a 1 in the pivot column plus
// the reciprocal pivot; every other row forms its multiplier f = a_ik / a_kk itself and eliminates;
// all rows are scaled by their own reciprocal pivot once at the end.
// Pivoting is implicit (rows never move): on return, thread i holds row q(i) of the inverse with
// column j of its registers being inverse column perm[j], where perm[k] is the pivot row chosen for
// column k and q = perm^-1.  Returns (CTA-uniform) whether any task left the diagonal pivot order; if
// not, perm is the identity and r is row a of the inverse as is.
// Barriers: one __syncthreads_or per elimination step (+2 on the rare search path).  The caller
// must place at least one CTA barrier between two consecutive calls.
template <int NB>
__device__ __forceinline__ bool gj_invert(c64 (&r)[NB], const Smem<NB>& sm, int t, int a, bool live,
                                          double theta2) {
  using G = Geo<NB>;
  double thr = 0.0;                      // row scale: squared 2-norm (cheaper than a NaN-aware max)
#pragma unroll
  for (int j = 0; j < NB; ++j) thr = fma(r[j].x, r[j].x, fma(r[j].y, r[j].y, thr));
  thr *= theta2;
  bool used = false;
  bool any_search = false;
  c64 dinv = make_double2(1.0, 0.0);
  // The loop over elimination steps is not unrolled: after every step the registers are rotated by
  // one column (folded into the destination registers of the elimination FMAs), so the pivot column
  // is always register column 0 and the new inverse column enters at column NB-1; after NB steps the
  // columns are back in order.  (Unrolled, the 2n = 34 wide inversions of sancho_rubio.cu are
  // ~100 KB of code each and the kernel stalls on instruction fetch.)
#pragma unroll 1
  for (int k = 0; k < NB; ++k) {
    const int buf = k & 1;
    c64* prow = sm.prow + ((size_t)buf * G::TPC + t) * (NB + 1);
    int bad = 0;
    if (a == k) {
      const double m = cabs2(r[0]);
      const bool accept = !used && (m >= thr) && (m > 0.0);
      if (accept) {
        const double rm = 1.0 / m;
        dinv = make_double2(r[0].x * rm, -r[0].y * rm);
        r[0] = make_double2(1.0, 0.0);
        used = true;
        if (live) {
#pragma unroll
          for (int j = 0; j < NB; ++j) prow[j] = r[j];
          prow[NB] = dinv;
          sm.pk[buf * G::TPC + t] = a;
          sm.perm[t * NB + k] = a;
        }
      }
      if (live) sm.ok[t] = accept ? 1 : 0;
      bad = (live && !accept) ? 1 : 0;
    }
    int p = k;
    if (__syncthreads_or(bad)) {
      // rare path: every task whose candidate was rejected searches column k over its unused rows
      any_search = true;
      const bool need = sm.ok[t] == 0;
      if (need && live) sm.mag[t * NB + a] = used ? -1.0 : cabs2(r[0]);
      __syncthreads();
      if (need) {
        int best = 0;
        double bm = sm.mag[t * NB];
        for (int i = 1; i < NB; ++i) {
          const double v = sm.mag[t * NB + i];
          if (v > bm) { bm = v; best = i; }
        }
        if (a == best) {
          const double rm = 1.0 / cabs2(r[0]);
          dinv = make_double2(r[0].x * rm, -r[0].y * rm);
          r[0] = make_double2(1.0, 0.0);
          used = true;
          if (live) {
#pragma unroll
            for (int j = 0; j < NB; ++j) prow[j] = r[j];
            prow[NB] = dinv;
            sm.pk[buf * G::TPC + t] = a;
            sm.perm[t * NB + k] = a;
          }
        }
      }
      __syncthreads();
      p = sm.pk[buf * G::TPC + t];
    }
    {
      const bool piv = (a == p);
      c64 f = cmul(r[0], prow[NB]);
      if (piv) f = make_double2(0.0, 0.0);
#pragma unroll
      for (int j = 0; j + 1 < NB; ++j) {
        c64 tmp = r[j + 1];
        cfms(tmp, f, prow[j + 1]);
        r[j] = tmp;
      }
      r[NB - 1] = make_double2((piv ? 1.0 : 0.0) - f.x, -f.y);
    }
  }
#pragma unroll
  for (int j = 0; j < NB; ++j) r[j] = cmul(r[j], dinv);
  return any_search;
}

// Write the inverse left in registers by gj_invert to the task's exchange matrix in logical
// (row, column) order.  Needs a barrier before anyone reads other rows.
template <int NB>
__device__ __forceinline__ void store_inverse(const c64 (&r)[NB], c64* mat_t, const Smem<NB>& sm, int t,
                                              int a, bool live, bool permuted) {
  if (!live) return;
  if (!permuted) {
#pragma unroll
    for (int j = 0; j < NB; ++j) mat_t[a * NB + j] = r[j];
  } else {
    const int* perm = sm.perm + t * NB;
    int row = 0;
#pragma unroll
    for (int k = 0; k < NB; ++k)
      if (perm[k] == a) row = k;
#pragma unroll
    for (int j = 0; j < NB; ++j) mat_t[row * NB + perm[j]] = r[j];
  }
}

// c[b] = sum_k arow[k] * X[k][b]   (row of A X: A row in registers, X in shared memory)
template <int NB>
__device__ __forceinline__ void gemm_row(c64 (&c)[NB], const c64 (&arow)[NB], const c64* X) {
#pragma unroll
  for (int b = 0; b < NB; ++b) c[b] = make_double2(0.0, 0.0);
#pragma unroll
  for (int k = 0; k < NB; ++k) {
    const c64 av = arow[k];
#pragma unroll
    for (int b = 0; b < NB; ++b) cfma(c[b], av, X[k * NB + b]);
  }
}

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

__device__ __forceinline__ double fermi(double E, double mu, double kT) {
  const double x = (E - mu) / kT;
  const double e = exp(-fabs(x));
  return x > 0.0 ? e / (1.0 + e) : 1.0 / (1.0 + e);
}

// Copy a CSR matrix from global to shared memory (all threads; caller barriers afterwards).
__device__ __forceinline__ char* csr_to_shared(Csr& dst, char* base, const int* g_rowptr, const int* g_col,
                                               const c64* g_val, int nb, int nnz_cap) {
  // layout: val[nnz_cap] (16-byte aligned), rowptr[nb+1], col[nnz_cap]
  c64* val = reinterpret_cast<c64*>(base);
  int* rowptr = reinterpret_cast<int*>(val + nnz_cap);
  int* col = rowptr + nb + 1;
  const int nnz = g_rowptr[nb];
  for (int i = threadIdx.x; i <= nb; i += blockDim.x) rowptr[i] = g_rowptr[i];
  for (int i = threadIdx.x; i < nnz; i += blockDim.x) {
    col[i] = g_col[i];
    val[i] = g_val[i];
  }
  dst.rowptr = rowptr;
  dst.col = col;
  dst.val = val;
  char* end = reinterpret_cast<char*>(col + nnz_cap);
  return reinterpret_cast<char*>((reinterpret_cast<uintptr_t>(end) + 15) & ~uintptr_t(15));
}
// Explicit shared-memory loads (32-bit shared addresses): the CSR tables are reached through
// pointers selected at run time, for which the compiler otherwise falls back to generic loads.
__device__ __forceinline__ unsigned smem_addr(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ int lds_i32(unsigned addr) {
  int v;
  asm volatile("ld.shared.s32 %0, [%1];" : "=r"(v) : "r"(addr));
  return v;
}
__device__ __forceinline__ c64 lds_c64(unsigned addr) {
  c64 v;
  asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(v.x), "=d"(v.y) : "r"(addr));
  return v;
}
struct CsrS {            // CSR matrix in shared memory, by shared address
  unsigned rowptr, col, val;
};
__device__ __forceinline__ CsrS csr_shared(const Csr& K) {
  return CsrS{smem_addr(K.rowptr), smem_addr(K.col), smem_addr(K.val)};
}

__host__ __device__ constexpr size_t csr_shared_bytes(int nb, int nnz_cap) {
  return ((sizeof(double2) * (size_t)nnz_cap + sizeof(int) * (size_t)(nb + 1 + nnz_cap)) + 15) / 16 * 16;
}

}  // namespace blk
}  // namespace negf
