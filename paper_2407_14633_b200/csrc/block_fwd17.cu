// Forward half of the block RGF sweep for n = 17, real-axis energies (step a2 of SURVEY.md 8(a);
// Algorithm 2 of PAPER.md:121-141 for the connected Green's functions ytilde_s):
//     d_s = z - U_s - K_s ytilde_{s-1} (- Sigma at the two ends),  g_s = d_s^-1,
//     ytilde_s = g_s K_{s+1}^dagger   (stored as written: the way back, block_back.cu, reads it),
// one half-sweep task (channel, energy, direction) per EIGHT lanes: four tasks per warp, eight per CTA,
// no CTA barrier and no shared-memory pivot traffic inside a ring (block_ops17.cuh).  A warp owns its four
// tasks for the whole sweep; the two warps of a CTA only share the coupling tables.
//
// CTA numbering, history layout (row-major records of kHistRec17 elements per task and ring, row stride
// 18) and the table of lead self-energies are those of block_sweep.cu / block_back.cu; a real-axis CTA of
// n = 17 holds kTpc17 = 8 consecutive energies.
#include "block_ops17.cuh"
#include "block_ops2.cuh"
#include "block_path.h"
#include "negf_internal.h"

namespace negf {
namespace blk {

namespace {

constexpr int NB = 17;
constexpr int MAT = NB * NB;
constexpr int kFwdThreads17 = 64;

__device__ __forceinline__ void st32(c64* dst, c64 a, c64 b) {          // one full 32-byte sector
  asm volatile("st.global.v4.f64 [%0], {%1, %2, %3, %4};" ::"l"(dst), "d"(a.x), "d"(a.y), "d"(b.x), "d"(b.y)
               : "memory");
}
// a row of ytilde_s: 17 elements + the padding element, nine full sectors
__device__ __forceinline__ void store_row17(c64* dst, const c64 (&row)[NB]) {
#pragma unroll
  for (int j = 0; j < 8; ++j) st32(dst + 2 * j, row[2 * j], row[2 * j + 1]);
  st32(dst + 16, row[16], make_double2(0.0, 0.0));
}

// A coupling matrix in shared memory as padded rows: W = row_nnz_max entries per row (value 0, column 0 where a
// row has fewer), [17][W] values and [17][W] column indices, by shared address.  No row pointers: every row
// loop has the same trip count, so the loads of one row are independent of each other.
struct EllS {
  unsigned val, col;
};

// rows l8, l8 + 8 and the lane's share of row 16 of  -K X   (X: the task's matrix in shared memory)
__device__ __forceinline__ void sparse_left17(c64 (&R)[2][NB], c64 (&S)[3], const EllS K, int W, unsigned X, int l8) {
#pragma unroll
  for (int q = 0; q < 2; ++q) {
#pragma unroll
    for (int b = 0; b < NB; ++b) R[q][b] = make_double2(0.0, 0.0);
    const int e0 = (l8 + 8 * q) * W;
#pragma unroll 1
    for (int e = e0; e < e0 + W; ++e) {
      const c64 v = lds_c64(K.val + 16 * e);
      const unsigned xr = X + (unsigned)lds_i32(K.col + 4 * e) * (NB * 16);
#pragma unroll
      for (int b = 0; b < NB; ++b) cfms(R[q][b], v, lds_c64(xr + 16 * b));
    }
  }
  S[0] = S[1] = S[2] = make_double2(0.0, 0.0);
#pragma unroll 1
  for (int e = 16 * W; e < 17 * W; ++e) {
    const c64 v = lds_c64(K.val + 16 * e);
    const unsigned xr = X + (unsigned)lds_i32(K.col + 4 * e) * (NB * 16);
    cfms(S[0], v, lds_c64(xr + 16 * l8));
    cfms(S[1], v, lds_c64(xr + 16 * (l8 + 8)));
    cfms(S[2], v, lds_c64(xr + 16 * 16));
  }
}

// one element of X K^dagger: sum over the W entries of row b of K of X[r][col] conj(val)   (xr: row r of X)
template <int WT>
__device__ __forceinline__ c64 ell_row_dot(const EllS K, int W, int b, unsigned xr) {
  c64 acc = make_double2(0.0, 0.0);
  if (WT > 0) {
#pragma unroll
    for (int w = 0; w < WT; ++w) {
      const int e = b * WT + w;
      cfma(acc, lds_c64(xr + 16u * (unsigned)lds_i32(K.col + 4 * e)), cconj(lds_c64(K.val + 16 * e)));
    }
  } else {
#pragma unroll 1
    for (int e = b * W; e < b * W + W; ++e)
      cfma(acc, lds_c64(xr + 16u * (unsigned)lds_i32(K.col + 4 * e)), cconj(lds_c64(K.val + 16 * e)));
  }
  return acc;
}

// ytilde = X K^dagger in place in the task's shared-memory matrix X, and the lane's share of it in R, S:
//     (X K^dagger)[r][b] = sum_{d in nz(K_b)} X[r][d] conj(K[b][d]).
// Rolled over the output column b on purpose (code size, block_ops17.cuh): an output row depends on the same
// input row only, so a lane forms a row in its private temporary row `tmp` and then replaces the input row;
// row 16 is spread over the lanes and held in registers until every lane has read it.
template <int WT>
__device__ __forceinline__ void sparse_right_dagger17(c64 (&R)[2][NB], c64 (&S)[3], const EllS K, int W, unsigned X,
                                                      c64* mat_t, unsigned tmp, int l8) {
  const unsigned x16 = X + 16 * (NB * 16);
  S[0] = ell_row_dot<WT>(K, W, l8, x16);
  S[1] = ell_row_dot<WT>(K, W, l8 + 8, x16);
  S[2] = ell_row_dot<WT>(K, W, 16, x16);
#pragma unroll
  for (int q = 0; q < 2; ++q) {
    const unsigned xr = X + (l8 + 8 * q) * (NB * 16);
#pragma unroll 2
    for (int b = 0; b < NB; ++b) {
      const c64 acc = ell_row_dot<WT>(K, W, b, xr);
      asm volatile("st.shared.v2.f64 [%0], {%1, %2};" ::"r"(tmp + 16u * b), "d"(acc.x), "d"(acc.y) : "memory");
    }
#pragma unroll
    for (int b = 0; b < NB; ++b) {
      R[q][b] = lds_c64(tmp + 16u * b);
      mat_t[(l8 + 8 * q) * NB + b] = R[q][b];
    }
  }
  __syncwarp();                              // every lane has read row 16 of X
  mat_t[16 * NB + l8] = S[0];
  mat_t[16 * NB + l8 + 8] = S[1];
  if (l8 == 0) mat_t[16 * NB + 16] = S[2];
}

// the lane's rows (17 columns) to the task's shared-memory matrix
__device__ __forceinline__ void rows_to_shared17(c64* mat_t, const c64 (&R)[2][NB], int l8) {
#pragma unroll
  for (int q = 0; q < 2; ++q)
#pragma unroll
    for (int b = 0; b < NB; ++b) mat_t[(l8 + 8 * q) * NB + b] = R[q][b];
}
__device__ __forceinline__ void from_shared17(c64 (&R)[2][NB], c64 (&S)[3], const c64* mat_t, int l8) {
#pragma unroll
  for (int q = 0; q < 2; ++q)
#pragma unroll
    for (int b = 0; b < NB; ++b) R[q][b] = mat_t[(l8 + 8 * q) * NB + b];
  S[0] = mat_t[16 * NB + l8];
  S[1] = mat_t[16 * NB + l8 + 8];
  S[2] = mat_t[16 * NB + 16];
}
// the task's matrix (registers, layout of block_ops17.cuh) to its shared-memory matrix, row-major
__device__ __forceinline__ void to_shared17(c64* mat_t, const c64 (&R)[2][NB], const c64 (&S)[3], int l8) {
#pragma unroll
  for (int q = 0; q < 2; ++q)
#pragma unroll
    for (int b = 0; b < NB; ++b) mat_t[(l8 + 8 * q) * NB + b] = R[q][b];
  mat_t[16 * NB + l8] = S[0];
  mat_t[16 * NB + l8 + 8] = S[1];
  if (l8 == 0) mat_t[16 * NB + 16] = S[2];
}

size_t ell_bytes(int W) { return ((size_t)NB * W * (sizeof(c64) + sizeof(int)) + 15) / 16 * 16; }
size_t fwd17_smem(int row_nnz_max) {
  // exchange matrices, one temporary row per thread, column-search records, the two couplings as padded rows
  // and their diagonals
  return sizeof(c64) * kTpc17 * MAT + sizeof(c64) * kFwdThreads17 * NB + sizeof(Rare17) * kTpc17 +
         2 * ell_bytes(row_nnz_max) + 2 * NB * sizeof(c64) + 32;
}

}  // namespace

__global__ void __launch_bounds__(kFwdThreads17, 4) block_fwd17_kernel(const SweepLaunch p, long long first_gid) {
  constexpr long long STEP = Geo2<NB>::STEP_ELEMS;
  extern __shared__ __align__(16) char smem_raw[];
  c64* mat = reinterpret_cast<c64*>(smem_raw);                    // [kTpc17][17 x 17]
  c64* tmp_all = mat + kTpc17 * MAT;                              // [threads][17]
  Rare17* rare_all = reinterpret_cast<Rare17*>(tmp_all + kFwdThreads17 * NB);
  char* nxt = reinterpret_cast<char*>(rare_all + kTpc17);
  const int tid = threadIdx.x, lane = tid & 31;
  const int l8 = lane & 7, base = lane & 24, t = tid >> 3;
  const int N = p.N;
  const long long gid = first_gid + blockIdx.x;
  // real-axis CTA numbering of block_sweep.cu: after the contour CTAs, (channel, group, direction)
  const long long rr = gid - p.n_eq_cta;
  const int per = 2 * p.gneq;
  const int c = (int)(rr / per);
  const int rem = (int)(rr - (long long)c * per);
  const int grp = rem >> 1, dir = rem & 1;
  int k = grp * kTpc17 + t;
  if (k >= p.K_neq) k = p.K_neq - 1;       // a padding task repeats the last energy; nobody reads its history
  const c64 z = p.z_neq[k];
  const size_t K_all = (size_t)p.K_eq + p.K_neq;
  const size_t tab_off = (((size_t)c * K_all + p.K_eq + k) * 2 + 0) * 2 * MAT;
#define NEGF_TAB_FIRST (p.table + tab_off + (dir ? 2 * MAT : 0))
#define NEGF_TAB_LAST (p.table + tab_off + (dir ? 0 : 2 * MAT))

  // couplings of this direction, by parity of the bond: [0] even bond, [1] odd bond (as in block_sweep.cu)
  // Nothing here is an array indexed by the parity: such arrays live in local memory, and a local load per
  // ring showed up as 10 % long-scoreboard stalls.  The two tables are a fixed stride apart instead.
  const int W = p.csr.row_nnz_max;
  const unsigned ell_stride = (unsigned)(((size_t)NB * W * (sizeof(c64) + sizeof(int)) + 15) / 16 * 16);
  const unsigned ell0 = smem_addr(nxt);            // table x: values at ell0 + x * ell_stride, then the columns
  c64* kd0 = reinterpret_cast<c64*>(nxt + 2 * ell_stride);   // diagonals: kd0 + x * NB
  int diag_bits = 0;                               // bit x: coupling x is a diagonal matrix
  {
    const int mm[2] = {dir ? CSR_E : CSR_EDAG, dir ? CSR_O : CSR_ODAG};
#pragma unroll
    for (int x = 0; x < 2; ++x) {
      c64* ev = reinterpret_cast<c64*>(nxt + x * ell_stride);
      int* ec = reinterpret_cast<int*>(ev + NB * W);
      const int* rp = p.csr.rowptr + mm[x] * (NB + 1);
      const int* gc = p.csr.col + (size_t)mm[x] * p.csr.nnz_cap;
      const c64* gv = p.csr.val + (size_t)mm[x] * p.csr.nnz_cap;
      for (int i = tid; i < NB * W; i += kFwdThreads17) {
        const int b = i / W, e = rp[b] + (i - b * W);
        const bool in = e < rp[b + 1];
        ev[i] = in ? gv[e] : make_double2(0.0, 0.0);
        ec[i] = in ? gc[e] : 0;
      }
      for (int i = tid; i < NB; i += kFwdThreads17) kd0[x * NB + i] = p.csr.diag[mm[x] * NB + i];
      diag_bits |= ((p.csr.diag_mask >> mm[x]) & 1) << x;
    }
  }
  auto ell = [&](int x) { return EllS{ell0 + x * ell_stride, ell0 + x * ell_stride + (unsigned)(NB * W * sizeof(c64))}; };
  Rare17* rare = rare_all + t;
  __syncthreads();                          // the only CTA barrier: from here every warp runs on its own

  c64* mat_t = mat + (size_t)t * MAT;
  const unsigned mat_s = smem_addr(mat_t);
  const unsigned tmp_s = smem_addr(tmp_all + (size_t)tid * NB);
  c64* hrec = p.hist + (size_t)(gid - p.cta_begin) * N * STEP + (size_t)t * kHistRec17;   // + s * STEP

  // Loop invariant at the top of step s > 0: R, S = the lane's share of ytilde_{s-1}; if the coupling
  // entering step s is not diagonal, ytilde_{s-1} is also in the task's shared-memory matrix.
  c64 R[2][NB], S[3];
  for (int s = 0; s < N; ++s) {
    const int i = dir ? N - 1 - s : s;
    const double u_i = p.U[(size_t)c * N + i];     // used after the product below: the load has time
    if (s == 0) {
      const c64* tab = NEGF_TAB_FIRST;
#pragma unroll
      for (int q = 0; q < 2; ++q)
#pragma unroll
        for (int b = 0; b < NB; ++b) {
          const c64 v = tab[(l8 + 8 * q) * NB + b];
          R[q][b] = make_double2(-v.x, -v.y);
        }
      const c64 v0 = tab[16 * NB + l8], v1 = tab[16 * NB + l8 + 8], v2 = tab[16 * NB + 16];
      S[0] = make_double2(-v0.x, -v0.y);
      S[1] = make_double2(-v1.x, -v1.y);
      S[2] = make_double2(-v2.x, -v2.y);
    } else {
      const int par = dir ? (i & 1) : ((i - 1) & 1);
      // d := -K_s ytilde_{s-1}
      if ((diag_bits >> par) & 1) {
        const c64* kdp = kd0 + par * NB;
        const c64 k0 = kdp[l8], k1 = kdp[l8 + 8], k2 = kdp[16];
        const c64 n0 = make_double2(-k0.x, -k0.y), n1 = make_double2(-k1.x, -k1.y);
        const c64 n2 = make_double2(-k2.x, -k2.y);
#pragma unroll
        for (int b = 0; b < NB; ++b) {
          R[0][b] = cmul(n0, R[0][b]);
          R[1][b] = cmul(n1, R[1][b]);
        }
        S[0] = cmul(n2, S[0]);
        S[1] = cmul(n2, S[1]);
        S[2] = cmul(n2, S[2]);
      } else {
        sparse_left17(R, S, ell(par), W, mat_s, l8);
      }
    }
    if (s == N - 1) {
      const c64* tab = NEGF_TAB_LAST;
#pragma unroll
      for (int q = 0; q < 2; ++q)
#pragma unroll
        for (int b = 0; b < NB; ++b) {
          const c64 v = tab[(l8 + 8 * q) * NB + b];
          R[q][b].x -= v.x;
          R[q][b].y -= v.y;
        }
      const c64 v0 = tab[16 * NB + l8], v1 = tab[16 * NB + l8 + 8], v2 = tab[16 * NB + 16];
      S[0].x -= v0.x; S[0].y -= v0.y;
      S[1].x -= v1.x; S[1].y -= v1.y;
      S[2].x -= v2.x; S[2].y -= v2.y;
    }
    const double zu = z.x - u_i;
#pragma unroll
    for (int b = 0; b < 8; ++b)
      if (b == l8) {
        R[0][b].x += zu; R[0][b].y += z.y;
        R[1][b + 8].x += zu; R[1][b + 8].y += z.y;
      }
    S[2].x += zu;
    S[2].y += z.y;

    __syncwarp();                            // the shared-memory matrix is free (scratch of the inversion)
    if (__all_sync(kFullMask, invert17_first_ok(S, p.theta2))) {
      const c64 dinv16 = invert17_core(R, S, p.theta2, l8, base, mat_t, rare);
      rows_to_shared17(mat_t, R, l8);        // G and -G b d^-1 beside c (row 16)
      __syncwarp();
      invert17_border(S, dinv16, mat_s, l8);
      __syncwarp();
      mat_t[16 * NB + l8] = S[0];            // the complete inverse is in shared memory
      mat_t[16 * NB + l8 + 8] = S[1];
      if (l8 == 0) mat_t[16 * NB + 16] = S[2];
    } else {
      to_shared17(mat_t, R, S, l8);          // rare: partial pivoting in shared memory for the whole warp
      __syncwarp();
      invert17_slow(mat_t, l8);
      from_shared17(R, S, mat_t, l8);
    }

    int parn = 0;
    bool next_diag = false;
    if (s < N - 1) {
      const int inext = dir ? i - 1 : i + 1;
      parn = dir ? (inext & 1) : ((inext - 1) & 1);
      next_diag = (diag_bits >> parn) & 1;
    }
    c64* h = hrec + (size_t)s * STEP;
    if (s == N - 1 || next_diag) {
      if (s < N - 1) {                       // ytilde_ab = g_ab conj(K_bb); last ring: G_(k,k) itself
        const c64* kdn = kd0 + parn * NB;
#pragma unroll
        for (int b = 0; b < NB; ++b) {
          const c64 kb = cconj(kdn[b]);
          R[0][b] = cmul(R[0][b], kb);
          R[1][b] = cmul(R[1][b], kb);
        }
        S[0] = cmul(S[0], cconj(kdn[l8]));
        S[1] = cmul(S[1], cconj(kdn[l8 + 8]));
        S[2] = cmul(S[2], cconj(kdn[16]));
        mat_t[16 * NB + l8] = S[0];          // row 16 goes out through shared memory: full sectors
        mat_t[16 * NB + l8 + 8] = S[1];
        if (l8 == 0) mat_t[16 * NB + 16] = S[2];
      }
    } else {
      // ytilde_s = g_s K_{s+1}^dagger
      if (W == 2) sparse_right_dagger17<2>(R, S, ell(parn), W, mat_s, mat_t, tmp_s, l8);
      else sparse_right_dagger17<0>(R, S, ell(parn), W, mat_s, mat_t, tmp_s, l8);
    }
    __syncwarp();
    store_row17(h + l8 * kHistLd17, R[0]);
    store_row17(h + (l8 + 8) * kHistLd17, R[1]);
    {
      const c64* r16 = mat_t + 16 * NB;
      st32(h + 16 * kHistLd17 + 2 * l8, r16[2 * l8], r16[2 * l8 + 1]);
      if (l8 == 0) st32(h + 16 * kHistLd17 + 16, r16[16], make_double2(0.0, 0.0));
    }
  }
#undef NEGF_TAB_FIRST
#undef NEGF_TAB_LAST
}

cudaError_t launch_block_fwd17(const SweepLaunch& p, cudaStream_t s) {
  // real-axis CTAs of this launch: global ids [max(cta_begin, n_eq_cta), cta_begin + n_cta)
  const long long first = p.cta_begin > p.n_eq_cta ? p.cta_begin : p.n_eq_cta;
  const long long n = p.cta_begin + p.n_cta - first;
  if (n <= 0) return cudaSuccess;
  const size_t smem = fwd17_smem(p.csr.row_nnz_max);
  cudaError_t e = cudaFuncSetAttribute(block_fwd17_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e != cudaSuccess) return e;
  block_fwd17_kernel<<<(unsigned)n, kFwdThreads17, smem, s>>>(p, first);
  return cudaGetLastError();
}

int block_fwd17_ctas_per_sm(int row_nnz_max) {
  int nb = 0;
  const size_t smem = fwd17_smem(row_nnz_max);
  if (cudaFuncSetAttribute(block_fwd17_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess)
    return 0;
  if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, block_fwd17_kernel, kFwdThreads17, smem) != cudaSuccess)
    return 0;
  return nb;
}

}  // namespace blk
}  // namespace negf
