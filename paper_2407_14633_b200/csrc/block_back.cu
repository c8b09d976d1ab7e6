// Way back of the block RGF sweep for n = 17 on the FP64 tensor cores (DMMA, mma.sync.m8n8k4.f64):
// the column recursion of Algorithm 1 steps 2-3 and 6-8 from the last lead k,
//     C_{N-1} = g_{N-1} F_k,   C_s = ytilde_s C_{s+1},   Tr A_k,(i,i) = ||C_s||_F^2,
//     T = ||F_first^dagger C_0||_F^2   (eq.(5)),
// with ytilde_s read from the history that block_fwd17_kernel wrote.
//
// This half of the sweep is a plain 17 x 17 complex product per ring with no pivoting, i.e. a dense
// contraction once the 17th row and column are split off: the 16 x 16 x 16 core is 2 x 2 output
// tiles x 4 k-steps x 4 real products = 64 DMMA instructions (256 FMAs each, no padding), the
// border (k = 16 term, last row, last column, corner: 17 % of the FMAs) runs on the FP64 SIMT pipe
// from the same fragments with quad shuffles.  The measured DMMA peak equals the DFMA peak on B200,
// so the gain is not peak: it is one issue slot per 256 FMAs instead of 8, and one 8-byte operand per
// lane per 128 FMAs instead of one 16-byte operand per 8, which is what bounded the SIMT version.
//
// One warp per half-sweep task, 8 warps per CTA (the 8 tasks of one block_fwd17 CTA, whose partial-
// charge row they share); no barrier inside a ring.  The history of a task and ring is the row-major
// matrix ytilde_s with row stride 18 (rows start on 32-byte sectors); A fragment (mt, ks) of lane l is
// element [8 mt + l/4][4 ks + l%4]: four lanes read one aligned 64-byte piece, 16 full sectors per load.
#include "block_ops17.cuh"
#include "block_ops2.cuh"
#include "block_path.h"
#include "negf_internal.h"

namespace negf {
namespace blk {

namespace {

constexpr int NB17 = 17;
constexpr int LDB = 18;            // leading dimension of the B operand in shared memory (conflict-free)
constexpr double kPi17 = 3.14159265358979323846;

__device__ __forceinline__ void dmma(double (&d)[2], double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
               : "+d"(d[0]), "+d"(d[1])
               : "d"(a), "d"(b));
}
__device__ __forceinline__ c64 shfl_c64(c64 v, int src) {
  return make_double2(__shfl_sync(0xffffffffu, v.x, src), __shfl_sync(0xffffffffu, v.y, src));
}
__device__ __forceinline__ double quad_sum(double v) {
  v += __shfl_xor_sync(0xffffffffu, v, 1);
  v += __shfl_xor_sync(0xffffffffu, v, 2);
  return v;
}
__device__ __forceinline__ c64 quad_sum(c64 v) { return make_double2(quad_sum(v.x), quad_sum(v.y)); }

struct CtaId17 {
  int c, grp, dir;
};
// real-axis CTA numbering of block_sweep.cu: after the C*geq*2 contour CTAs, (channel, group, direction)
__device__ __forceinline__ CtaId17 decode_real_cta(const SweepLaunch& p, long long gid) {
  const long long r = gid - p.n_eq_cta;
  const int per = 2 * p.gneq;
  CtaId17 id;
  id.c = (int)(r / per);
  const int rem = (int)(r - (long long)id.c * per);
  id.grp = rem >> 1;
  id.dir = rem & 1;
  return id;
}

}  // namespace

__global__ void __launch_bounds__(kBackThreads17, 2) block_back17_kernel(const SweepLaunch p, long long first_gid) {
  using G = Geo2<NB17>;
  constexpr int TPC = kTpc17;                       // 8 tasks = 8 warps
  constexpr long long STEP = G::STEP_ELEMS;
  constexpr int MAT = NB17 * NB17;
  __shared__ __align__(16) c64 Bs_all[TPC][NB17 * LDB];
  __shared__ double red[TPC][32];
  const int tid = threadIdx.x;
  const int lane = tid & 31, t = tid >> 5;
  const int g = lane >> 2, q4 = lane & 3;
  const int N = p.N;
  const long long gid = first_gid + blockIdx.x;
  const CtaId17 id = decode_real_cta(p, gid);
  const int dir = id.dir;
  const size_t slot = (size_t)(gid - p.cta_begin);
  int k = id.grp * TPC + t;
  const bool active = k < p.K_neq;
  if (!active) k = p.K_neq - 1;
  const c64 z = p.z_neq[k];
  const size_t K_all = (size_t)p.K_eq + p.K_neq;
  const c64* tabL = p.table + (((size_t)id.c * K_all + p.K_eq + k) * 2 + 0) * 2 * MAT;
  const c64* tabR = tabL + 2 * MAT;
  const c64* F_last = (dir ? tabL : tabR) + MAT;
  const c64* F_first = (dir ? tabR : tabL) + MAT;
  const int R = p.geq + 2 * p.gneq;
  double* prow_out = p.partial + ((size_t)id.c * R + p.geq + 2 * id.grp + dir) * N;
  const double f_last = fermi(z.x, dir ? p.mu_s : p.mu_d, p.kT);
  const double wt = active ? p.deg * p.w_neq[k] * (1.0 / (2.0 * kPi17)) * f_last : 0.0;

  c64* Bs = Bs_all[t];
  for (int e = lane; e < MAT; e += 32) Bs[(e / NB17) * LDB + (e % NB17)] = F_last[e];   // C_N := F_k
  const c64* hrec = p.hist + (slot * (size_t)N + (N - 1)) * STEP + (size_t)t * kHistRec17;
  const int off_frag = g * kHistLd17 + q4;                               // + mt*8*18 + ks*4
  const int off_bord = lane < 16 ? lane * kHistLd17 + 16 : 16 * kHistLd17 + (lane - 16);

  double keep = 0.0;
  int cnt = 0;                                       // rings done; ring N-1-cnt is next
  for (int s = N - 1; s >= 0; --s, hrec -= STEP, ++cnt) {
    // ---- operands of this ring: A fragments and border of ytilde_s
    c64 Ar[2][4];
#pragma unroll
    for (int mt = 0; mt < 2; ++mt)
#pragma unroll
      for (int ks = 0; ks < 4; ++ks) Ar[mt][ks] = hrec[off_frag + mt * 8 * kHistLd17 + ks * 4];
    const c64 bord = hrec[off_bord];                 // lane l < 16: ytilde[l][16]; lane 16+j: ytilde[16][j]
    const c64 acorner = hrec[16 * kHistLd17 + 16];   // ytilde[16][16]
    if (s > 0) {                                     // next ring's 39 lines towards L2
      const char* nx = reinterpret_cast<const char*>(hrec - STEP);
      asm volatile("prefetch.global.L2 [%0];" ::"l"(nx + 128 * lane));
      if (lane < 7) asm volatile("prefetch.global.L2 [%0];" ::"l"(nx + 128 * (32 + lane)));
    }
    __syncwarp();                                    // C_{s+1} of the previous ring is in Bs

    double cre[2][2][2], cim[2][2][2];
#pragma unroll
    for (int mt = 0; mt < 2; ++mt)
#pragma unroll
      for (int nt = 0; nt < 2; ++nt) cre[mt][nt][0] = cre[mt][nt][1] = cim[mt][nt][0] = cim[mt][nt][1] = 0.0;
    c64 colp[2] = {make_double2(0.0, 0.0), make_double2(0.0, 0.0)};   // C[8 mt + g][16], partial over q4
    c64 rowp[2] = {make_double2(0.0, 0.0), make_double2(0.0, 0.0)};   // C[16][8 nt + g]
    c64 cornp = make_double2(0.0, 0.0);                               // C[16][16]
#pragma unroll
    for (int ks = 0; ks < 4; ++ks) {
      const int kr = 4 * ks + q4;
      const c64 b0 = Bs[kr * LDB + g], b1 = Bs[kr * LDB + 8 + g];     // B fragments, nt = 0, 1
      const c64 b16 = Bs[kr * LDB + 16];
      const c64 a16 = shfl_c64(bord, 16 + kr);                        // ytilde[16][kr]
#pragma unroll
      for (int mt = 0; mt < 2; ++mt) {
        const c64 av = Ar[mt][ks];
        const double nai = -av.y;
        dmma(cre[mt][0], av.x, b0.x);
        dmma(cre[mt][0], nai, b0.y);
        dmma(cim[mt][0], av.x, b0.y);
        dmma(cim[mt][0], av.y, b0.x);
        dmma(cre[mt][1], av.x, b1.x);
        dmma(cre[mt][1], nai, b1.y);
        dmma(cim[mt][1], av.x, b1.y);
        dmma(cim[mt][1], av.y, b1.x);
        cfma(colp[mt], av, b16);
      }
      cfma(rowp[0], a16, b0);
      cfma(rowp[1], a16, b1);
      cfma(cornp, a16, b16);
    }
    // ---- k = 16 terms and the quad reductions of the border sums
    const c64 b1616 = Bs[16 * LDB + 16];
    c64 colv[2], rowv[2];
#pragma unroll
    for (int mt = 0; mt < 2; ++mt) {
      const c64 ar16 = shfl_c64(bord, 8 * mt + g);                    // ytilde[8 mt + g][16]
#pragma unroll
      for (int nt = 0; nt < 2; ++nt)
#pragma unroll
        for (int i2 = 0; i2 < 2; ++i2) {
          const c64 bl = Bs[16 * LDB + 8 * nt + 2 * q4 + i2];
          cre[mt][nt][i2] = fma(ar16.x, bl.x, cre[mt][nt][i2]);
          cre[mt][nt][i2] = fma(-ar16.y, bl.y, cre[mt][nt][i2]);
          cim[mt][nt][i2] = fma(ar16.x, bl.y, cim[mt][nt][i2]);
          cim[mt][nt][i2] = fma(ar16.y, bl.x, cim[mt][nt][i2]);
        }
      colv[mt] = quad_sum(colp[mt]);
      cfma(colv[mt], ar16, b1616);
    }
#pragma unroll
    for (int nt = 0; nt < 2; ++nt) {
      rowv[nt] = quad_sum(rowp[nt]);
      cfma(rowv[nt], acorner, Bs[16 * LDB + 8 * nt + g]);
    }
    c64 cornv = quad_sum(cornp);
    cfma(cornv, acorner, b1616);

    // ---- Tr A_k,(i,i) = ||C_s||_F^2
    double v = 0.0;
#pragma unroll
    for (int mt = 0; mt < 2; ++mt)
#pragma unroll
      for (int nt = 0; nt < 2; ++nt)
#pragma unroll
        for (int i2 = 0; i2 < 2; ++i2) v = fma(cre[mt][nt][i2], cre[mt][nt][i2], fma(cim[mt][nt][i2], cim[mt][nt][i2], v));
    if (q4 == 0) v += cabs2(colv[0]) + cabs2(colv[1]) + cabs2(rowv[0]) + cabs2(rowv[1]);
    if (lane == 0) v += cabs2(cornv);
    v = warp_sum(v);
    if (lane == (cnt & 31)) keep = wt * v;
    if (p.probe && (dir ? N - 1 - s : s) == p.probe_ring && lane == 0 && active)
      p.probe[((size_t)id.c * 2 + dir) * p.K_neq + k] = wt * v;

    // ---- C_s becomes the B operand of the next ring
    __syncwarp();                                    // every lane has read C_{s+1}
#pragma unroll
    for (int mt = 0; mt < 2; ++mt)
#pragma unroll
      for (int nt = 0; nt < 2; ++nt)
#pragma unroll
        for (int i2 = 0; i2 < 2; ++i2)
          Bs[(8 * mt + g) * LDB + 8 * nt + 2 * q4 + i2] = make_double2(cre[mt][nt][i2], cim[mt][nt][i2]);
    if (q4 == 0) {
      Bs[g * LDB + 16] = colv[0];
      Bs[(8 + g) * LDB + 16] = colv[1];
      Bs[16 * LDB + g] = rowv[0];
      Bs[16 * LDB + 8 + g] = rowv[1];
    }
    if (lane == 0) Bs[16 * LDB + 16] = cornv;

    // ---- first stage of eq.(4): every 32 rings the CTA sums its 8 tasks (fixed order)
    if ((cnt & 31) == 31 || s == 0) {
      red[t][lane] = keep;
      keep = 0.0;
      __syncthreads();
      const int first = cnt & ~31;                   // rings N-1-first-j, j = 0 .. cnt-first
      if (t == 0 && first + lane <= cnt) {
        double tot = 0.0;
#pragma unroll
        for (int w = 0; w < TPC; ++w) tot += red[w][lane];
        const int sj = N - 1 - (first + lane);
        prow_out[dir ? N - 1 - sj : sj] = tot;
      }
      __syncthreads();
    }
  }
  // ------------------------------------------------------------------ transmission (direction 0)
  if (dir == 0) {
    __syncwarp();                                    // C_0 = G_(0,N-1) F_R is in Bs
    double v = 0.0;
    for (int e = lane; e < MAT; e += 32) {           // element (a, b) of F_first^dagger C_0
      const int a = e / NB17, b = e - a * NB17;
      c64 acc = make_double2(0.0, 0.0);
      for (int c2 = 0; c2 < NB17; ++c2) cfma(acc, cconj(F_first[c2 * NB17 + a]), Bs[c2 * LDB + b]);
      v += cabs2(acc);
    }
    v = warp_sum(v);
    if (lane == 0 && active) p.T[(size_t)id.c * p.K_neq + k] = v;
  }
}

cudaError_t launch_block_back17(const SweepLaunch& p, cudaStream_t s) {
  // real-axis CTAs of this launch: global ids [max(cta_begin, n_eq_cta), cta_begin + n_cta)
  const long long first = p.cta_begin > p.n_eq_cta ? p.cta_begin : p.n_eq_cta;
  const long long n = p.cta_begin + p.n_cta - first;
  if (n <= 0) return cudaSuccess;
  block_back17_kernel<<<(unsigned)n, kBackThreads17, 0, s>>>(p, first);
  return cudaGetLastError();
}

}  // namespace blk
}  // namespace negf
