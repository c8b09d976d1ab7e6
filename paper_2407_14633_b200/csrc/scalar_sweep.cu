// Scalar (mode-space) RGF sweep kernel: steps a1s, a2, a3, a4 and the first stage of a5 of
// SURVEY.md 8(a) for block == 1 (BASELINE.json configs[0..1]).
//
// Formulation: every (channel, mode, real-axis energy) is split into two
// independent half-sweep tasks, one per direction.  A task runs the connected-Green's-function
// recursion of Algorithm 2 away from its first lead,
//     g_s = 1 / (z - U_i - |beta|^2 g_{s-1}),            (ytilde / xtilde of Alg.2 for scalars)
// stores only r_s = |g_s|^2 (8 B) per ring, then walks back with the column recursion of Algorithm 1
// steps 2-3, which for scalars needs only moduli:
//     |G_(i,k)|^2 = r_i |beta|^2 |G_(i+-1,k)|^2,         k = index of the task's last lead,
// giving Tr A_l,(i,i) = Gamma_l |G_(i,k)|^2 and, at the far end, T(E) (eq.(5)).
// Contour points need the complex diagonal G_(i,i) = [alpha_i - x_i - y_i]^-1 (Alg.1 step 1) and run
// as single tasks (right-connected pass stored as complex, left-connected pass on the fly).
// Energy reduction (eq.(4)): each warp transposes 16 rings x 32 energies through shared
// memory, sums them and writes one partial per ring; a deterministic second stage sums the warps.
#include "negf_internal.h"

namespace negf {
namespace {

constexpr int kTile = 16;           // ring steps per transposed warp reduction
constexpr int kWarpsPerBlock = 4;
constexpr double kPi = 3.14159265358979323846;

struct cplx {
  double re, im;
};

__device__ __forceinline__ cplx cmul(cplx a, cplx b) {
  return {a.re * b.re - a.im * b.im, a.re * b.im + a.im * b.re};
}
__device__ __forceinline__ cplx cadd(cplx a, cplx b) { return {a.re + b.re, a.im + b.im}; }
__device__ __forceinline__ cplx csub(cplx a, cplx b) { return {a.re - b.re, a.im - b.im}; }
__device__ __forceinline__ cplx crcp(cplx d) {
  double r = 1.0 / (d.re * d.re + d.im * d.im);
  return {d.re * r, -d.im * r};
}
__device__ __forceinline__ cplx cdiv(cplx a, cplx b) { return cmul(a, crcp(b)); }

// principal square root (branch cut on the negative real axis, +0 imaginary part maps to +i)
__device__ __forceinline__ cplx csqrt_principal(cplx z) {
  double r = sqrt(z.re * z.re + z.im * z.im);
  if (r == 0.0) return {0.0, 0.0};
  if (z.re >= 0.0) {
    double a = sqrt(0.5 * (r + z.re));
    return {a, z.im / (2.0 * a)};
  }
  double b = copysign(sqrt(0.5 * (r - z.re)), z.im);
  return {z.im / (2.0 * b), b};
}

// Retarded surface Green's function of a semi-infinite chain with bonds a, b, a, ... (a = first bond
// inside the lead), zero on-site energy: root of  z b^2 g^2 - (z^2 - a^2 + b^2) g + z = 0  with
// S = sqrt(z-(a+b)) sqrt(z-(a-b)) sqrt(z-(b-a)) sqrt(z+(a+b)),  g = 2z/(X+S) = (X-S)/(2 z b^2)
// (R8; "analytical expression ... for CNTs [23]").
__device__ cplx surface_gf_alternating(cplx z, double a, double b) {
  cplx X = cmul(z, z);
  X.re += (b - a) * (b + a);
  cplx S = cmul(cmul(csqrt_principal({z.re - (a + b), z.im}), csqrt_principal({z.re - (a - b), z.im})),
                cmul(csqrt_principal({z.re - (b - a), z.im}), csqrt_principal({z.re + (a + b), z.im})));
  if (X.re * S.re + X.im * S.im >= 0.0) {
    cplx num = {2.0 * z.re, 2.0 * z.im};
    return cdiv(num, cadd(X, S));
  }
  double bb2 = 2.0 * b * b;
  cplx den = {bb2 * z.re, bb2 * z.im};
  return cdiv(csub(X, S), den);
}

__device__ __forceinline__ double fermi(double E, double mu, double kT) {
  double x = (E - mu) / kT;
  double e = exp(-fabs(x));
  return x > 0.0 ? e / (1.0 + e) : 1.0 / (1.0 + e);
}

// Sum a [cnt <= 16 rings][32 lanes] tile over lanes and write one value per ring.
// ring index of tile row t is ring0 + sign * t.
__device__ __forceinline__ void flush_tile(double (*tile)[33], int lane, int cnt, double* prow,
                                           int ring0, int sign) {
  __syncwarp();
  int row = lane & (kTile - 1);
  int half = lane >> 4;
  double acc = 0.0;
#pragma unroll
  for (int t = 0; t < 16; ++t) acc += tile[row][half * 16 + t];
  acc += __shfl_xor_sync(0xffffffffu, acc, 16);
  if (lane < cnt) prow[ring0 + sign * row] = acc;
  __syncwarp();
}

__global__ void __launch_bounds__(kWarpsPerBlock * 32, 8)
scalar_sweep_kernel(const ScalarLaunch p) {
  __shared__ double tiles[kWarpsPerBlock][kTile][33];
  const int lane = threadIdx.x & 31;
  const int wib = threadIdx.x >> 5;
  const int w = p.warp_begin + blockIdx.x * kWarpsPerBlock + wib;   // global warp index
  if (w >= p.warp_end) return;
  double(*tile)[33] = tiles[wib];

  const int N = p.N;
  const int wpc = p.cwarps_per_channel + 2 * p.rwarps_per_channel;
  const int c = w / wpc;
  const int local = w - c * wpc;
  const double* __restrict__ U = p.U + (size_t)c * N;
  double* __restrict__ prow = p.partial + (size_t)w * N;

  // history offset of this warp inside the launch's workspace
  auto cw_before = [&](int ww) { return (ww / wpc) * p.cwarps_per_channel + min(ww % wpc, p.cwarps_per_channel); };
  const long long cwb = cw_before(w) - cw_before(p.warp_begin);
  const long long rwb = (long long)(w - p.warp_begin) - cwb;
  char* hbase = reinterpret_cast<char*>(p.hist_r) + (cwb * 16 + rwb * 8) * (long long)N * 32;

  const double U0 = __ldg(U), UN = __ldg(U + N - 1);

  if (local >= p.cwarps_per_channel) {
    // ------------------------------------------------------------------ real-axis half-sweep task
    const int rl = local - p.cwarps_per_channel;
    const int dir = rl & 1;                 // 0: left -> right (last lead = drain), 1: right -> left
    const int grp = rl >> 1;
    const int ntask = p.n_modes * p.K_neq;
    int e = grp * 32 + lane;
    const bool active = e < ntask;
    if (!active) e = ntask - 1;
    const int mode = e / p.K_neq;
    const int k = e - mode * p.K_neq;
    const cplx z = {p.z_neq[k].x, p.z_neq[k].y};
    const double be = __ldg(p.bsq_even + mode), bo = __ldg(p.bsq_odd + mode);

    // lead self-energies (a1s).  Bond (j, j+1) is even-type for even j; left lead: tau = bond(-1) (odd),
    // first interior bond(-2) (even); right lead: tau = bond(N-1), interior bond(N).
    const double tauL2 = bo, t1L2 = be;
    const double tauR2 = ((N - 1) & 1) ? bo : be, t1R2 = ((N - 1) & 1) ? be : bo;
    cplx gl = surface_gf_alternating({z.re - U0, z.im}, sqrt(t1L2), sqrt(tauL2));
    cplx gr = surface_gf_alternating({z.re - UN, z.im}, sqrt(t1R2), sqrt(tauR2));
    const cplx sigL = {tauL2 * gl.re, tauL2 * gl.im};
    const cplx sigR = {tauR2 * gr.re, tauR2 * gr.im};
    const double gamL = -2.0 * sigL.im, gamR = -2.0 * sigR.im;   // Gamma = i(Sigma - Sigma^dagger)
    const cplx sig_first = dir ? sigR : sigL;
    const cplx sig_last = dir ? sigL : sigR;
    const double f_last = dir ? fermi(z.re, p.mu_s, p.kT) : fermi(z.re, p.mu_d, p.kT);
    const double gam_last = dir ? gamL : gamR;
    const double w_last = active ? __ldg(p.mode_w + mode) * __ldg(p.w_neq + k) * (1.0 / (2.0 * kPi)) * f_last * gam_last
                                 : 0.0;

    double* __restrict__ hist = reinterpret_cast<double*>(hbase) + lane;
    // bond type (0 even, 1 odd) joining phase-1 steps s-1 and s:
    //   dir 0: bond (i-1, i), i = s      -> parity of s-1
    //   dir 1: bond (i, i+1), i = N-1-s  -> parity of N-1-s
    const int par0 = dir ? ((N - 1) & 1) : 1;    // bond type at s = 0 (unused), flips every step
    // ---- phase 1: connected Green's function away from the first lead (Alg.2)
    double gre, gim, r;
    {
      const int i0 = dir ? N - 1 : 0;
      double dre = z.re - __ldg(U + i0) - sig_first.re;
      double dim = z.im - sig_first.im;
      r = 1.0 / (dre * dre + dim * dim);
      gre = dre * r;
      gim = -dim * r;
      hist[0] = r;
    }
    const int istep = dir ? -1 : 1;
    int i = dir ? N - 2 : 1;
    int par = par0 ^ 1;
#pragma unroll 4
    for (int s = 1; s < N - 1; ++s, i += istep, par ^= 1) {
      const double b2 = par ? bo : be;
      double dre = (z.re - __ldg(U + i)) - b2 * gre;
      double dim = z.im - b2 * gim;
      r = 1.0 / (dre * dre + dim * dim);
      gre = dre * r;
      gim = -dim * r;
      hist[(size_t)s * 32] = r;
    }
    {
      const double b2 = par ? bo : be;
      double dre = (z.re - __ldg(U + i)) - b2 * gre - sig_last.re;
      double dim = z.im - b2 * gim - sig_last.im;
      r = 1.0 / (dre * dre + dim * dim);     // |G_(k,k)|^2 at the last lead's ring
      hist[(size_t)(N - 1) * 32] = r;
    }
    // ---- phase 2: column recursion back towards the first lead (Alg.1 steps 2-3, moduli only)
    // step q handles phase-1 step s = N-1-q; |G_(i,k)|^2 = r_s * |bond(s, s+1)|^2 * |G_(i',k)|^2.
    const int ring0 = dir ? 0 : N - 1;
    const int sign = dir ? 1 : -1;
    double c2 = 1.0;
    // bond between steps s and s+1 has the type computed for step s+1: par(s+1) = par0 ^ ((s+1)&1)
    for (int q0 = 0; q0 < N; q0 += kTile) {
      const int cnt = min(kTile, N - q0);
      double h[kTile];
#pragma unroll
      for (int t = 0; t < kTile; ++t) {
        const int s = N - 1 - (q0 + t);
        h[t] = (t < cnt) ? hist[(size_t)s * 32] : 0.0;
      }
#pragma unroll
      for (int t = 0; t < kTile; ++t) {
        const int q = q0 + t;
        const int s = N - 1 - q;
        const int pt = par0 ^ ((s + 1) & 1);
        const double b2 = (q == 0) ? 1.0 : (pt ? bo : be);
        c2 *= h[t] * b2;
        tile[t][lane] = (t < cnt) ? w_last * c2 : 0.0;
        if (t == cnt - 1 && q == N - 1 && dir == 0 && active) {
          // G_(0,N-1): transmission (eq.(5)), a4
          p.T_part[((size_t)c * p.n_modes + mode) * p.K_neq + k] = __ldg(p.mode_w_T + mode) * gamL * gamR * c2;
        }
      }
      flush_tile(tile, lane, cnt, prow, ring0 + sign * q0, sign);
    }
  } else {
    // ------------------------------------------------------------------ contour task
    const int ntask = p.n_modes * p.K_eq;
    int e = local * 32 + lane;
    const bool active = e < ntask;
    if (!active) e = ntask - 1;
    const int mode = e / p.K_eq;
    const int k = e - mode * p.K_eq;
    const cplx z = {p.z_eq[k].x, p.z_eq[k].y};
    const cplx W = {p.w_eq[k].x, p.w_eq[k].y};
    const double be = __ldg(p.bsq_even + mode), bo = __ldg(p.bsq_odd + mode);
    const double tauL2 = bo, t1L2 = be;
    const double tauR2 = ((N - 1) & 1) ? bo : be, t1R2 = ((N - 1) & 1) ? be : bo;
    cplx gl = surface_gf_alternating({z.re - U0, z.im}, sqrt(t1L2), sqrt(tauL2));
    cplx gr = surface_gf_alternating({z.re - UN, z.im}, sqrt(t1R2), sqrt(tauR2));
    const cplx sigL = {tauL2 * gl.re, tauL2 * gl.im};
    const cplx sigR = {tauR2 * gr.re, tauR2 * gr.im};
    const double wc = active ? -__ldg(p.mode_w + mode) / kPi : 0.0;   // deg * mode_weight * (-1/pi)

    double2* __restrict__ hist = reinterpret_cast<double2*>(hbase) + lane;
    // pass 1: x_i = |beta_i|^2 gR_{i+1} for i = N-2..0 (right-connected, Alg.2 xtilde); store x_i
    cplx x = sigR;                                   // plays the role of x_{N-1} (lead instead of a ring)
    for (int i = N - 1; i >= 1; --i) {
      cplx d = {z.re - __ldg(U + i) - x.re, z.im - x.im};
      cplx g = crcp(d);
      const double b2 = ((i - 1) & 1) ? bo : be;     // bond (i-1, i)
      x = {b2 * g.re, b2 * g.im};
      hist[(size_t)(i - 1) * 32] = make_double2(x.re, x.im);
    }
    // pass 2: y_i on the fly (left-connected), G_ii = 1/(alpha_i - x_i - y_i)  (Alg.1 step 1)
    cplx y = sigL;
    for (int q0 = 0; q0 < N; q0 += kTile) {
      const int cnt = min(kTile, N - q0);
#pragma unroll 4
      for (int t = 0; t < kTile; ++t) {
        const int i = q0 + t;
        double v = 0.0;
        if (t < cnt) {
          cplx xi;
          if (i < N - 1) {
            double2 hx = hist[(size_t)i * 32];
            xi = {hx.x, hx.y};
          } else {
            xi = sigR;
          }
          const double u = __ldg(U + i);
          cplx dl = {z.re - u - y.re, z.im - y.im};            // alpha_i - y_i
          cplx G = crcp({dl.re - xi.re, dl.im - xi.im});        // G_ii
          v = wc * (W.re * G.im + W.im * G.re);                 // -(deg/pi) Im(W G)
          cplx gL = crcp(dl);
          const double b2 = (i & 1) ? bo : be;                  // bond (i, i+1)
          y = {b2 * gL.re, b2 * gL.im};
        }
        tile[t][lane] = v;
      }
      flush_tile(tile, lane, cnt, prow, q0, 1);
    }
  }
}

}  // namespace

cudaError_t launch_scalar_sweep(const ScalarLaunch& p, cudaStream_t s) {
  const int nwarps = p.warp_end - p.warp_begin;
  if (nwarps <= 0) return cudaSuccess;
  const int blocks = (nwarps + kWarpsPerBlock - 1) / kWarpsPerBlock;
  scalar_sweep_kernel<<<blocks, kWarpsPerBlock * 32, 0, s>>>(p);
  return cudaGetLastError();
}

}  // namespace negf
