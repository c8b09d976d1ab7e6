// Scalar (mode-space) RGF sweep kernel: steps a1s, a2, a3, a4 and the first stage of a5 of
// SURVEY.md 8(a) for block == 1 (BASELINE.json configs[0..1]).
//
// Formulation: every (channel, mode, real-axis energy) is split into two
// independent half-sweep tasks, one per direction.  A task runs the connected-Green's-function
// recursion of Algorithm 2 away from its first lead,
//     g_s = 1 / (z - U_i - |beta|^2 g_{s-1}),            (ytilde / xtilde of Alg.2 for scalars)
// in homogeneous coordinates g_s = P_s / P_{s+1} (a three-term recurrence, no division on the
// dependent chain), stores only h_s = |P_s|^2 (8 B) per ring, then walks
// back with the column recursion of Algorithm 1 steps 2-3, which for scalars
// needs only moduli and telescopes:
//     |G_(i,k)|^2 = |g_i|^2 |beta|^2 |G_(i+-1,k)|^2 = h_i (prod |beta|^2) / |D|^2,   k = last lead,
// giving Tr A_l,(i,i) = Gamma_l |G_(i,k)|^2 and, at the far end, T(E) (eq.(5)).
// Contour points need the complex diagonal G_(i,i) = [alpha_i - x_i - y_i]^-1 (Alg.1 step 1) and run
// as single tasks (right-connected pass stored as complex, left-connected pass on the fly).
// Energy reduction (eq.(4)): each warp transposes 16 rings x 32 energies through shared
// memory, sums them and writes one partial per ring; a deterministic second stage sums the warps.
#include <algorithm>

#include "negf_internal.h"

namespace negf {
namespace {

constexpr int kTile = 16;           // ring steps per transposed warp reduction
constexpr int kWarpsPerBlock = 2;
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

// The way back met a step that the forward recursion rescaled (stored -h): undo the power of two.
__device__ __noinline__ double cross_marker(double c2, double h) {
  return c2 * ((fabs(h) >= 1.0) ? 0x1p-400 : 0x1p400);
}

__global__ void __launch_bounds__(kWarpsPerBlock * 32, 16)
scalar_real_kernel(const ScalarLaunch p, const int n_warps) {
  __shared__ double tiles[kWarpsPerBlock][kTile][33];
  const int lane = threadIdx.x & 31;
  const int wib = threadIdx.x >> 5;
  const int ord = blockIdx.x * kWarpsPerBlock + wib;      // ordinal among this launch's real-axis warps
  if (ord >= n_warps) return;
  double(*tile)[33] = tiles[wib];

  const int N = p.N;
  const int wpc = p.cwarps_per_channel + 2 * p.rwarps_per_channel;
  auto cw_before = [&](int ww) { return (ww / wpc) * p.cwarps_per_channel + min(ww % wpc, p.cwarps_per_channel); };
  const int cw0 = cw_before(p.warp_begin);
  const int g = (p.warp_begin - cw0) + ord;               // global real-axis warp ordinal
  const int c = g / (2 * p.rwarps_per_channel);
  const int local = p.cwarps_per_channel + (g - c * 2 * p.rwarps_per_channel);
  const int w = c * wpc + local;                          // global warp index
  const double* __restrict__ U = p.U + (size_t)c * N;
  double* __restrict__ prow = p.partial + (size_t)w * N;
  // history offset of this warp inside the launch's workspace
  const long long cwb = cw_before(w) - cw0;
  const long long rwb = (long long)(w - p.warp_begin) - cwb;
  char* hbase = reinterpret_cast<char*>(p.hist_r) + (cwb * 16 + rwb * 8) * (long long)N * 32;
  const double U0 = __ldg(U), UN = __ldg(U + N - 1);
  {
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
    // Bond type (0 even, 1 odd) joining steps s-1 and s of this direction:
    //   dir 0: bond (i-1, i), i = s      -> parity of s-1
    //   dir 1: bond (i, i+1), i = N-1-s  -> parity of N-1-s
    // i.e. type(s) = par0 ^ (s & 1) with par0 the (virtual) type at s = 0.
    const int par0 = dir ? ((N - 1) & 1) : 1;
    const double b2_odd_s = par0 ? be : bo;      // |bond|^2 entering odd steps s
    const double b2_even_s = par0 ? bo : be;     // |bond|^2 entering even steps s >= 2
    const int istep = dir ? -1 : 1;
    const int i0 = dir ? N - 1 : 0;

    // ---- phase 1: left-connected recursion of Alg.2 in homogeneous (division-free) form.
    // With g_s = P_s / P_{s+1} the recursion g_s = 1/(alpha_s - b2_s g_{s-1}) becomes
    //     P_{s+1} = alpha_s P_s - b2_s P_{s-1},   P_0 = 1,  P_1 = alpha_0 - Sigma_first,
    // and the product of |ytilde|^2 that Alg.1 steps 2-3 need telescopes:
    //     prod_{s=i}^{N-2} b2_{s+1} |g_s|^2 = (prod b2) |P_i|^2 / |P_{N-1}|^2.
    // Only h_s = |P_s|^2 is stored (8 B per ring).  |P| is kept in range by exact power-of-two
    // rescaling, checked every 4 steps; a rescaled step stores -h_s as the marker the way back reads.
    double pr = 1.0, pi_ = 0.0, qr = 0.0, qi = 0.0;       // P_s, P_{s-1}
    hist[0] = 1.0;
    {
      const double ar = z.re - __ldg(U + i0) - sig_first.re;
      const double ai = z.im - sig_first.im;
      qr = pr; qi = pi_;
      pr = ar; pi_ = ai;                                   // P_1 = alpha_0 * 1
    }
    int i = i0 + istep;
    double m = fma(pr, pr, pi_ * pi_);                     // |P_1|^2
    int s = 1;
    // Invariant at the top of a step: (pr,pi_) = P_s, (qr,qi) = P_{s-1}, m = |P_s|^2 (negative if
    // P_s was just rescaled), i = ring of step s.  A step stores h_s and produces P_{s+1}.
#define NEGF_STEP(B2)                                                      \
    {                                                                      \
      hist[(size_t)s * 32] = m;                                            \
      const double ar = z.re - __ldg(U + i);                               \
      const double nr = fma(ar, pr, fma(-z.im, pi_, -(B2) * qr));          \
      const double ni = fma(ar, pi_, fma(z.im, pr, -(B2) * qi));           \
      qr = pr; qi = pi_; pr = nr; pi_ = ni;                                \
      m = fma(pr, pr, pi_ * pi_);                                          \
      i += istep; ++s;                                                     \
    }
#define NEGF_RANGE()                                                       \
    {                                                                      \
      const unsigned ex = (unsigned)(__double2hiint(m) >> 20) - 623u;      \
      if (ex > 800u && m > 0.0) {                                          \
        const bool big = ex < 0x80000000u;                                 \
        const double sc = big ? 0x1p-200 : 0x1p200;                        \
        pr *= sc; pi_ *= sc; qr *= sc; qi *= sc;                           \
        m = -(m * (big ? 0x1p-400 : 0x1p400));                             \
      }                                                                    \
    }
    // steps s = 1 .. N-2 produce P_2 .. P_{N-1}; step s uses the bond entering step s.
    while (s + 3 < N - 1) {                                // s is odd at the top
      NEGF_STEP(b2_odd_s)
      NEGF_STEP(b2_even_s)
      NEGF_STEP(b2_odd_s)
      NEGF_STEP(b2_even_s)
      NEGF_RANGE()
    }
    while (s < N - 1) {
      const double b2 = (s & 1) ? b2_odd_s : b2_even_s;
      NEGF_STEP(b2)
      NEGF_RANGE()
    }
#undef NEGF_STEP
#undef NEGF_RANGE
    // here s == N-1 (or N == 2: s == 1 == N-1): (pr,pi_) = P_{N-1}, m = +-|P_{N-1}|^2
    hist[(size_t)(N - 1) * 32] = m;
    double c2;
    {
      const double b2 = ((N - 1) & 1) ? b2_odd_s : b2_even_s;
      const double ar = z.re - __ldg(U + i) - sig_last.re;
      const double ai = z.im - sig_last.im;
      // D = (alpha_{N-1} - Sigma_last) P_{N-1} - b2 P_{N-2};  G_(k,k) = P_{N-1} / D
      const double dr = fma(ar, pr, fma(-ai, pi_, -b2 * qr));
      const double di = fma(ar, pi_, fma(ai, pr, -b2 * qi));
      c2 = 1.0 / fma(dr, dr, di * di);
    }
    // ---- phase 2: column recursion back towards the first lead (Alg.1 steps 2-3, moduli only):
    // |G_(i,k)|^2 = F_s h_s with F_{N-1} = 1/|D|^2, F_{s-1} = F_s * b2_s (* 2^-+400 across a marker).
    const int ring0 = dir ? 0 : N - 1;
    const int sign = dir ? 1 : -1;
    // bond entering step ss = N-1-(q0+t): kTile is even, so its type depends on the parity of t only
    const double b2_t_even = ((N - 1) & 1) ? b2_odd_s : b2_even_s;
    const double b2_t_odd = ((N - 1) & 1) ? b2_even_s : b2_odd_s;
    const double* __restrict__ hrd = hist + (size_t)(N - 1) * 32;   // walks down the history
    double g2 = 0.0;
    int q0 = 0;
    // probe: way-back position of the ring whose per-energy contributions are recorded
    const int probe_pos = (p.probe_ring >= 0 && p.probe) ? sign * (p.probe_ring - ring0) : -1;
    double* __restrict__ probe_out =
        p.probe ? p.probe + (((size_t)c * 2 + dir) * p.n_modes + mode) * p.K_neq + k : nullptr;
    for (; q0 + kTile <= N; q0 += kTile, hrd -= (size_t)kTile * 32) {   // full tiles: no tail tests
      double h[kTile];
#pragma unroll
      for (int t = 0; t < kTile; ++t) h[t] = *(hrd - (size_t)t * 32);
#pragma unroll
      for (int t = 0; t < kTile; ++t) {
        g2 = c2 * fabs(h[t]);                              // |G_(i,k)|^2
        tile[t][lane] = w_last * g2;
        if (__double2hiint(h[t]) < 0) c2 = cross_marker(c2, h[t]);   // rare: a rescaled step
        c2 *= (t & 1) ? b2_t_odd : b2_t_even;
      }
      if ((unsigned)(probe_pos - q0) < (unsigned)kTile && active) *probe_out = tile[probe_pos - q0][lane];
      flush_tile(tile, lane, kTile, prow, ring0 + sign * q0, sign);
    }
    if (q0 < N) {                                          // ragged last tile
      const int cnt = N - q0;
#pragma unroll 1
      for (int t = 0; t < kTile; ++t) {
        double v = 0.0;
        if (t < cnt) {
          const double hv = *(hrd - (size_t)t * 32);
          g2 = c2 * fabs(hv);
          v = w_last * g2;
          if (hv < 0.0) c2 = cross_marker(c2, hv);
          c2 *= (t & 1) ? b2_t_odd : b2_t_even;
        }
        tile[t][lane] = v;
      }
      if ((unsigned)(probe_pos - q0) < (unsigned)cnt && active) *probe_out = tile[probe_pos - q0][lane];
      flush_tile(tile, lane, cnt, prow, ring0 + sign * q0, sign);
    }
    // the last value is |G_(first,last)|^2: transmission through the chain (eq.(5)), a4
    if (dir == 0 && active)
      p.T_part[((size_t)c * p.n_modes + mode) * p.K_neq + k] = __ldg(p.mode_w_T + mode) * gamL * gamR * g2;
  }
}

// ---------------------------------------------------------------------------------- contour tasks
// One contour half-sweep task = (channel, mode, contour point, direction); a warp holds 32 of them.
// Direction 0 stores y_i (left-connected), direction 1 stores x_i (right-connected), both indexed by
// ring; scalar_combine_kernel then forms G_(i,i) (Alg.1 step 1).
struct ContourTask {
  int N, dir, istep, i0;
  cplx z, sig_first;
  double b2_odd_s, b2_even_s;       // |bond|^2 entering odd / even steps s
  const double* U;                  // on-site energies of the task's channel
  double2* hist;                    // [ring][32 lanes], already offset by the lane
};

__device__ __forceinline__ ContourTask contour_task(const ScalarLaunch& p, int ord, int lane) {
  ContourTask t;
  const int N = p.N;
  const int wpc = p.cwarps_per_channel + 2 * p.rwarps_per_channel;
  auto cw_before = [&](int ww) { return (ww / wpc) * p.cwarps_per_channel + min(ww % wpc, p.cwarps_per_channel); };
  const int cw0 = cw_before(p.warp_begin);
  const int g = cw0 + ord;                                // global contour warp ordinal
  const int c = g / p.cwarps_per_channel;
  const int local = g - c * p.cwarps_per_channel;         // = 2 * group + direction
  const int w = c * wpc + local;                          // global warp index
  t.N = N;
  t.U = p.U + (size_t)c * N;
  // history offset of this warp inside the launch's workspace
  const long long cwb = cw_before(w) - cw0;
  const long long rwb = (long long)(w - p.warp_begin) - cwb;
  char* hbase = reinterpret_cast<char*>(p.hist_r) + (cwb * 16 + rwb * 8) * (long long)N * 32;
  t.hist = reinterpret_cast<double2*>(hbase) + lane;
  t.dir = local & 1;
  const int grp = local >> 1;
  const int ntask = p.n_modes * p.K_eq;
  int e = grp * 32 + lane;
  if (e >= ntask) e = ntask - 1;
  const int mode = e / p.K_eq;
  const int k = e - mode * p.K_eq;
  t.z = {p.z_eq[k].x, p.z_eq[k].y};
  const double be = __ldg(p.bsq_even + mode), bo = __ldg(p.bsq_odd + mode);
  if (t.dir == 0) {
    const cplx gl = surface_gf_alternating({t.z.re - __ldg(t.U), t.z.im}, sqrt(be), sqrt(bo));
    t.sig_first = {bo * gl.re, bo * gl.im};
  } else {
    const double tauR2 = ((N - 1) & 1) ? bo : be, t1R2 = ((N - 1) & 1) ? be : bo;
    const cplx gr = surface_gf_alternating({t.z.re - __ldg(t.U + N - 1), t.z.im}, sqrt(t1R2), sqrt(tauR2));
    t.sig_first = {tauR2 * gr.re, tauR2 * gr.im};
  }
  const int par0 = t.dir ? ((N - 1) & 1) : 1;       // bond type entering step s is par0 ^ (s & 1)
  t.b2_odd_s = par0 ? be : bo;
  t.b2_even_s = par0 ? bo : be;
  t.istep = t.dir ? -1 : 1;
  t.i0 = t.dir ? N - 1 : 0;
  return t;
}

// Steps s = s0 .. s1-1 of the homogeneous form of Alg.2 (see scalar_real_kernel): on entry (pr, pi_) = P_s0,
// (qr, qi) = P_{s0-1}; every step stores y_s = b2_s g_{s-1} = b2_s P_{s-1} / P_s (x_i for direction 1) at its
// ring -- formed off the dependent chain and invariant under the power-of-two rescaling -- and advances
// P_{s+1} = alpha_s P_s - b2_s P_{s-1}.
__device__ __forceinline__ void contour_steps(const ContourTask& t, int s0, int s1, double& pr, double& pi_,
                                              double& qr, double& qi) {
  int i = t.i0 + t.istep * s0;
  for (int s = s0; s < s1; ++s, i += t.istep) {
    const double b2 = (s & 1) ? t.b2_odd_s : t.b2_even_s;
    // y_s = b2 P_{s-1} conj(P_s) / |P_s|^2
    const double m = fma(pr, pr, pi_ * pi_);
    const double r = b2 / m;
    const double tr = fma(qr, pr, qi * pi_), ti = fma(qi, pr, -qr * pi_);
    t.hist[(size_t)i * 32] = make_double2(tr * r, ti * r);
    const double ar = t.z.re - __ldg(t.U + i);
    double nr = fma(ar, pr, fma(-t.z.im, pi_, -b2 * qr));
    double ni = fma(ar, pi_, fma(t.z.im, pr, -b2 * qi));
    qr = pr; qi = pi_; pr = nr; pi_ = ni;
    if ((s & 3) == 0) {
      const unsigned ex = (unsigned)(__double2hiint(m) >> 20) - 623u;
      if (ex > 800u && m > 0.0) {
        const double sc = (ex < 0x80000000u) ? 0x1p-200 : 0x1p200;
        pr *= sc; pi_ *= sc; qr *= sc; qi *= sc;
      }
    }
  }
}

__global__ void __launch_bounds__(kWarpsPerBlock * 32, 8)
scalar_contour_kernel(const ScalarLaunch p, const int n_warps) {
  const int lane = threadIdx.x & 31;
  const int ord = blockIdx.x * kWarpsPerBlock + (threadIdx.x >> 5);   // ordinal among this launch's contour warps
  if (ord >= n_warps) return;
  const ContourTask t = contour_task(p, ord, lane);
  t.hist[(size_t)t.i0 * 32] = make_double2(t.sig_first.re, t.sig_first.im);   // the lead plays ring "-1"
  double qr = 1.0, qi = 0.0;                                                   // P_0
  double pr = t.z.re - __ldg(t.U + t.i0) - t.sig_first.re, pi_ = t.z.im - t.sig_first.im;   // P_1
  contour_steps(t, 1, t.N, pr, pi_, qr, qi);
}

// ---------------------------------------------------------------------------------- parallel in N
// Long channels with few contour points (the shape of the paper's Table 2: N = 524 288 rings, 90 points,
// PAPER.md:325-335) leave the serial pass above with a few dozen warps.  The recursion is
// linear in (P_s, P_{s-1}),  [P_{s+1}; P_s] = T_s [P_s; P_{s-1}],  T_s = [[alpha_s, -b2_s], [1, 0]],  so the
// steps 1 .. N-1 are cut into S segments of L steps and done in three passes:
//   A  (parallel over tasks x segments)  M_m = product of the segment's T_s, as the images of the two unit
//      vectors, with one common power-of-two rescaling (only ratios of P are ever used);
//   B  (parallel over tasks, serial over the S segments)  the state at every segment start, v_{m+1} = M_m v_m;
//   C  (parallel over tasks x segments)  the very steps of the serial kernel from the segment's start state.
// Pass C computes every stored y_s by the same recurrence as the serial kernel; the segment start states
// differ from the serial ones only by the rounding of the 2 x 2 products.  For Im z > 0 the forward recursion
// is dominated by its growing solution, so M_m v_m has no cancellation.  (This is NOT the transfer-matrix
// scan of |G| on the real axis that SURVEY 7 warns about: only the contour tasks use it.)
__device__ __forceinline__ void seg_range(const ScalarLaunch& p, int m, int& s0, int& s1) {
  s0 = 1 + m * p.seg_L;
  s1 = min(s0 + p.seg_L, p.N);
}

__global__ void __launch_bounds__(128, 8) scalar_contour_segA_kernel(const ScalarLaunch p, const int n_warps) {
  const int lane = threadIdx.x & 31;
  const long long job = (long long)blockIdx.x * 4 + (threadIdx.x >> 5);
  const int ord = (int)(job / p.seg_S), m = (int)(job - (long long)ord * p.seg_S);
  if (ord >= n_warps) return;
  const ContourTask t = contour_task(p, ord, lane);
  int s0, s1;
  seg_range(p, m, s0, s1);
  // columns of M_m: start states (P_s0, P_{s0-1}) = (1, 0) and (0, 1)
  double ar_ = 1.0, ai_ = 0.0, br_ = 0.0, bi_ = 0.0;      // first column: P_s, P_{s-1}
  double cr_ = 0.0, ci_ = 0.0, dr_ = 1.0, di_ = 0.0;      // second column
  int i = t.i0 + t.istep * s0;
  for (int s = s0; s < s1; ++s, i += t.istep) {
    const double b2 = (s & 1) ? t.b2_odd_s : t.b2_even_s;
    const double al = t.z.re - __ldg(t.U + i);
    const double n1r = fma(al, ar_, fma(-t.z.im, ai_, -b2 * br_)), n1i = fma(al, ai_, fma(t.z.im, ar_, -b2 * bi_));
    const double n2r = fma(al, cr_, fma(-t.z.im, ci_, -b2 * dr_)), n2i = fma(al, ci_, fma(t.z.im, cr_, -b2 * di_));
    br_ = ar_; bi_ = ai_; ar_ = n1r; ai_ = n1i;
    dr_ = cr_; di_ = ci_; cr_ = n2r; ci_ = n2i;
    if ((s & 3) == 0) {
      const double mm = fmax(fma(ar_, ar_, ai_ * ai_), fma(cr_, cr_, ci_ * ci_));
      const unsigned ex = (unsigned)(__double2hiint(mm) >> 20) - 623u;
      if (ex > 800u && mm > 0.0) {
        const double sc = (ex < 0x80000000u) ? 0x1p-200 : 0x1p200;
        ar_ *= sc; ai_ *= sc; br_ *= sc; bi_ *= sc; cr_ *= sc; ci_ *= sc; dr_ *= sc; di_ *= sc;
      }
    }
  }
  double2* M = p.seg_M + ((size_t)job * 4) * 32 + lane;      // [job][component][lane]
  M[0] = make_double2(ar_, ai_);     // M11: P_s1   from (1, 0)
  M[32] = make_double2(cr_, ci_);    // M12: P_s1   from (0, 1)
  M[64] = make_double2(br_, bi_);    // M21: P_s1-1 from (1, 0)
  M[96] = make_double2(dr_, di_);    // M22
}

__global__ void __launch_bounds__(kWarpsPerBlock * 32, 8)
scalar_contour_segB_kernel(const ScalarLaunch p, const int n_warps) {
  const int lane = threadIdx.x & 31;
  const int ord = blockIdx.x * kWarpsPerBlock + (threadIdx.x >> 5);
  if (ord >= n_warps) return;
  const ContourTask t = contour_task(p, ord, lane);
  double qr = 1.0, qi = 0.0;                                                   // P_0
  double pr = t.z.re - __ldg(t.U + t.i0) - t.sig_first.re, pi_ = t.z.im - t.sig_first.im;   // P_1
  const double2* M = p.seg_M + ((size_t)ord * p.seg_S * 4) * 32 + lane;
  double2* v = p.seg_v + ((size_t)ord * p.seg_S * 2) * 32 + lane;
  for (int m = 0; m < p.seg_S; ++m, M += 4 * 32, v += 2 * 32) {
    v[0] = make_double2(pr, pi_);                 // state at the start of segment m: P_s0, P_{s0-1}
    v[32] = make_double2(qr, qi);
    const double2 m11 = M[0], m12 = M[32], m21 = M[64], m22 = M[96];
    const double nr = fma(m11.x, pr, fma(-m11.y, pi_, fma(m12.x, qr, -m12.y * qi)));
    const double ni = fma(m11.x, pi_, fma(m11.y, pr, fma(m12.x, qi, m12.y * qr)));
    const double or_ = fma(m21.x, pr, fma(-m21.y, pi_, fma(m22.x, qr, -m22.y * qi)));
    const double oi = fma(m21.x, pi_, fma(m21.y, pr, fma(m22.x, qi, m22.y * qr)));
    pr = nr; pi_ = ni; qr = or_; qi = oi;
    const double mm = fma(pr, pr, pi_ * pi_);
    const unsigned ex = (unsigned)(__double2hiint(mm) >> 20) - 623u;
    if (ex > 800u && mm > 0.0) {
      const double sc = (ex < 0x80000000u) ? 0x1p-200 : 0x1p200;
      pr *= sc; pi_ *= sc; qr *= sc; qi *= sc;
    }
  }
}

__global__ void __launch_bounds__(128, 8) scalar_contour_segC_kernel(const ScalarLaunch p, const int n_warps) {
  const int lane = threadIdx.x & 31;
  const long long job = (long long)blockIdx.x * 4 + (threadIdx.x >> 5);
  const int ord = (int)(job / p.seg_S), m = (int)(job - (long long)ord * p.seg_S);
  if (ord >= n_warps) return;
  const ContourTask t = contour_task(p, ord, lane);
  int s0, s1;
  seg_range(p, m, s0, s1);
  if (m == 0) t.hist[(size_t)t.i0 * 32] = make_double2(t.sig_first.re, t.sig_first.im);   // the lead plays ring "-1"
  const double2* v = p.seg_v + ((size_t)job * 2) * 32 + lane;
  const double2 P = v[0], Q = v[32];
  double pr = P.x, pi_ = P.y, qr = Q.x, qi = Q.y;
  contour_steps(t, s0, s1, pr, pi_, qr, qi);
}

// Contour combine: G_(i,i) = 1 / (alpha_i - x_i - y_i) (Alg.1 step 1) and the first term
// of eq.(4): -(deg/pi) Im[W_k G_(i,i)], summed over the 32 (mode, energy) tasks of a warp pair.
// grid = (ring chunks of 32 * kWarpsPerBlock... see launcher, pairs); one warp per (pair, 32 rings).
__global__ void __launch_bounds__(128)
scalar_combine_kernel(const ScalarLaunch p, const int pair0) {
  __shared__ double tiles[4][32][33];
  const int lane = threadIdx.x & 31;
  const int wib = threadIdx.x >> 5;
  const int pair = pair0 + blockIdx.y;
  const int N = p.N;
  const int i0 = (blockIdx.x * 4 + wib) * 32;
  if (i0 >= N) return;
  const int wpc = p.cwarps_per_channel + 2 * p.rwarps_per_channel;
  auto cw_before = [&](int ww) { return (ww / wpc) * p.cwarps_per_channel + min(ww % wpc, p.cwarps_per_channel); };
  const int cw0 = cw_before(p.warp_begin);
  const int g = cw0 + 2 * pair;                            // global contour warp ordinal of direction 0
  const int c = g / p.cwarps_per_channel;
  const int local = g - c * p.cwarps_per_channel;
  const int w = c * wpc + local;
  const double* __restrict__ U = p.U + (size_t)c * N;
  const long long cwb = cw_before(w) - cw0;
  const long long rwb = (long long)(w - p.warp_begin) - cwb;
  const char* hbase = reinterpret_cast<const char*>(p.hist_r) + (cwb * 16 + rwb * 8) * (long long)N * 32;
  const double2* __restrict__ hy = reinterpret_cast<const double2*>(hbase) + lane;
  const double2* __restrict__ hx = hy + (size_t)N * 32;   // the direction-1 warp follows directly

  const int ntask = p.n_modes * p.K_eq;
  int e = (local >> 1) * 32 + lane;
  const bool active = e < ntask;
  if (!active) e = ntask - 1;
  const int mode = e / p.K_eq;
  const int k = e - mode * p.K_eq;
  const cplx z = {p.z_eq[k].x, p.z_eq[k].y};
  const cplx W = {p.w_eq[k].x, p.w_eq[k].y};
  const double wc = active ? -__ldg(p.mode_w + mode) / kPi : 0.0;   // deg * mode_weight * (-1/pi)
  double(*tile)[33] = tiles[wib];
  const int cnt = min(32, N - i0);
  for (int t = 0; t < cnt; ++t) {
    const int i = i0 + t;
    const double2 y = hy[(size_t)i * 32], x = hx[(size_t)i * 32];
    const cplx G = crcp({z.re - __ldg(U + i) - x.x - y.x, z.im - x.y - y.y});
    tile[t][lane] = wc * (W.re * G.im + W.im * G.re);
  }
  __syncwarp();
  double acc = 0.0;
  if (lane < cnt) {
#pragma unroll
    for (int j = 0; j < 32; ++j) acc += tile[lane][j];
    p.partial[(size_t)w * N + i0 + lane] = acc;
    p.partial[(size_t)(w + 1) * N + i0 + lane] = 0.0;      // the direction-1 warp's row carries nothing
  }
}

}  // namespace

cudaError_t launch_scalar_sweep(const ScalarLaunch& p, cudaStream_t s) {
  const int nwarps = p.warp_end - p.warp_begin;
  if (nwarps <= 0) return cudaSuccess;
  const int wpc = p.cwarps_per_channel + 2 * p.rwarps_per_channel;
  auto cw_before = [&](int ww) {
    const int r = ww % wpc;
    return (ww / wpc) * p.cwarps_per_channel + (r < p.cwarps_per_channel ? r : p.cwarps_per_channel);
  };
  const int n_c = cw_before(p.warp_end) - cw_before(p.warp_begin);
  const int n_r = nwarps - n_c;
  // The few contour warps are latency-bound (a dependent pass over N rings); they start first on the
  // side stream, their combine kernel follows them there, and the real-axis kernel fills the rest of
  // the machine beside both.
  cudaError_t e;
  if (n_c > 0) {
    if (n_c & 1) return cudaErrorInvalidValue;             // batches never split a contour pair
    if ((e = cudaEventRecord(p.ev_fork, s)) != cudaSuccess) return e;
    if ((e = cudaStreamWaitEvent(p.side, p.ev_fork, 0)) != cudaSuccess) return e;
    if (p.seg_M) {                                          // parallel in N (long channels)
      const long long jobs = (long long)n_c * p.seg_S;
      const unsigned blocks = (unsigned)((jobs + 3) / 4);
      scalar_contour_segA_kernel<<<blocks, 128, 0, p.side>>>(p, n_c);
      scalar_contour_segB_kernel<<<(n_c + kWarpsPerBlock - 1) / kWarpsPerBlock, kWarpsPerBlock * 32, 0, p.side>>>(p, n_c);
      scalar_contour_segC_kernel<<<blocks, 128, 0, p.side>>>(p, n_c);
    } else {
      scalar_contour_kernel<<<(n_c + kWarpsPerBlock - 1) / kWarpsPerBlock, kWarpsPerBlock * 32, 0, p.side>>>(p, n_c);
    }
    if ((e = cudaGetLastError()) != cudaSuccess) return e;
    for (int pair0 = 0; pair0 < n_c / 2; pair0 += 65535) {   // grid.y is limited to 65535
      dim3 grid((p.N + 127) / 128, std::min(65535, n_c / 2 - pair0));
      scalar_combine_kernel<<<grid, 128, 0, p.side>>>(p, pair0);
      if ((e = cudaGetLastError()) != cudaSuccess) return e;
    }
    if ((e = cudaEventRecord(p.ev_join, p.side)) != cudaSuccess) return e;
  }
  if (n_r > 0) {
    scalar_real_kernel<<<(n_r + kWarpsPerBlock - 1) / kWarpsPerBlock, kWarpsPerBlock * 32, 0, s>>>(p, n_r);
    if ((e = cudaGetLastError()) != cudaSuccess) return e;
  }
  if (n_c > 0 && (e = cudaStreamWaitEvent(s, p.ev_join, 0)) != cudaSuccess) return e;
  return cudaSuccess;
}

}  // namespace negf
