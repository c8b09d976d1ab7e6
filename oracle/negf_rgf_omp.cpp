// Tier O3 oracle in plain C++17 + OpenMP: the paper's block-tridiagonal recursion
// (Algorithm 2 + Algorithm 1), one energy point per thread.
//
// TEST INFRASTRUCTURE ONLY (see oracle/__init__.py): only tests/, __graft_entry__.smoke() and the
// cpu_baseline / --impl reference legs of bench.py may build, load or call this file.  It shares no
// source, header, table or helper with paper_2407_14633_b200/csrc/ and is never linked into
// libnegf_b200.so.  It restates oracle/negf_rgf.py + oracle/selfenergy.py (numpy) so that full-size
// devices (2 112 ... 66 560 energy points of 1000-4000 rings with 17 x 17 blocks) have a CPU result
// in minutes instead of hours; it must itself match the dense definition (oracle/negf_dense.py) on
// shrunk devices and the numpy tier at full N (tests/test_oracle_rgf.py).
//
// What it computes, per channel / chain (notation of PAPER.md:82, :172; readings R1, R2, R6-R10, R12
// of DESIGN.md):
//   alpha_j = z - U_j - [j=0] Sigma_L - [j=N-1] Sigma_R,  beta_j = -H_{j,j+1},  gamma_j = -H_{j,j+1}^dagger
//   H_{j,j+1} = coup_even for even j, coup_odd for odd j.
//   Algorithm 2 (beta/gamma placed for non-commuting blocks, R1):
//     y_0 = x_{N-1} = 0
//     ytilde_n = [alpha_{n-1} - y_{n-1}]^-1 beta_{n-1},  y_n = gamma_{n-1} ytilde_n      n = 1..N-1
//     xtilde_n = [alpha_{n+1} - x_{n+1}]^-1 gamma_n,     x_n = beta_n xtilde_n           n = N-2..0
//   Algorithm 1 (steps 1-4 restored, R2):
//     1.   G_(T,T)   = [alpha_T - x_T - y_T]^-1
//     2.   G_(n+1,T) = -xtilde_n G_(n,T)   (n >= T)        3.  G_(n-1,T) = -ytilde_n G_(n,T)   (n <= T)
//     6-8. A_l,(T,T) = G_(T,k) Gamma_l G_(T,k)^dagger, G_(T,k) from steps 2/3 started at the lead block k
//   Gamma_l = i (Sigma_l - Sigma_l^dagger);  T(E) = Tr[Gamma_L G_(0,N-1) Gamma_R G_(0,N-1)^dagger]
//   (eq.(5));  charge per ring, eq.(4) in the sign convention R12:
//     n_i = -(1/pi) Im sum_k W_k Tr G_(i,i)(z_k) + (1/2pi) sum_k w_k (f_S Tr A_L,(i,i) + f_D Tr A_R,(i,i))
//   (without deg and mode weight: the Python wrapper applies them, as oracle/negf_rgf.py does).
//   Self-energies: closed form of the alternating chain (R8) for lead_kind 0; Sancho-Rubio decimation
//   on the two-ring principal layer with the Newton polish of the fixed point (R9, R10) for lead_kind 1.
//
// Every dense operation is the textbook triple loop / Gaussian elimination with partial pivoting; nothing is
// blocked, fused or reordered beyond what the algorithm states.
#include <algorithm>
#include <cmath>
#include <complex>
#include <cstdint>
#include <cstring>
#include <vector>

#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

typedef std::complex<double> cx;
typedef std::vector<cx> mat;          // row-major m x m

const double PI = 3.14159265358979323846;

// C = A B  (m x m)
void mul(int m, const cx* A, const cx* B, cx* C) {
  for (int i = 0; i < m; ++i)
    for (int j = 0; j < m; ++j) C[i * m + j] = cx(0.0, 0.0);
  for (int i = 0; i < m; ++i)
    for (int k = 0; k < m; ++k) {
      const cx a = A[i * m + k];
      if (a == cx(0.0, 0.0)) continue;
      for (int j = 0; j < m; ++j) C[i * m + j] += a * B[k * m + j];
    }
}
mat mul(int m, const mat& A, const mat& B) {
  mat C((size_t)m * m);
  mul(m, A.data(), B.data(), C.data());
  return C;
}
mat dagger(int m, const mat& A) {
  mat D((size_t)m * m);
  for (int i = 0; i < m; ++i)
    for (int j = 0; j < m; ++j) D[(size_t)j * m + i] = std::conj(A[(size_t)i * m + j]);
  return D;
}
mat neg(const mat& A) {
  mat B(A.size());
  for (size_t i = 0; i < A.size(); ++i) B[i] = -A[i];
  return B;
}

// Solve A X = B in place by Gaussian elimination with partial pivoting and back substitution (A: m x m,
// B: m x r, both row-major, both overwritten; X is left in B).  Returns false if a pivot is exactly zero.
bool gauss_solve(int m, int r, cx* A, cx* B) {
  for (int k = 0; k < m; ++k) {
    int p = k;
    double best = std::abs(A[(size_t)k * m + k]);
    for (int i = k + 1; i < m; ++i) {
      const double v = std::abs(A[(size_t)i * m + k]);
      if (v > best) { best = v; p = i; }
    }
    if (best == 0.0) return false;
    if (p != k) {
      for (int j = 0; j < m; ++j) std::swap(A[(size_t)k * m + j], A[(size_t)p * m + j]);
      for (int j = 0; j < r; ++j) std::swap(B[(size_t)k * r + j], B[(size_t)p * r + j]);
    }
    const cx inv = cx(1.0, 0.0) / A[(size_t)k * m + k];
    for (int i = k + 1; i < m; ++i) {
      const cx f = A[(size_t)i * m + k] * inv;
      if (f == cx(0.0, 0.0)) continue;
      for (int j = k + 1; j < m; ++j) A[(size_t)i * m + j] -= f * A[(size_t)k * m + j];
      for (int j = 0; j < r; ++j) B[(size_t)i * r + j] -= f * B[(size_t)k * r + j];
    }
  }
  for (int k = m - 1; k >= 0; --k) {                       // U X = B'
    const cx inv = cx(1.0, 0.0) / A[(size_t)k * m + k];
    for (int j = 0; j < r; ++j) B[(size_t)k * r + j] *= inv;
    for (int i = 0; i < k; ++i) {
      const cx f = A[(size_t)i * m + k];
      if (f == cx(0.0, 0.0)) continue;
      for (int j = 0; j < r; ++j) B[(size_t)i * r + j] -= f * B[(size_t)k * r + j];
    }
  }
  return true;
}
// A^-1 (A is not modified)
mat inverse(int m, const mat& A) {
  mat W = A, I((size_t)m * m, cx(0.0, 0.0));
  for (int i = 0; i < m; ++i) I[(size_t)i * m + i] = cx(1.0, 0.0);
  if (!gauss_solve(m, m, W.data(), I.data())) std::fill(I.begin(), I.end(), cx(NAN, NAN));
  return I;
}

double fermi(double E, double mu, double kT) {          // F_l(E) = 1/(1 + exp((E - mu_l)/kT))
  const double x = (E - mu) / kT;
  const double e = std::exp(-std::fabs(x));
  return x > 0 ? e / (1.0 + e) : 1.0 / (1.0 + e);
}

// ---------------------------------------------------------------------------------- self-energies

// Retarded surface Green's function of a semi-infinite chain with bonds t1, t2, t1, ... from the
// surface site (reading R8): root of z t2^2 g^2 - (z^2 - t1^2 + t2^2) g + z = 0 with
// S = sqrt(z-(a+b)) sqrt(z-(a-b)) sqrt(z-(b-a)) sqrt(z+(a+b)), principal roots; the form that does
// not cancel is used.
cx surface_gf_alternating(cx z, double t1, double t2) {
  const double a = std::fabs(t1), b = std::fabs(t2);
  const cx X = z * z + (b - a) * (b + a);
  const cx S = std::sqrt(z - (a + b)) * std::sqrt(z - (a - b)) * std::sqrt(z - (b - a)) * std::sqrt(z + (a + b));
  const bool same_side = (X.real() * S.real() + X.imag() * S.imag()) >= 0.0;
  return same_side ? 2.0 * z / (X + S) : (X - S) / (2.0 * z * b * b);
}

// One Newton step on F(g) = [z - H00 - H01 g H01^dagger]^-1 - g = 0 (reading R10; the numpy
// statement is oracle/selfenergy.py::polish_surface_gf).  Only the block X = g[S, S] enters, S = the
// columns in which H01 is non-zero: with B = H01[:, S],  G(X) = [z - H00 - B X B^dagger]^-1,
// dG[S, S] = P dX Q, P = G[S, :] B, Q = B^dagger G[:, S]; solve dX - P dX Q = G[S, S] - X as a dense
// |S|^2 x |S|^2 system (row-major vec: vec(P dX Q) = (P kron Q^T) vec(dX)); return G(X + dX).
mat polish_surface_gf(int m, cx z, const mat& H00, const mat& H01, const mat& g) {
  std::vector<int> S;
  for (int c = 0; c < m; ++c) {
    double s = 0.0;
    for (int r = 0; r < m; ++r) s += std::abs(H01[(size_t)r * m + c]);
    if (s > 0.0) S.push_back(c);
  }
  const int ns = (int)S.size();
  auto G_of = [&](const std::vector<cx>& X) {            // [z - H00 - B X B^dagger]^-1
    mat M((size_t)m * m);
    for (int i = 0; i < m; ++i)
      for (int j = 0; j < m; ++j) M[(size_t)i * m + j] = (i == j ? z : cx(0.0, 0.0)) - H00[(size_t)i * m + j];
    for (int i = 0; i < m; ++i)
      for (int a = 0; a < ns; ++a) {
        const cx bia = H01[(size_t)i * m + S[a]];
        if (bia == cx(0.0, 0.0)) continue;
        for (int b = 0; b < ns; ++b) {
          const cx t = bia * X[(size_t)a * ns + b];
          for (int j = 0; j < m; ++j) M[(size_t)i * m + j] -= t * std::conj(H01[(size_t)j * m + S[b]]);
        }
      }
    return inverse(m, M);
  };
  std::vector<cx> X((size_t)ns * ns);
  for (int a = 0; a < ns; ++a)
    for (int b = 0; b < ns; ++b) X[(size_t)a * ns + b] = g[(size_t)S[a] * m + S[b]];
  const mat G = G_of(X);
  std::vector<cx> P((size_t)ns * ns, cx(0.0, 0.0)), Q((size_t)ns * ns, cx(0.0, 0.0));
  for (int a = 0; a < ns; ++a)
    for (int b = 0; b < ns; ++b) {
      cx p(0.0, 0.0), q(0.0, 0.0);
      for (int r = 0; r < m; ++r) {
        p += G[(size_t)S[a] * m + r] * H01[(size_t)r * m + S[b]];                    // (G[S,:] B)_ab
        q += std::conj(H01[(size_t)r * m + S[a]]) * G[(size_t)r * m + S[b]];         // (B^dagger G[:,S])_ab
      }
      P[(size_t)a * ns + b] = p;
      Q[(size_t)a * ns + b] = q;
    }
  const int D = ns * ns;
  std::vector<cx> A((size_t)D * D), rhs((size_t)D);
  for (int a = 0; a < ns; ++a)
    for (int b = 0; b < ns; ++b) {
      const int row = a * ns + b;
      rhs[row] = G[(size_t)S[a] * m + S[b]] - X[(size_t)a * ns + b];
      for (int c = 0; c < ns; ++c)
        for (int d = 0; d < ns; ++d)
          A[(size_t)row * D + c * ns + d] =
              (row == c * ns + d ? cx(1.0, 0.0) : cx(0.0, 0.0)) - P[(size_t)a * ns + c] * Q[(size_t)d * ns + b];
    }
  gauss_solve(D, 1, A.data(), rhs.data());
  for (int i = 0; i < D; ++i) X[i] += rhs[i];
  return G_of(X);
}

// Sancho-Rubio decimation (refs [33,34]; reading R10):
//   eps_s = eps = H00, a = H01, b = H01^dagger
//   repeat: g = (z - eps)^-1; eps_s += a g b; eps += a g b + b g a; a <- a g a; b <- b g b
//   until max|a|, max|b| < tol, then `extra` more iterations; g_surf = (z - eps_s)^-1; `polish` Newton steps.
mat sancho_rubio(int m, cx z, const mat& H00, const mat& H01, double tol, int maxit, int extra, int polish,
                 int* iters_out) {
  mat eps_s = H00, eps = H00, a = H01, b = dagger(m, H01);
  int remaining = -1, iters = 0;
  for (int it = 0; it < maxit; ++it) {
    mat M((size_t)m * m);
    for (int i = 0; i < m; ++i)
      for (int j = 0; j < m; ++j) M[(size_t)i * m + j] = (i == j ? z : cx(0.0, 0.0)) - eps[(size_t)i * m + j];
    const mat g = inverse(m, M);
    const mat ag = mul(m, a, g), bg = mul(m, b, g);
    const mat agb = mul(m, ag, b), bga = mul(m, bg, a);
    for (size_t i = 0; i < eps.size(); ++i) {
      eps_s[i] += agb[i];
      eps[i] += agb[i] + bga[i];
    }
    a = mul(m, ag, a);
    b = mul(m, bg, b);
    ++iters;
    double mx = 0.0;
    for (size_t i = 0; i < a.size(); ++i) mx = std::max(mx, std::max(std::abs(a[i]), std::abs(b[i])));
    const bool conv = mx < tol;
    if (remaining < 0 && conv) remaining = extra;
    else if (remaining > 0) --remaining;
    if (remaining == 0) break;
  }
  if (iters_out) *iters_out = iters;
  mat M((size_t)m * m);
  for (int i = 0; i < m; ++i)
    for (int j = 0; j < m; ++j) M[(size_t)i * m + j] = (i == j ? z : cx(0.0, 0.0)) - eps_s[(size_t)i * m + j];
  mat g = inverse(m, M);
  for (int p = 0; p < polish; ++p) g = polish_surface_gf(m, z, H00, H01, g);
  return g;
}

struct Leads {            // principal layers of the two leads (reading R9; oracle/selfenergy.py::block_lead_layers)
  mat H00L, H01L, tauL, H00R, H01R, tauR;
};

Leads block_lead_layers(int n, const mat& ce, const mat& co, int N, double U_left, double U_right) {
  auto bond = [&](long j) -> const mat& { return (((j % 2) + 2) % 2 == 0) ? ce : co; };   // H_{j,j+1}
  const int m = 2 * n;
  auto assemble = [&](const mat& a00, const mat& a01, const mat& a10, const mat& a11) {
    mat M((size_t)m * m, cx(0.0, 0.0));
    for (int i = 0; i < n; ++i)
      for (int j = 0; j < n; ++j) {
        M[(size_t)i * m + j] = a00[(size_t)i * n + j];
        M[(size_t)i * m + n + j] = a01[(size_t)i * n + j];
        M[(size_t)(n + i) * m + j] = a10[(size_t)i * n + j];
        M[(size_t)(n + i) * m + n + j] = a11[(size_t)i * n + j];
      }
    return M;
  };
  mat Z((size_t)n * n, cx(0.0, 0.0)), UL = Z, UR = Z;
  for (int i = 0; i < n; ++i) {
    UL[(size_t)i * n + i] = U_left;
    UR[(size_t)i * n + i] = U_right;
  }
  Leads L;
  // left lead, layer p = rings (-1-2p, -2-2p): H00 = [[U, H_{-1,-2}], [H_{-2,-1}, U]], H_{-2,-1} = bond(-2)
  L.H00L = assemble(UL, dagger(n, bond(-2)), bond(-2), UL);
  L.H01L = assemble(Z, Z, dagger(n, bond(-3)), Z);          // H_{-2,-3} = bond(-3)^dagger
  L.tauL = bond(-1);                                        // H_{-1,0}
  // right lead, layer p = rings (N+2p, N+1+2p)
  L.H00R = assemble(UR, bond(N), dagger(n, bond(N)), UR);
  L.H01R = assemble(Z, Z, bond(N + 1), Z);
  L.tauR = dagger(n, bond(N - 1));                          // H_{N,N-1}
  return L;
}

// Sigma = tau^dagger g[:n,:n] tau   (eq.(2))
mat sigma_from_surface(int n, const mat& g2, const mat& tau) {
  mat gs((size_t)n * n);
  for (int i = 0; i < n; ++i)
    for (int j = 0; j < n; ++j) gs[(size_t)i * n + j] = g2[(size_t)i * 2 * n + j];
  return mul(n, mul(n, dagger(n, tau), gs), tau);
}

struct Problem {
  int N, n;
  const double* U;
  mat ce, co;
  int lead_kind;
  double sr_tol;
  int sr_maxit;
  Leads leads;
  double tauL, t1L, tauR, t1R;     // scalar leads (oracle/selfenergy.py::scalar_lead_bonds)
};

void self_energies(const Problem& P, cx z, mat& sigL, mat& sigR, int* iters) {
  const int n = P.n;
  if (P.lead_kind == 0) {
    sigL.assign(1, P.tauL * P.tauL * surface_gf_alternating(z - P.U[0], P.t1L, P.tauL));
    sigR.assign(1, P.tauR * P.tauR * surface_gf_alternating(z - P.U[P.N - 1], P.t1R, P.tauR));
    if (iters) *iters = 0;
    return;
  }
  int itL = 0, itR = 0;
  const mat gL = sancho_rubio(2 * n, z, P.leads.H00L, P.leads.H01L, P.sr_tol, P.sr_maxit, 1, 2, &itL);
  const mat gR = sancho_rubio(2 * n, z, P.leads.H00R, P.leads.H01R, P.sr_tol, P.sr_maxit, 1, 2, &itR);
  sigL = sigma_from_surface(n, gL, P.leads.tauL);
  sigR = sigma_from_surface(n, gR, P.leads.tauR);
  if (iters) *iters = std::max(itL, itR);
}

// Algorithms 2 and 1 at one energy.  trG[N] (complex), trAL[N], trAR[N], T.
void chain_rgf(const Problem& P, cx z, const mat& sigL, const mat& sigR, bool want_G, bool want_A,
               cx* trG, double* trAL, double* trAR, double* T_out) {
  const int N = P.N, n = P.n;
  const size_t nn = (size_t)n * n;
  auto H = [&](int j) -> const mat& { return (j % 2 == 0) ? P.ce : P.co; };
  auto beta = [&](int j) { return neg(H(j)); };                    // -H_{j,j+1}
  auto gamma = [&](int j) { return neg(dagger(n, H(j))); };        // -H_{j+1,j}
  auto alpha = [&](int j) {
    mat a(nn, cx(0.0, 0.0));
    for (int i = 0; i < n; ++i) a[(size_t)i * n + i] = z - P.U[j];
    if (j == 0)
      for (size_t i = 0; i < nn; ++i) a[i] -= sigL[i];
    if (j == N - 1)
      for (size_t i = 0; i < nn; ++i) a[i] -= sigR[i];
    return a;
  };
  auto sub = [&](mat a, const mat& b) {
    for (size_t i = 0; i < nn; ++i) a[i] -= b[i];
    return a;
  };
  // ---------------- Algorithm 2
  std::vector<mat> ytil(N), y(N), xtil(N), x(N);
  y[0] = mat(nn, cx(0.0, 0.0));
  for (int m = 1; m < N; ++m) {
    ytil[m] = mul(n, inverse(n, sub(alpha(m - 1), y[m - 1])), beta(m - 1));
    y[m] = mul(n, gamma(m - 1), ytil[m]);
  }
  x[N - 1] = mat(nn, cx(0.0, 0.0));
  for (int m = N - 2; m >= 0; --m) {
    xtil[m] = mul(n, inverse(n, sub(alpha(m + 1), x[m + 1])), gamma(m));
    x[m] = mul(n, beta(m), xtil[m]);
  }
  // ---------------- Algorithm 1, step 1: diagonal of G^R
  mat G00, GNN;
  for (int Tt = 0; Tt < N; ++Tt) {
    if (!want_G && Tt != 0 && Tt != N - 1) continue;
    const mat GTT = inverse(n, sub(sub(alpha(Tt), x[Tt]), y[Tt]));
    if (want_G) {
      cx tr(0.0, 0.0);
      for (int i = 0; i < n; ++i) tr += GTT[(size_t)i * n + i];
      trG[Tt] = tr;
    }
    if (Tt == 0) G00 = GTT;
    if (Tt == N - 1) GNN = GTT;
  }
  if (!want_A) return;
  mat gamL(nn), gamR(nn);
  for (int i = 0; i < n; ++i)
    for (int j = 0; j < n; ++j) {
      gamL[(size_t)i * n + j] = cx(0.0, 1.0) * (sigL[(size_t)i * n + j] - std::conj(sigL[(size_t)j * n + i]));
      gamR[(size_t)i * n + j] = cx(0.0, 1.0) * (sigR[(size_t)i * n + j] - std::conj(sigR[(size_t)j * n + i]));
    }
  auto tr_A = [&](const mat& Gc, const mat& gam) {          // Tr[G_(T,k) Gamma G_(T,k)^dagger]
    const mat GG = mul(n, Gc, gam);
    double s = 0.0;
    for (size_t i = 0; i < nn; ++i) s += (GG[i] * std::conj(Gc[i])).real();
    return s;
  };
  // lead k = 0 (step 2: downwards from the diagonal)
  mat Gc = G00;
  trAL[0] = tr_A(Gc, gamL);
  for (int m = 0; m < N - 1; ++m) {
    Gc = neg(mul(n, xtil[m], Gc));
    trAL[m + 1] = tr_A(Gc, gamL);
  }
  // lead k = N-1 (step 3: upwards from the diagonal)
  Gc = GNN;
  trAR[N - 1] = tr_A(Gc, gamR);
  for (int m = N - 1; m > 0; --m) {
    Gc = neg(mul(n, ytil[m], Gc));
    trAR[m - 1] = tr_A(Gc, gamR);
  }
  // T = Tr[Gamma_L G_(0,N-1) Gamma_R G_(0,N-1)^dagger]
  const mat t1 = mul(n, mul(n, gamL, Gc), gamR);
  double Tsum = 0.0;
  for (size_t i = 0; i < nn; ++i) Tsum += (t1[i] * std::conj(Gc[i])).real();
  *T_out = Tsum;
}

}  // namespace

extern "C" {

// Charge per ring (without deg / mode weight) and T(E) of ONE chain (n = 1) or ONE real-space channel.
// Complex arrays are interleaved (re, im) doubles.  Returns 0, or 1 for bad arguments.
//   n_ring[N], T[K_neq] are outputs; sr_iters_max (may be null) gets the largest Sancho-Rubio iteration count;
//   sigma_out (may be null): [K_eq + K_neq][2][n*n] complex, the self-energies used (for tests).
int o3_chain_charge(int N, int n, const double* U, const double* coup_even, const double* coup_odd,
                    int K_eq, const double* z_eq, const double* w_eq, int K_neq, const double* z_neq,
                    const double* w_neq, double mu_s, double mu_d, double kT, int lead_kind, double sr_tol,
                    int sr_maxit, int n_threads, double* n_ring, double* T, int* sr_iters_max,
                    double* sigma_out) {
  if (N < 2 || n < 1 || !U || !coup_even || !coup_odd || !n_ring || (lead_kind == 0 && n != 1)) return 1;
  Problem P;
  P.N = N; P.n = n; P.U = U; P.lead_kind = lead_kind; P.sr_tol = sr_tol; P.sr_maxit = sr_maxit;
  const size_t nn = (size_t)n * n;
  P.ce.resize(nn); P.co.resize(nn);
  for (size_t i = 0; i < nn; ++i) {
    P.ce[i] = cx(coup_even[2 * i], coup_even[2 * i + 1]);
    P.co[i] = cx(coup_odd[2 * i], coup_odd[2 * i + 1]);
  }
  if (lead_kind == 0) {
    const double even = std::abs(P.ce[0]), odd = std::abs(P.co[0]);
    P.tauL = odd; P.t1L = even;                         // left: device-lead bond (-1,0) odd, first interior (-2,-1) even
    if ((N - 1) % 2 == 1) { P.tauR = odd; P.t1R = even; } else { P.tauR = even; P.t1R = odd; }
  } else {
    P.leads = block_lead_layers(n, P.ce, P.co, N, U[0], U[N - 1]);
  }
  const int K = K_eq + K_neq;
#ifdef _OPENMP
  const int nt = n_threads > 0 ? n_threads : omp_get_max_threads();
#else
  const int nt = 1;
#endif
  std::vector<std::vector<double>> acc(nt, std::vector<double>(N, 0.0));
  int it_max = 0;
#pragma omp parallel num_threads(nt)
  {
#ifdef _OPENMP
    const int tid = omp_get_thread_num();
#else
    const int tid = 0;
#endif
    std::vector<cx> trG(N);
    std::vector<double> trAL(N), trAR(N);
    int my_it = 0;
#pragma omp for schedule(dynamic, 1)
    for (int k = 0; k < K; ++k) {
      const bool contour = k < K_eq;
      const int kk = contour ? k : k - K_eq;
      const cx z = contour ? cx(z_eq[2 * kk], z_eq[2 * kk + 1]) : cx(z_neq[2 * kk], z_neq[2 * kk + 1]);
      mat sigL, sigR;
      int it = 0;
      self_energies(P, z, sigL, sigR, &it);
      my_it = std::max(my_it, it);
      if (sigma_out)
        for (size_t i = 0; i < nn; ++i) {
          sigma_out[(((size_t)k * 2 + 0) * nn + i) * 2] = sigL[i].real();
          sigma_out[(((size_t)k * 2 + 0) * nn + i) * 2 + 1] = sigL[i].imag();
          sigma_out[(((size_t)k * 2 + 1) * nn + i) * 2] = sigR[i].real();
          sigma_out[(((size_t)k * 2 + 1) * nn + i) * 2 + 1] = sigR[i].imag();
        }
      double Tk = 0.0;
      if (contour) {
        chain_rgf(P, z, sigL, sigR, true, false, trG.data(), nullptr, nullptr, &Tk);
        const cx W(w_eq[2 * kk], w_eq[2 * kk + 1]);
        for (int i = 0; i < N; ++i) acc[tid][i] += (-1.0 / PI) * (W * trG[i]).imag();     // eq.(4), first term
      } else {
        chain_rgf(P, z, sigL, sigR, false, true, nullptr, trAL.data(), trAR.data(), &Tk);
        const double fS = fermi(z.real(), mu_s, kT), fD = fermi(z.real(), mu_d, kT);
        const double w = w_neq[kk] / (2.0 * PI);
        for (int i = 0; i < N; ++i) acc[tid][i] += w * (fS * trAL[i] + fD * trAR[i]);     // eq.(4), second term
        if (T) T[kk] = Tk;
      }
    }
#pragma omp critical
    it_max = std::max(it_max, my_it);
  }
  for (int i = 0; i < N; ++i) {
    double s = 0.0;
    for (int t = 0; t < nt; ++t) s += acc[t][i];        // fixed order over threads
    n_ring[i] = s;
  }
  if (sr_iters_max) *sr_iters_max = it_max;
  return 0;
}

int o3_max_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

}  // extern "C"
