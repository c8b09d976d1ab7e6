"""Input generators for the five workloads of BASELINE.json (``configs[0..4]``).

Everything here is *input construction*: potentials, coupling blocks, energy
grids with their quadrature weights, and the fixed linear map that stands in
for Poisson in config 5.  The recipe follows SURVEY.md 8(d) and is restated in
DESIGN.md.  The paper's devices give the shapes:
(17,0) zigzag tube, |t| = 2.5 eV, N = 512..4096 rings, 400..12000 real-axis
points + ~90 contour points, several channels coupled only through
electrostatics.

Conventions:
  * energies in eV, potentials phi in volts, on-site energy U_i = -phi_i
    (diagonal of H is -e*phi);
  * ring i -> i+1 coupling is ``coup_even`` for even i, ``coup_odd`` for odd i;
  * real-axis nodes are handed over as z = E + i*eta, contour nodes as they are;
  * contour weights already contain dz/dtheta, the Gauss-Legendre weight and the
    Fermi function of the lowest-mu lead, so that
        n_i += deg * (-1/pi) * Im[ W_k * Tr G_ii(z_k) ]        (eq.(4) 1st term)
"""
from __future__ import annotations

from dataclasses import dataclass, field, replace
from typing import Optional

import numpy as np

CNT_N = 17          # (17,0) zigzag tube
T_HOP = -2.5        # eV, nearest-neighbour coupling (|t| = 2.5 eV)
ETA = 1.0e-6        # eV, "infinitesimal constant" of eq.(2), PAPER.md:82 (value: BASELINE.json configs[0])
KT = 0.0259         # eV
MU_S = 0.0          # eV
MU_D = -0.1         # eV
DEG = 2.0           # g_s
E_B = -8.5          # eV, lower end of the contour: below the band bottom -3|t| - max U
F_TAIL = 14.0       # f_1 = f_2 = 14


@dataclass
class Workload:
    """All inputs of one ``negf_create`` + ``negf_set_potential`` call."""
    name: str
    kind: str                     # "scalar" (block == 1) or "block"
    C: int                        # channels
    N: int                        # rings per channel
    n: int                        # block size (1 scalar, 17 real space)
    n_modes: int                  # scalar: chains per channel; block: 1
    coup_even: np.ndarray         # scalar: (n_modes,) c128; block: (n, n) c128  -- H_{i,i+1}, i even
    coup_odd: np.ndarray          # same, i odd
    mode_weight: np.ndarray       # (n_modes,) f64
    phi: np.ndarray               # (C, N) f64, volts; U = -phi
    z_eq: np.ndarray              # (K_eq,) c128 contour nodes
    w_eq: np.ndarray              # (K_eq,) c128 contour weights (see module docstring)
    z_neq: np.ndarray             # (K_neq,) c128 = E_k + i*eta
    w_neq: np.ndarray             # (K_neq,) f64 real-axis weights
    mu_s: float = MU_S
    mu_d: float = MU_D
    kT: float = KT
    deg: float = DEG
    lead_kind: int = 0            # 0 closed form (scalar), 1 Sancho-Rubio (block)
    sr_tol: float = 1.0e-12
    sr_maxit: int = 200
    eta: float = ETA
    seed: int = 0
    extra: dict = field(default_factory=dict)

    @property
    def K_eq(self) -> int:
        return int(self.z_eq.shape[0])

    @property
    def K_neq(self) -> int:
        return int(self.z_neq.shape[0])

    @property
    def sweeps(self) -> int:
        """Energy-point RGF sweeps per charge evaluation (BASELINE.json metric unit)."""
        return self.C * self.n_modes * (self.K_eq + self.K_neq)

    def subset(self, neq_idx=None, eq_idx=None, channels=None) -> "Workload":
        """Same device, a sample of its energy points / channels (weights kept)."""
        w = replace(self)
        if neq_idx is not None:
            neq_idx = np.asarray(neq_idx, dtype=np.int64)
            w.z_neq = self.z_neq[neq_idx].copy()
            w.w_neq = self.w_neq[neq_idx].copy()
        if eq_idx is not None:
            eq_idx = np.asarray(eq_idx, dtype=np.int64)
            w.z_eq = self.z_eq[eq_idx].copy()
            w.w_eq = self.w_eq[eq_idx].copy()
        if channels is not None:
            channels = np.asarray(channels, dtype=np.int64)
            w.phi = self.phi[channels].copy()
            w.C = int(channels.shape[0])
        return w


# --------------------------------------------------------------------------- grids

def fermi(z, mu: float, kT: float):
    """Fermi function 1/(1+exp((z-mu)/kT)) for real or complex z."""
    z = np.asarray(z)
    x = (z - mu) / kT
    if np.iscomplexobj(x):
        return 1.0 / (1.0 + np.exp(x))
    out = np.empty_like(x, dtype=np.float64)
    pos = x > 0
    out[~pos] = 1.0 / (1.0 + np.exp(x[~pos]))
    e = np.exp(-x[pos])
    out[pos] = e / (1.0 + e)
    return out


def real_axis_uniform(e_lo: float, e_hi: float, K: int, eta: float = ETA):
    """Uniform grid with trapezoid weights (config 1: BASELINE.json configs[0])."""
    E = np.linspace(e_lo, e_hi, K)
    dE = (e_hi - e_lo) / (K - 1)
    w = np.full(K, dE)
    w[0] = w[-1] = 0.5 * dE
    return (E + 1j * eta).astype(np.complex128), w.astype(np.float64)


def real_axis_gauss_legendre(e_lo: float, e_hi: float, K: int, eta: float = ETA):
    """One Gauss-Legendre rule on [e_lo, e_hi] (Gauss-Legendre per
    sub-region; 'the smallest channel length can be simulated with just one
    integration path')."""
    x, w = np.polynomial.legendre.leggauss(K)
    half = 0.5 * (e_hi - e_lo)
    E = 0.5 * (e_hi + e_lo) + half * x
    return (E + 1j * eta).astype(np.complex128), (half * w).astype(np.float64)


def contour_semicircle(e_b: float, e_min: float, K: int, mu_min: float, kT: float):
    """Semicircle in the upper half plane from e_b to e_min with a Gauss-Legendre
    rule in the angle ('contour integration ... Gauss-Legendre
    mapping'; the shape is not given in the paper -- DESIGN.md reading R13).

    z(theta) = c + R exp(i theta), theta_k = (pi/2)(x_k + 1).
    int_{e_b}^{e_min} f dE = -int_0^pi f(z) i R exp(i theta) dtheta, hence
    W_k = -i R exp(i theta_k) (pi/2) w_k F_min(z_k).
    """
    if K == 0:
        return np.zeros(0, np.complex128), np.zeros(0, np.complex128)
    x, w = np.polynomial.legendre.leggauss(K)
    theta = 0.5 * np.pi * (x + 1.0)
    c = 0.5 * (e_b + e_min)
    R = 0.5 * (e_min - e_b)
    z = c + R * np.exp(1j * theta)
    W = -1j * R * np.exp(1j * theta) * (0.5 * np.pi * w) * fermi(z, mu_min, kT)
    return z.astype(np.complex128), W.astype(np.complex128)


def contour_equilibrium(e_b: float, mu: float, kT: float, K: int, f_tail: float = F_TAIL, K_cap: int = 64):
    """Equilibrium-only contour ("At equilibrium ... the charge density
    can be calculated solely using the residue theorem by setting E_l = E_u = mu + f k_bT").

    The real-axis integral int_{e_b}^{E_u} G^R F dE is closed in the upper half plane, where G^R is
    analytic and the Fermi function has the simple poles z_p = mu + i pi kT (2p + 1) with residue -kT:
        int_{e_b}^{E_u} G F dE = -int_arcs G F dz - 2 pi i kT sum_{p inside} G(z_p).
    The path is two semicircles: the large one of ``contour_semicircle`` from e_b to mu - r (left of
    the Fermi edge, where F is smooth) and a small cap of radius r around mu from mu - r to
    E_u = mu + r, r = 2 pi kT m with the smallest integer m for which r >= f_tail kT -- the cap
    crosses Re z = mu midway between the poles m - 1 and m, so that no pole sits on the path and
    the K_cap Gauss-Legendre points of the cap resolve the pole structure (a single large semicircle
    crossing the pole line converges only at ~500 points).  Node list: K points of the large arc,
    K_cap points of the cap, then the m enclosed poles with weight W_p = -2 pi i kT.
    Returns (z, W, number of poles).  DESIGN.md reading R24."""
    m = int(np.ceil(f_tail / (2.0 * np.pi)))
    r = 2.0 * np.pi * kT * m
    za, Wa = contour_semicircle(e_b, mu - r, K, mu, kT)
    zc, Wc = contour_semicircle(mu - r, mu + r, K_cap, mu, kT)
    zp = mu + 1j * np.pi * kT * (2.0 * np.arange(m) + 1.0)          # Im z_p < r
    Wp = np.full(m, -2.0j * np.pi * kT, dtype=np.complex128)
    return (np.concatenate([za, zc, zp]).astype(np.complex128),
            np.concatenate([Wa, Wc, Wp]).astype(np.complex128), m)


def contour_neutral(e_b: float, K: int, e_u: float = 0.0):
    """Contour of the neutral charge density rho_0 ("computed with E_l = E_u = 0"):
    all states below E = 0 -- the charge-neutrality point of the tube -- filled, no thermal smearing,
    so the occupation factor is 1 on the whole arc and no pole is enclosed (reading R24)."""
    if K == 0:
        return np.zeros(0, np.complex128), np.zeros(0, np.complex128)
    x, w = np.polynomial.legendre.leggauss(K)
    theta = 0.5 * np.pi * (x + 1.0)
    c = 0.5 * (e_b + e_u)
    R = 0.5 * (e_u - e_b)
    z = c + R * np.exp(1j * theta)
    W = -1j * R * np.exp(1j * theta) * (0.5 * np.pi * w)
    return z.astype(np.complex128), W.astype(np.complex128)


def real_axis_three_segment(e_min: float, e_l1: float, e_l2: float, e_max: float, kT: float,
                            density=(500.0, 1600.0, 50.0), eta: float = ETA, k_max: int = 1 << 20):
    """Semi-adaptive real-axis path of PAPER.md:353: [e_min, e_l1], [e_l1, e_l2],
    [e_l2, e_max], each with its own density of integration points per kT (the paper's largest
    device: (500, 1600, 50), ~12 000 points in total) and its own Gauss-Legendre rule.  Empty
    segments (e.g. e_l1 <= e_min) are dropped.  Returns (z = E + i eta, w, points per segment)."""
    edges = [e_min, min(max(e_l1, e_min), e_max), min(max(e_l2, e_l1, e_min), e_max), e_max]
    zs, ws, counts = [], [], []
    for s in range(3):
        lo, hi = edges[s], edges[s + 1]
        if hi - lo <= 0.0:
            counts.append(0)
            continue
        k = int(min(max(np.ceil(density[s] * (hi - lo) / kT), 2), k_max))
        z, w = real_axis_gauss_legendre(lo, hi, k, eta)
        zs.append(z)
        ws.append(w)
        counts.append(k)
    return np.concatenate(zs), np.concatenate(ws), tuple(counts)


def refine_segment_limits(E, integrand, kT: float, a: float = 3.0, b: float = 1.0):
    """The refresh step of the semi-adaptive path: locate the peak E_s of the integrand
    A_1 F_1 + A_2 F_2 at the centre of the channel and put the dense segment around it,
    E_l1 = E_s - a kT, E_l2 = E_s + b kT (a = 3, b = 1 "typically").  The paper prints
    "E_l1 = E_l1 - akT", read as E_s - akT (reading R25).  Returns (E_s, E_l1, E_l2)."""
    E = np.asarray(E, dtype=np.float64)
    k = int(np.argmax(np.asarray(integrand, dtype=np.float64)))
    e_s = float(E[k])
    return e_s, e_s - a * kT, e_s + b * kT


def _window(mu_s: float, mu_d: float, kT: float):
    return min(mu_s, mu_d) - F_TAIL * kT, max(mu_s, mu_d) + F_TAIL * kT


# --------------------------------------------------------------------------- devices

def barrier_profile(N: int) -> np.ndarray:
    """p_i = 1/2 [tanh((i - N/4)/w) - tanh((i - 3N/4)/w)], w = N/40: a smooth gate
    barrier like the band profiles of PAPER.md Fig.4(c) (:345)."""
    i = np.arange(N, dtype=np.float64)
    w = N / 40.0
    return 0.5 * (np.tanh((i - N / 4.0) / w) - np.tanh((i - 3.0 * N / 4.0) / w))


def cnt_mode_couplings(t: float = T_HOP, n: int = CNT_N):
    """Mode-space couplings of a (n,0) zigzag tube: the bond between rings
    alternates between 2 t cos(pi j / n) (two bonds per atom) and t (one bond per
    atom), j = 0..n-1  (BASELINE.json configs[1]; mode space of ref [23],
    PAPER.md:47, :113)."""
    j = np.arange(n, dtype=np.float64)
    even = (2.0 * t * np.cos(np.pi * j / n)).astype(np.complex128)
    odd = np.full(n, t, dtype=np.complex128)
    return even, odd


def cnt_realspace_couplings(t: float = T_HOP, n: int = CNT_N):
    """Real-space ring-to-ring blocks of a (n,0) tube: atom a bonded to atoms a and
    a+1 (cyclic) of the next ring on even bonds, atom a to atom a on odd bonds
    (BASELINE.json configs[2])."""
    eye = np.eye(n)
    P = np.roll(eye, 1, axis=1)          # P[a, (a+1) % n] = 1
    even = (t * (eye + P)).astype(np.complex128)
    odd = (t * eye).astype(np.complex128)
    return even, odd


def _grids(K_neq, K_eq, mu_s=MU_S, mu_d=MU_D, kT=KT, eta=ETA, e_b=E_B):
    e_min, e_max = _window(mu_s, mu_d, kT)
    z_neq, w_neq = real_axis_gauss_legendre(e_min, e_max, K_neq, eta)
    z_eq, w_eq = contour_semicircle(e_b, e_min, K_eq, min(mu_s, mu_d), kT)
    return z_eq, w_eq, z_neq, w_neq


def config1(N: int = 100, K_neq: int = 1000, seed: int = 1001) -> Workload:
    """configs[0]: one uniform 1D chain, analytic leads, uniform real-axis grid."""
    rng = np.random.default_rng(seed)
    U = -0.2 * np.arange(N) / (N - 1) + rng.uniform(-0.01, 0.01, N)
    z_neq, w_neq = real_axis_uniform(-1.0, 1.0, K_neq, ETA)
    t = np.array([T_HOP], dtype=np.complex128)
    return Workload(
        name="config1", kind="scalar", C=1, N=N, n=1, n_modes=1,
        coup_even=t.copy(), coup_odd=t.copy(), mode_weight=np.ones(1),
        phi=(-U)[None, :].copy(),
        z_eq=np.zeros(0, np.complex128), w_eq=np.zeros(0, np.complex128),
        z_neq=z_neq, w_neq=w_neq, lead_kind=0, seed=seed)


def _gate_potential(N, height, noise, rng):
    return height * barrier_profile(N) + rng.uniform(-noise, noise, N)


def config2(N: int = 1000, K_neq: int = 4096, K_eq: int = 64, seed: int = 1002) -> Workload:
    """configs[1]: (17,0) tube in mode space, 17 scalar chains."""
    rng = np.random.default_rng(seed)
    U = _gate_potential(N, 0.3, 0.005, rng)
    even, odd = cnt_mode_couplings()
    z_eq, w_eq, z_neq, w_neq = _grids(K_neq, K_eq)
    return Workload(
        name="config2", kind="scalar", C=1, N=N, n=1, n_modes=CNT_N,
        coup_even=even, coup_odd=odd, mode_weight=np.ones(CNT_N),
        phi=(-U)[None, :].copy(), z_eq=z_eq, w_eq=w_eq, z_neq=z_neq, w_neq=w_neq,
        lead_kind=0, seed=seed)


def config3(N: int = 1000, K_neq: int = 2048, K_eq: int = 64, seed: int = 1002) -> Workload:
    """configs[2]: the same tube in real space, 17x17 blocks, Sancho-Rubio leads.
    Same seed (hence potential) as config 2 so that pin P7 (real space == sum of
    modes) can be checked between the two paths."""
    rng = np.random.default_rng(seed)
    U = _gate_potential(N, 0.3, 0.005, rng)
    even, odd = cnt_realspace_couplings()
    z_eq, w_eq, z_neq, w_neq = _grids(K_neq, K_eq)
    return Workload(
        name="config3", kind="block", C=1, N=N, n=CNT_N, n_modes=1,
        coup_even=even, coup_odd=odd, mode_weight=np.ones(1),
        phi=(-U)[None, :].copy(), z_eq=z_eq, w_eq=w_eq, z_neq=z_neq, w_neq=w_neq,
        lead_kind=1, seed=seed)


def _array_potential(C, N, seed0):
    phi = np.empty((C, N))
    heights = np.empty(C)
    for c in range(C):
        rng = np.random.default_rng(seed0 + c)
        heights[c] = rng.uniform(0.1, 0.4)
        phi[c] = -_gate_potential(N, heights[c], 0.005, rng)
    return phi, heights


def config4(C: int = 16, N: int = 2000, K_neq: int = 4096, K_eq: int = 64,
            seed: int = 1004) -> Workload:
    """configs[3]: array of C misaligned tubes, each its own barrier height."""
    phi, heights = _array_potential(C, N, seed)
    even, odd = cnt_realspace_couplings()
    z_eq, w_eq, z_neq, w_neq = _grids(K_neq, K_eq)
    return Workload(
        name="config4", kind="block", C=C, N=N, n=CNT_N, n_modes=1,
        coup_even=even, coup_odd=odd, mode_weight=np.ones(1), phi=phi,
        z_eq=z_eq, w_eq=w_eq, z_neq=z_neq, w_neq=w_neq, lead_kind=1, seed=seed,
        extra={"heights": heights})


@dataclass
class PoissonStandIn:
    """Fixed seeded, diagonally dominant sparse linear map K standing in for the
    electrostatics of PAPER.md:59-65 (BASELINE.json configs[4]):
        phi_out = phi_ext - K (n - n0).
    K_(c,i),(c,i) = kappa; K_(c,i),(c,i+-d) = kappa*(0.25, 0.10, 0.05), d = 1,2,3;
    K_(c,i),(c+-1,i) = kappa*0.05*r_(c,i), r ~ U(0.5,1).  Off-diagonal row sum
    <= 0.9 kappa.  ``apply`` works on numpy arrays and torch tensors alike (it only
    slices, scales and adds): it is harness code, not part of the library."""
    kappa: float
    r: np.ndarray                 # (C-1, N): coupling between channel c and c+1 at ring i
    n0: float
    along: tuple = (0.25, 0.10, 0.05)

    def apply_K(self, q, r=None):
        """K q for q of shape (C, N); ``r`` may be a device copy of self.r."""
        r = self.r if r is None else r
        out = self.kappa * q
        for d, a in enumerate(self.along, start=1):
            out[:, d:] += (self.kappa * a) * q[:, :-d]
            out[:, :-d] += (self.kappa * a) * q[:, d:]
        if q.shape[0] > 1:
            out[1:] += (self.kappa * 0.05) * r * q[:-1]
            out[:-1] += (self.kappa * 0.05) * r * q[1:]
        return out

    def phi_out(self, phi_ext, n, r=None):
        return phi_ext - self.apply_K(n - self.n0, r)

    def as_csr(self, C: int, N: int):
        """The same map K as one (C N) x (C N) sparse matrix in CSR form (row pointers, column indices,
        values), row-major over (channel, ring): one SpMV instead of ~15 slice operations."""
        idx = np.arange(C * N).reshape(C, N)
        rows, cols, vals = [idx.ravel()], [idx.ravel()], [np.full(C * N, self.kappa)]
        for d, a in enumerate(self.along, start=1):
            for src, dst in ((idx[:, :-d], idx[:, d:]), (idx[:, d:], idx[:, :-d])):
                rows.append(dst.ravel())
                cols.append(src.ravel())
                vals.append(np.full(src.size, self.kappa * a))
        if C > 1:
            w = (self.kappa * 0.05) * np.asarray(self.r)
            rows += [idx[1:].ravel(), idx[:-1].ravel()]
            cols += [idx[:-1].ravel(), idx[1:].ravel()]
            vals += [w.ravel(), w.ravel()]
        rows, cols, vals = np.concatenate(rows), np.concatenate(cols), np.concatenate(vals)
        order = np.lexsort((cols, rows))
        rows, cols, vals = rows[order], cols[order], vals[order]
        rowptr = np.zeros(C * N + 1, dtype=np.int64)
        np.add.at(rowptr, rows + 1, 1)
        return np.cumsum(rowptr), cols.astype(np.int64), vals.astype(np.float64)


def config5(C: int = 64, N: int = 4000, K_neq: int = 8192, K_eq: int = 128,
            seed: int = 1005, kappa: float = 0.2) -> Workload:
    """configs[4]: self-consistent loop on a C-channel array; the returned workload
    carries phi_ext as ``phi`` and the Poisson stand-in in ``extra['poisson']``;
    20 modified-Broyden iterations, history 8, mixing 0.1."""
    phi, heights = _array_potential(C, N, seed)
    even, odd = cnt_realspace_couplings()
    z_eq, w_eq, z_neq, w_neq = _grids(K_neq, K_eq)
    rng = np.random.default_rng(seed + 1500)
    r = rng.uniform(0.5, 1.0, (max(C - 1, 0), N))
    poisson = PoissonStandIn(kappa=kappa, r=r, n0=DEG * CNT_N / 2.0)
    return Workload(
        name="config5", kind="block", C=C, N=N, n=CNT_N, n_modes=1,
        coup_even=even, coup_odd=odd, mode_weight=np.ones(1), phi=phi,
        z_eq=z_eq, w_eq=w_eq, z_neq=z_neq, w_neq=w_neq, lead_kind=1, seed=seed,
        extra={"heights": heights, "poisson": poisson, "broyden_iters": 20,
               "broyden_history": 8, "broyden_zeta": 0.1})


def scalar_twin(block_wl: Workload) -> Workload:
    """Mode-space (scalar) workload with the potential and grids of a real-space
    (17,0) workload: for pin P7 (ring-uniform potential => the block-circulant
    real-space tube equals the sum of its 17 mode chains)."""
    even, odd = cnt_mode_couplings()
    return replace(block_wl, name=block_wl.name + "_modes", kind="scalar", n=1,
                   n_modes=CNT_N, coup_even=even, coup_odd=odd,
                   mode_weight=np.ones(CNT_N), lead_kind=0)


def table2(N: int = 524288, n_modes: int = 8, K_arc: int = 23, K_cap: int = 64, seed: int = 2002,
           mu: float = 0.0) -> Workload:
    """The long-channel, few-energy workload of the paper's Table 2:
    N = 524 288 rings, equilibrium (contour only), 90 contour points, modes 1..n_modes of the (17,0)
    tube in mode space, each doubly degenerate ("modes 1 to 8 (all doubly-degenerate)").
    90 points = 23 on the large arc + 64 on the cap around mu + the 3 enclosed Fermi poles
    (``contour_equilibrium``).  Potential: the gate barrier of configs 2-5 stretched to N rings, height
    0.3 eV, +-5 meV noise.  The parallelism over energies is scarce here (90 x 8 chains): the sweep is a
    serial pass over 524 288 rings per chain."""
    rng = np.random.default_rng(seed)
    U = _gate_potential(N, 0.3, 0.005, rng)
    j = np.arange(1, n_modes + 1, dtype=np.float64)
    even = (2.0 * T_HOP * np.cos(np.pi * j / CNT_N)).astype(np.complex128)
    odd = np.full(n_modes, T_HOP, dtype=np.complex128)
    z, W, n_poles = contour_equilibrium(E_B, mu, KT, K_arc, K_cap=K_cap)
    return Workload(
        name="table2", kind="scalar", C=1, N=N, n=1, n_modes=n_modes,
        coup_even=even, coup_odd=odd, mode_weight=np.full(n_modes, 2.0),
        phi=(-U)[None, :].copy(), z_eq=z, w_eq=W,
        z_neq=np.zeros(0, np.complex128), w_neq=np.zeros(0, np.float64),
        mu_s=mu, mu_d=mu, lead_kind=0, seed=seed, extra={"n_poles": n_poles})


_FACTORIES = {1: config1, 2: config2, 3: config3, 4: config4, 5: config5, 6: table2}


def make_config(idx: int, **overrides) -> Workload:
    """``make_config(3, N=40, K_neq=16, K_eq=8)`` gives the shrunk variant of
    config 3 produced by the same generator."""
    return _FACTORIES[idx](**overrides)


def equilibrium_variant(wl: Workload, mu: Optional[float] = None, K_eq: int = 64, e_b: float = E_B) -> Workload:
    """Equilibrium-only evaluation of a workload: mu_S = mu_D = mu, no real-axis points,
    the contour of ``contour_equilibrium`` with the enclosed Fermi poles appended."""
    mu = wl.mu_s if mu is None else mu
    z, W, n_poles = contour_equilibrium(e_b, mu, wl.kT, K_eq)
    return replace(wl, name=wl.name + "_equilibrium", mu_s=mu, mu_d=mu, z_eq=z, w_eq=W,
                   z_neq=np.zeros(0, np.complex128), w_neq=np.zeros(0, np.float64),
                   extra=dict(wl.extra, n_poles=n_poles))


def two_part_equilibrium_variant(wl: Workload, mu: Optional[float] = None, K_eq: int = 64,
                                 K_neq: int = 256) -> Workload:
    """The same physical quantity through the two-part path of eq.(4) at mu_S = mu_D = mu (the pin of the
    equilibrium-only contour: both must give the same charge)."""
    mu = wl.mu_s if mu is None else mu
    z_eq, w_eq, z_neq, w_neq = _grids(K_neq, K_eq, mu_s=mu, mu_d=mu, kT=wl.kT, eta=wl.eta)
    return replace(wl, name=wl.name + "_twopart", mu_s=mu, mu_d=mu, z_eq=z_eq, w_eq=w_eq,
                   z_neq=z_neq, w_neq=w_neq)


def neutral_variant(wl: Workload, K_eq: int = 64, e_b: float = E_B) -> Workload:
    """Neutral charge density rho_0 of a workload: ``contour_neutral``, no real-axis points."""
    z, W = contour_neutral(e_b, K_eq)
    return replace(wl, name=wl.name + "_neutral", z_eq=z, w_eq=W,
                   z_neq=np.zeros(0, np.complex128), w_neq=np.zeros(0, np.float64))
