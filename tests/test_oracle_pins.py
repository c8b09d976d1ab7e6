"""Pins of the CPU oracle against what the paper and the mathematics fix.

None of these compares the oracle with itself: each expected value is a closed
form typed out here, a value printed in the paper (tests/golden/paper_values.txt),
an exact identity, or a brute-force computation on a tiny case.
"Pins" (P1..P12) for the list and what mistake each one catches.
"""
import os

import numpy as np
import pytest
from scipy import integrate

import workloads as wlmod
from oracle import negf_dense as od
from oracle import negf_rgf as orgf
from oracle import negf_rgf_omp as omp
from oracle import selfenergy as se

HERE = os.path.dirname(os.path.abspath(__file__))
T = wlmod.T_HOP


def _paper_values():
    vals = {}
    with open(os.path.join(HERE, "golden", "paper_values.txt")) as fh:
        for line in fh:
            line = line.strip()
            if not line or line.startswith("#"):
                continue
            key, val = line.split()[:2]
            vals[key] = float(val)
    return vals


# ------------------------------------------------------------------ P1: 1D closed form

def test_p1_uniform_chain_surface_gf_closed_form():
    """north_star: g = (E - sqrt(E^2 - 4t^2))/(2t^2).  Inside the band the retarded
    value is (E - i sqrt(4t^2 - E^2))/(2t^2); outside it is real and decays like 1/E."""
    t = 2.5
    E = np.linspace(-4.9, 4.9, 197)
    g = se.surface_gf_alternating(E + 1e-13j, t, t)
    expect = (E - 1j * np.sqrt(4 * t * t - E * E)) / (2 * t * t)
    assert np.max(np.abs(g - expect)) < 1e-11        # eta = 1e-13 moves g by ~eta/|t| near the edges
    Eo = np.array([-9.0, -5.5, 5.5, 9.0, 40.0])
    g = se.surface_gf_alternating(Eo + 0j + 1e-300j, t, t)
    expect = (Eo - np.sign(Eo) * np.sqrt(Eo * Eo - 4 * t * t)) / (2 * t * t)
    assert np.max(np.abs(g - expect) / np.abs(expect)) < 1e-13


def test_p1_semicircle_ldos_sum_rule():
    """-Im g/pi is the semicircle sqrt(4t^2-E^2)/(2 pi t^2); it integrates to 1."""
    t = 2.5
    val, _ = integrate.quad(
        lambda E: -se.surface_gf_alternating(np.array([E + 1e-12j]), t, t)[0].imag / np.pi,
        -2 * t, 2 * t, limit=400)
    assert abs(val - 1.0) < 1e-8


def test_p1_small_z_no_cancellation():
    """At z -> 0 (t1 = t2) the exact value is g = -i/|t| + z/(2t^2) + O(z^2); the
    cancelling form loses ~eps/|z|^2 there."""
    t = 2.5
    z = np.array([1e-6j, 1e-6 + 1e-6j, -3e-7 + 1e-6j])
    g = se.surface_gf_alternating(z, t, t)
    series = -1j / t + z / (2 * t * t) + 1j * z * z / (8 * t ** 3)
    assert np.max(np.abs(g - series)) < 1e-15


# ------------------------------------------------------------------ P2: alternating chain

@pytest.mark.parametrize("t1,t2", [(2.5, 2.5), (4.9, 2.5), (0.46, 2.5), (2.5, 0.46), (1.1, 3.3)])
def test_p2_alternating_chain_is_fixed_point_and_retarded(t1, t2):
    """g must satisfy its own continued fraction and have Im g <= 0 (retarded)."""
    rng = np.random.default_rng(5)
    z = rng.uniform(-9, 9, 400) + 1j * 10.0 ** rng.uniform(-9, 0.5, 400)
    g = se.surface_gf_alternating(z, t1, t2)
    gp = 1.0 / (z - t2 * t2 * g)
    resid = g - 1.0 / (z - t1 * t1 * gp)
    assert np.max(np.abs(resid) / np.abs(g)) < 1e-9
    assert np.all(g.imag <= 1e-18)


@pytest.mark.parametrize("t1,t2", [(2.5, 2.5), (4.9, 2.5), (0.46, 2.5)])
def test_p2_alternating_chain_vs_long_finite_chain(t1, t2):
    """Brute force: (0,0) element of the Green's function of a 3000-site chain at
    eta = 0.05 eV (the truncation error decays like exp(-L*eta/|t|))."""
    L = 3000
    bonds = np.where(np.arange(L - 1) % 2 == 0, t1, t2)
    for E in (-6.0, -2.2, -0.3, 0.0, 0.9, 2.6, 5.2):
        z = E + 0.05j
        # tridiagonal solve for the first column of (z - H)^-1 by the Thomas recursion from
        # the far end is itself the continued fraction, so use a dense library solve instead
        H = np.diag(bonds, 1) + np.diag(bonds, -1)
        e0 = np.zeros(L, dtype=np.complex128)
        e0[0] = 1.0
        col = np.linalg.solve(z * np.eye(L) - H, e0)
        g = se.surface_gf_alternating(np.array([z]), t1, t2)[0]
        assert abs(col[0] - g) < 1e-11 * max(1.0, abs(g))


def test_p2_sancho_rubio_equals_closed_form_scalar():
    """Decimation on the 2-site principal layer of an alternating chain (independent
    algorithm) against the closed form."""
    t1, t2 = 4.7, 2.5
    H00 = np.array([[0.0, t1], [t1, 0.0]], dtype=np.complex128)
    H01 = np.array([[0.0, 0.0], [t2, 0.0]], dtype=np.complex128)
    z = np.array([-7.3, -2.0, -0.1, 0.0, 0.4, 2.3, 6.9]) + 1e-6j
    g, iters = se.sancho_rubio(z, H00, H01, tol=1e-12, maxit=200, extra=1)
    closed = se.surface_gf_alternating(z, t1, t2)
    assert np.max(np.abs(g[:, 0, 0] - closed)) < 1e-11
    assert iters.max() < 60


def test_p2_sancho_rubio_cnt_lead_fourier_diagonal():
    """The real-space (17,0) lead is block-circulant: F^dagger g_surf F is diagonal with
    entries g_alt(z; |b_q|, |t|), b_q = t (1 + exp(2 pi i q / 17))."""
    n = wlmod.CNT_N
    ce, co = wlmod.cnt_realspace_couplings()
    layers = se.block_lead_layers(ce, co, 10, 0.0, 0.0)
    H00, H01, tau = layers["left"]
    # includes the hard cases of the raw decimation: next to the zigzag edge state of the modes
    # with |b_q| < |t| (g ~ 1/z at z -> 0), and next to the pole of the isolated layer at
    # -2|t| cos(8 pi/17) = -0.4614 eV, where the unpolished iteration is off by 1e-8
    z = np.array([-0.4626, -0.4614, -0.4, -1e-3, 4e-4, 0.05, 0.2, 0.2713, 0.31, 0.6, 1.3, 3.0]) + 1e-6j
    g, _ = se.sancho_rubio(z, H00, H01)
    gs = g[:, :n, :n]
    F = np.exp(2j * np.pi * np.outer(np.arange(n), np.arange(n)) / n) / np.sqrt(n)
    gd = F.conj().T @ gs @ F
    off = gd - np.einsum("kii->ki", gd)[:, :, None] * np.eye(n)
    scale = np.abs(gs).max(axis=(1, 2))
    assert np.max(np.abs(off).max(axis=(1, 2)) / scale) < 1e-13
    bq = np.abs(T * (1 + np.exp(2j * np.pi * np.arange(n) / n)))
    # 0.2713 eV sits on the van Hove edge |t| - |b_6|, where g ~ sqrt(z - E_c) is itself ill
    # conditioned at eta = 1e-6; everywhere else the match is at rounding level
    tol = np.where(np.abs(z.real - 0.2713) < 1e-9, 2e-12, 1e-13)
    for q in range(n):
        closed = se.surface_gf_alternating(z, bq[q], abs(T))
        assert np.all(np.abs(gd[:, q, q] - closed) / scale < tol)
    # the Newton polish is what delivers this: the raw decimation misses it by orders of magnitude
    graw, _ = se.sancho_rubio(z[:2], H00, H01, polish=0)
    assert np.max(np.abs(graw[:, :n, :n] - gs[:2])) > 1e-10


def test_p2_surface_gf_is_fixed_point_of_adding_a_layer():
    """Defining property (refs [33,34]): g = [z - H00 - H01 g H01^dagger]^-1, for a random
    non-Hermitian-coupled lead where no closed form exists."""
    rng = np.random.default_rng(42)
    m = 6
    H00 = rng.normal(size=(m, m)) + 1j * rng.normal(size=(m, m))
    H00 = 0.5 * (H00 + H00.conj().T)
    H01 = 0.7 * (rng.normal(size=(m, m)) + 1j * rng.normal(size=(m, m)))
    z = np.array([-1.3, -0.2, 0.0, 0.45, 2.1]) + 1e-6j
    g, iters = se.sancho_rubio(z, H00, H01)
    assert iters.max() < 200
    for k in range(len(z)):
        G = np.linalg.inv(z[k] * np.eye(m) - H00 - H01 @ g[k] @ H01.conj().T)
        assert np.max(np.abs(G - g[k])) < 1e-12 * max(1.0, np.abs(g[k]).max())
        assert np.all(np.linalg.eigvalsh((g[k] - g[k].conj().T) / 2j) < 1e-9)   # retarded: Im g <= 0


@pytest.mark.parametrize("N,n,seed", [(4, 3, 0), (5, 3, 1), (5, 2, 2), (3, 4, 3)])
def test_p2_block_leads_brute_force_non_commuting_couplings(N, n, seed):
    """Brute force of the block-lead construction (eq.(2): Sigma = tau^dagger g tau;
    decimation; readings R7, R9).  On the (17,0) tube every coupling commutes, so a
    dagger/transpose or left/right mix-up in ``block_lead_layers`` / ``sigma_block`` would be
    invisible there.  Here the couplings are random complex NON-commuting n x n blocks; the leads are
    written out explicitly as L rings per side continuing the even/odd bond pattern of the device
    (bond (j, j+1) is coup_even for even j, coup_odd for odd j, for every integer j) at the end
    ring's on-site energy, and the whole (N + 2L) n matrix is inverted densely.  Its device block
    must equal the Green's function the oracle gets from Sancho-Rubio self-energies.  eta = 0.4
    makes the truncation error exp(-O(L eta)) negligible at L = 320."""
    rng = np.random.default_rng(300 + seed)
    ce = rng.normal(size=(n, n)) + 1j * rng.normal(size=(n, n))
    co = rng.normal(size=(n, n)) + 1j * rng.normal(size=(n, n))
    assert np.max(np.abs(ce @ co - co @ ce)) > 0.1          # the point of the test
    U = rng.uniform(-0.5, 0.5, N)
    L = 320
    tot = N + 2 * L

    def bond(j):                                              # H_{j,j+1}, j any integer
        return ce if j % 2 == 0 else co

    for z in (0.37 + 0.4j, -1.1 + 0.4j):
        Hbig = np.zeros((tot * n, tot * n), dtype=np.complex128)
        for r in range(tot):
            j = r - L                                         # ring index; device is 0 .. N-1
            Uj = U[0] if j < 0 else (U[N - 1] if j >= N else U[j])
            Hbig[r * n:(r + 1) * n, r * n:(r + 1) * n] = Uj * np.eye(n)
            if r + 1 < tot:
                B = bond(j)
                Hbig[r * n:(r + 1) * n, (r + 1) * n:(r + 2) * n] = B
                Hbig[(r + 1) * n:(r + 2) * n, r * n:(r + 1) * n] = B.conj().T
        Gbig = np.linalg.inv(z * np.eye(tot * n) - Hbig)
        Gdev = Gbig[L * n:(L + N) * n, L * n:(L + N) * n]
        G, sL, sR = od.green_dense(U, ce, co, n, z, lead_kind=1)
        assert np.max(np.abs(G - Gdev)) < 1e-9 * np.max(np.abs(Gdev))
        # and the two self-energies on their own: Sigma = M_dev - G_dev^-1 restricted to the end blocks
        Mdev = z * np.eye(N * n) - od.build_hamiltonian(U, ce, co, n)
        S = Mdev - np.linalg.inv(Gdev)
        assert np.max(np.abs(S[:n, :n] - sL)) < 1e-8 * np.max(np.abs(sL))
        assert np.max(np.abs(S[-n:, -n:] - sR)) < 1e-8 * np.max(np.abs(sR))
        assert np.max(np.abs(S[n:-n, n:-n])) < 1e-8            # only the end blocks carry Sigma


# ------------------------------------------------------------------ P3: values printed in the paper

def test_p3_paper_bandgap_and_degeneracy():
    pv = _paper_values()
    n = int(pv["cnt_chirality_n"])
    assert n == wlmod.CNT_N and abs(abs(wlmod.T_HOP) - pv["hopping_abs_eV"]) < 1e-15
    even, odd = wlmod.cnt_mode_couplings()
    gaps = 2 * np.abs(np.abs(odd) - np.abs(even))          # gap of subband j of an alternating chain
    gap = np.sort(gaps.real)
    assert abs(gap[0] - 0.5426) < 1e-4                     # 2|t| min_q |1 - 2 cos(pi q/17)|
    assert round(gap[0], 2) == 0.54 and abs(gap[0] - pv["bandgap_eV"]) < 0.01
    assert abs(gap[0] - gap[1]) < 1e-12                    # doubly degenerate
    ce, _ = wlmod.cnt_realspace_couplings()
    ev = np.sort(np.abs(np.linalg.eigvals(ce / T)))
    assert np.allclose(ev, np.sort(np.abs(2 * np.cos(np.pi * np.arange(n) / n))), atol=1e-12)


def test_p3_ring_pitch():
    """512 rings <-> 54.53 nm = 3/4 a_cc per ring, a_cc = 0.142 nm."""
    pv = _paper_values()
    assert abs(pv["rings_N512_length_nm"] / 512 - 0.75 * 0.142) < 2e-4


# ------------------------------------------------------------------ P4: integer transmission

def _open_modes(E):
    even, odd = wlmod.cnt_mode_couplings()
    b, t = np.abs(even), np.abs(odd)
    return int(np.sum((np.abs(t - b) < abs(E)) & (abs(E) < t + b)))


@pytest.mark.parametrize("kind", ["scalar", "block"])
def test_p4_integer_transmission_ideal_tube(kind):
    E = np.array([0.2, 0.3, 0.6, 1.2, 3.0])
    expect = np.array([_open_modes(e) for e in E])
    assert list(expect) == [0, 2, 4, 8, 15]
    w = wlmod.make_config(3 if kind == "block" else 2, N=8, K_neq=8, K_eq=0)
    w.phi[:] = 0.0
    w.z_neq = E + 1e-10j
    w.w_neq = np.ones(len(E))
    _, Tm = od.charge_and_transmission(w)
    assert np.max(np.abs(Tm[0] - expect)) < 1e-6


def test_p4_uniform_chain_transmission_is_one():
    w = wlmod.config1(N=12, K_neq=9)
    w.phi[:] = 0.3
    w.z_neq = np.linspace(-4.5, 4.5, 9) - 0.3 + 1e-11j
    _, Tm = od.charge_and_transmission(w)
    assert np.max(np.abs(Tm[0] - 1.0)) < 1e-7
    w.z_neq = np.array([-5.4, 5.3]) + 1e-11j
    w.w_neq = np.ones(2)
    _, Tm = od.charge_and_transmission(w)
    assert np.max(np.abs(Tm[0])) < 1e-6


# ------------------------------------------------------------------ P5/P6: exact identities

@pytest.mark.parametrize("cfg", [2, 3])
def test_p5_spectral_identity_and_hermiticity(cfg):
    """i(G - G^dagger) = G (Gamma_L + Gamma_R + 2 eta I) G^dagger  exactly."""
    w = wlmod.make_config(cfg, N=10, K_neq=4, K_eq=0)
    n = w.n
    eta = 1e-3
    for E in (-0.35, 0.05, 0.62):
        if cfg == 2:
            ce, co = w.coup_even[5:6], w.coup_odd[5:6]
        else:
            ce, co = w.coup_even, w.coup_odd
        G, sL, sR = od.green_dense(-w.phi[0], ce, co, n, E + 1j * eta, w.lead_kind)
        D = G.shape[0]
        gam = np.zeros((D, D), dtype=np.complex128)
        gam[:n, :n] = 1j * (sL - sL.conj().T)
        gam[D - n:, D - n:] = 1j * (sR - sR.conj().T)
        lhs = 1j * (G - G.conj().T)
        rhs = G @ (gam + 2 * eta * np.eye(D)) @ G.conj().T
        assert np.max(np.abs(lhs - rhs)) < 1e-12 * max(1.0, np.max(np.abs(lhs)))
        AL = G[:, :n] @ gam[:n, :n] @ G[:, :n].conj().T
        assert np.max(np.abs(AL - AL.conj().T)) < 1e-13
        assert np.all(np.diagonal(AL).real > -1e-14)
        # reciprocity for real H: T_LR = T_RL
        gL, gR = gam[:n, :n], gam[D - n:, D - n:]
        TLR = np.trace(gL @ G[:n, D - n:] @ gR @ G[:n, D - n:].conj().T).real
        TRL = np.trace(gR @ G[D - n:, :n] @ gL @ G[D - n:, :n].conj().T).real
        assert abs(TLR - TRL) < 1e-12 * max(1.0, abs(TLR))


# ------------------------------------------------------------------ eq.(5)-(6): current, conductance

def _ideal_tube(kind, N, E_lo, E_hi, K, mu_s, mu_d, kT, eta=1e-9):
    w = wlmod.make_config(3 if kind == "block" else 2, N=N, K_neq=K, K_eq=0)
    w.phi[:] = 0.0
    w.z_neq, w.w_neq = wlmod.real_axis_gauss_legendre(E_lo, E_hi, K, eta)
    w.mu_s, w.mu_d, w.kT = mu_s, mu_d, kT
    return w


@pytest.mark.parametrize("kind", ["scalar", "block"])
def test_f1_landauer_current_of_ideal_tube_counts_open_modes(kind):
    """eq.(5): for an ideal tube every open subband transmits perfectly, so at low kT
    with both chemical potentials inside one transmission plateau I = (g_s e/h) M (mu_S - mu_D),
    M = number of open modes (2 between the first subband edge 0.2713 eV and the second 0.5127 eV);
    I_S + I_D = 0 (current conservation, P6); G = M G_0 (eq.(6))."""
    mu_s, mu_d, kT = 0.42, 0.36, 0.004
    lo, hi = mu_d - 14 * kT, mu_s + 14 * kT                   # [0.304, 0.476] inside the plateau
    w = _ideal_tube(kind, 6, lo, hi, 160, mu_s, mu_d, kT)
    I_S, I_D, G = od.landauer_dense(w)
    assert abs(I_S[0] - 2.0 * (mu_s - mu_d)) < 1e-6           # O(N eta) + Fermi tails exp(-14)
    assert abs(I_S[0] + I_D[0]) < 1e-9 * abs(I_S[0])
    assert abs(G[0] - 2.0) < 1e-5


def test_f1_current_equals_transmission_form_and_changes_sign():
    """Tr[F_S Gamma_S A + i Gamma_S G^<] = T_SD (F_S - F_D) for two leads (algebra on eq.(5)); the
    definition-based oracle must agree with the T(E)-based sum of the other oracle path, vanish at
    mu_S = mu_D and flip sign with the bias."""
    w = wlmod.make_config(2, N=14, K_neq=12, K_eq=0)
    I_S, I_D, _ = od.landauer_dense(w)
    _, T = od.charge_and_transmission(w)
    fS = od.fermi_real(w.z_neq.real, w.mu_s, w.kT)
    fD = od.fermi_real(w.z_neq.real, w.mu_d, w.kT)
    expect = np.sum(w.w_neq * T[0] * (fS - fD))
    assert abs(I_S[0] - expect) < 1e-12 * abs(expect)
    assert abs(I_S[0] + I_D[0]) < 1e-10 * abs(I_S[0])         # real H: T_SD = T_DS exactly (P6)
    w.mu_s, w.mu_d = w.mu_d, w.mu_s
    I_S2, _, _ = od.landauer_dense(w)
    assert abs(I_S2[0] + I_S[0]) < 1e-12 * abs(I_S[0])
    w.mu_d = w.mu_s
    I_S3, _, _ = od.landauer_dense(w)
    assert abs(I_S3[0]) < 1e-14


# ------------------------------------------------------------------ P7: real space == sum of modes

def test_p7_real_space_equals_sum_of_modes():
    wb = wlmod.make_config(3, N=12, K_neq=10, K_eq=6)
    ws = wlmod.scalar_twin(wb)
    nb, Tb = od.charge_and_transmission(wb)
    ns, Ts = od.charge_and_transmission(ws)
    assert np.max(np.abs(nb - ns) / np.abs(ns)) < 1e-10
    assert np.max(np.abs(Tb - Ts)) < 1e-9


# ------------------------------------------------------------------ P8/P9: energy reduction

def _chain_workload(N, K_neq, K_eq, mu_s, mu_d, kT=wlmod.KT, e_b=-6.0):
    w = wlmod.config1(N=N, K_neq=8)
    w.phi[:] = 0.0
    e_min = min(mu_s, mu_d) - wlmod.F_TAIL * kT
    e_max = max(mu_s, mu_d) + wlmod.F_TAIL * kT
    w.z_neq, w.w_neq = wlmod.real_axis_gauss_legendre(e_min, e_max, K_neq)
    w.z_eq, w.w_eq = wlmod.contour_semicircle(e_b, e_min, K_eq, min(mu_s, mu_d), kT)
    w.mu_s, w.mu_d, w.kT = mu_s, mu_d, kT
    return w


def test_p8_half_filling():
    """phi = 0, mu_S = mu_D = 0: exactly 1/2 electron per orbital per spin
    (bipartite lattice); pins sign, 1/pi vs 1/2pi, deg, contour weights, Fermi factors.
    Accuracy is eta-limited (the missing 2 eta G G^dagger of P5): ~5e-8."""
    w = _chain_workload(N=14, K_neq=96, K_eq=48, mu_s=0.0, mu_d=0.0)
    n, _ = od.charge_and_transmission(w)
    assert np.max(np.abs(n[0] / w.deg - 0.5)) < 5e-7


def test_p9_biased_uniform_chain_density():
    """Uniform chain under bias: n per spin = int LDOS(E) (f_S + f_D)/2 dE with
    LDOS = 1/(pi sqrt(4t^2 - E^2)) (bulk site of an infinite chain)."""
    mu_s, mu_d, kT, t = 0.0, -0.1, 0.0259, 2.5

    def f(E, mu):
        return 1.0 / (1.0 + np.exp((E - mu) / kT))

    val, _ = integrate.quad(
        lambda E: (f(E, mu_s) + f(E, mu_d)) / 2 / (np.pi * np.sqrt(4 * t * t - E * E)),
        -2 * t, 2 * t, points=[mu_d, mu_s], limit=500, epsabs=1e-12, epsrel=1e-12)
    assert abs(val - 0.4968165483) < 1e-8                   # value quoted in SURVEY P9
    w = _chain_workload(N=14, K_neq=128, K_eq=48, mu_s=mu_s, mu_d=mu_d)
    n, _ = od.charge_and_transmission(w)
    assert np.max(np.abs(n[0] / w.deg - val)) < 5e-7


# ------------------------------------------------------------------ contours and grids

def test_f3_equilibrium_contour_closed_form():
    """contour_equilibrium on a function with a closed-form answer: for G(z) = 1/(z - a), a in the
    lower half plane, int_{e_b}^{E_u} G F dE is a plain 1D integral (scipy.quad); the contour sum
    (two arcs + enclosed Fermi poles with weight -2 pi i kT) must reproduce it.  A wrong pole sign,
    weight or count misses by ~2 pi kT |G| ~ 0.1."""
    kT, mu, eb = 0.0259, -0.05, -8.5
    G = lambda z: 1.0 / (z + 1.0 + 0.3j) + 0.5 / (z - 0.02 + 0.05j)
    z, W, m = wlmod.contour_equilibrium(eb, mu, kT, 64)
    assert m == 3 and len(z) == 64 + 64 + 3
    e_u = mu + 2 * np.pi * kT * m
    assert e_u >= mu + wlmod.F_TAIL * kT
    f = lambda E: 1.0 / (1.0 + np.exp((E - mu) / kT))
    re = integrate.quad(lambda E: (G(E) * f(E)).real, eb, e_u, limit=2000, points=[mu, -1, 0.02])[0]
    im = integrate.quad(lambda E: (G(E) * f(E)).imag, eb, e_u, limit=2000, points=[mu, -1, 0.02])[0]
    assert abs(np.sum(W * G(z)) - (re + 1j * im)) < 5e-6


@pytest.mark.parametrize("which", ["chain", "tube"])
def test_f3_equilibrium_only_equals_two_part_result(which):
    """at equilibrium (mu_S = mu_D) the residue-theorem contour alone gives the charge;
    it must equal the two-part result of eq.(4) at mu_S = mu_D (SURVEY 8(f)-3 pin).  Devices whose
    van Hove edges lie outside the Fermi window, so that the two-part real-axis quadrature is itself
    accurate; the remaining difference is the 2 eta G G^dagger term of P5 (~1e-7)."""
    if which == "chain":
        base = wlmod.make_config(1, N=12, K_neq=8)
        mu, e_b = 0.3, -6.0
    else:
        base = wlmod.make_config(3, N=8, K_neq=8, K_eq=8)
        base.phi[:] = 0.01 * np.linspace(-1.0, 1.0, 8)
        base.kT = 0.004
        mu, e_b = 0.4, wlmod.E_B                           # window [0.34, 0.46] inside the first plateau
    weq = wlmod.equilibrium_variant(base, mu=mu, K_eq=48, e_b=e_b)
    n_eq, _ = od.charge_and_transmission(weq)
    w2 = wlmod.two_part_equilibrium_variant(base, mu=mu, K_eq=48, K_neq=128)
    w2.z_eq, w2.w_eq = wlmod.contour_semicircle(e_b, mu - wlmod.F_TAIL * base.kT, 48, mu, base.kT)
    n_2, _ = od.charge_and_transmission(w2)
    assert weq.K_neq == 0 and weq.extra["n_poles"] == 3
    assert np.max(np.abs(n_eq - n_2) / n_2) < 2e-6


def test_f3_neutral_charge_of_ideal_tube_is_half_filling():
    """rho_0 ("E_l = E_u = 0"): all states below the charge-neutrality point filled.
    For the ideal tube (bipartite lattice, phi = 0) that is exactly one electron per atom:
    n = deg * 17 / 2 = 17 per ring."""
    w = wlmod.neutral_variant(wlmod.make_config(3, N=6, K_neq=4, K_eq=4), K_eq=48)
    w.phi[:] = 0.0
    n, _ = od.charge_and_transmission(w)
    assert np.max(np.abs(n - 17.0)) < 1e-6
    ws = wlmod.neutral_variant(wlmod.make_config(2, N=9, K_neq=4, K_eq=4), K_eq=48)
    ws.phi[:] = 0.0
    n, _ = od.charge_and_transmission(ws)
    assert np.max(np.abs(n - 17.0)) < 1e-6


def test_f2_three_segment_grid():
    """three sub-regions with their own density of points per kT, Gauss-Legendre in each;
    the paper's densities (500, 1600, 50) on its window give ~12 000 points."""
    kT = 0.0259
    e_min, e_max = -0.1 - 14 * kT, 0.0 + 14 * kT
    z, w, counts = wlmod.real_axis_three_segment(e_min, -0.30, -0.25, e_max, kT, (500, 1600, 50))
    assert len(z) == sum(counts) == len(w)
    assert counts == (int(np.ceil(500 * (-0.30 - e_min) / kT)), int(np.ceil(1600 * 0.05 / kT)),
                      int(np.ceil(50 * (e_max + 0.25) / kT)))
    assert 5000 < len(z) < 20000
    E = z.real
    assert np.all(np.diff(E) > 0) and np.all(z.imag == wlmod.ETA)
    assert abs(w.sum() - (e_max - e_min)) < 1e-13                     # weights cover the window exactly
    assert abs(np.sum(w * E ** 5) - (e_max ** 6 - e_min ** 6) / 6) < 1e-13   # exact for polynomials
    # a sharp peak inside the dense segment is integrated to 1e-9; with one 64-point rule it is not
    lor = lambda x: (1e-3 / np.pi) / ((x + 0.27) ** 2 + 1e-6)
    exact = (np.arctan((e_max + 0.27) / 1e-3) - np.arctan((e_min + 0.27) / 1e-3)) / np.pi
    assert abs(np.sum(w * lor(E)) - exact) < 1e-9
    z1, w1 = wlmod.real_axis_gauss_legendre(e_min, e_max, 64)
    assert abs(np.sum(w1 * lor(z1.real)) - exact) > 1e-2
    # degenerate limits collapse to fewer segments
    z2, w2, c2 = wlmod.real_axis_three_segment(e_min, e_min - 1.0, e_min - 0.5, e_max, kT, (500, 1600, 50))
    assert c2[0] == 0 and c2[1] == 0 and abs(w2.sum() - (e_max - e_min)) < 1e-13


def test_f2_refine_segment_limits_brackets_the_peak():
    E = np.linspace(-0.4, 0.3, 701)
    integrand = 1.0 / np.sqrt(np.abs(E + 0.2713) + 1e-4)              # van Hove-like edge
    e_s, l1, l2 = wlmod.refine_segment_limits(E, integrand, 0.0259)
    assert abs(e_s + 0.2713) < 1e-3 and l1 == e_s - 3 * 0.0259 and l2 == e_s + 0.0259


def test_f2_integrand_sums_to_the_real_axis_charge():
    """integrand_dense is the energy-resolved second term of eq.(4): deg/(2 pi) sum_k w_k I(E_k) must give the
    real-axis charge of that ring; for the ideal tube deep in a band it equals 2 pi x the local density
    of states summed over the open modes times the occupation (A_S + A_D = 2 pi LDOS, P5)."""
    w = wlmod.make_config(2, N=11, K_neq=14, K_eq=0)
    I = od.integrand_dense(w, 5)
    n, _ = od.charge_and_transmission(w)
    assert abs(w.deg / (2 * np.pi) * np.sum(w.w_neq * I[0]) - n[0, 5]) < 1e-13 * n[0, 5]
    # ideal uniform chain, E inside the band, both leads fully occupied: A_S + A_D = 2 pi LDOS = 2 / sqrt(4t^2 - E^2)
    c = wlmod.make_config(1, N=9, K_neq=5)
    c.phi[:] = 0.0
    c.mu_s = c.mu_d = 50.0
    c.z_neq = (np.array([-1.0, -0.3, 0.0, 0.4, 2.0]) + 1e-9j).astype(np.complex128)
    I = od.integrand_dense(c, 4)
    assert np.max(np.abs(I[0] - 2.0 / np.sqrt(4 * 2.5 ** 2 - c.z_neq.real ** 2))) < 1e-7


# ------------------------------------------------------------------ P10: brute force, O1 vs O3

def _random_hermitian_device(rng, N, n):
    ce = rng.normal(size=(n, n)) + 1j * rng.normal(size=(n, n))
    co = rng.normal(size=(n, n)) + 1j * rng.normal(size=(n, n))
    U = rng.uniform(-0.5, 0.5, N)
    return U, ce, co


@pytest.mark.parametrize("N,n", [(2, 3), (5, 3), (6, 4), (7, 1), (8, 1)])
def test_p10_dense_vs_paper_recursion_random_complex_blocks(N, n):
    """Non-symmetric complex coupling blocks catch beta/gamma and dagger/transpose
    mistakes; both lead parities (N even / odd) are exercised."""
    rng = np.random.default_rng(100 + 10 * N + n)
    U, ce, co = _random_hermitian_device(rng, N, n)
    if n == 1:
        ce, co = ce.reshape(1), co.reshape(1)
    z_neq = rng.uniform(-3, 3, 6) + 1e-3j
    w_neq = rng.uniform(0.5, 1.5, 6)
    z_eq = rng.uniform(-3, 3, 4) + 1j * rng.uniform(0.1, 2.0, 4)
    w_eq = rng.normal(size=4) + 1j * rng.normal(size=4)
    lead_kind = 0 if n == 1 else 1
    args = (U, ce, co, n, z_eq, w_eq, z_neq, w_neq, 0.1, -0.2, 0.05, lead_kind)
    n1, T1 = od.chain_dense(*args)
    n3, T3 = orgf.chain_charge(*args)
    assert np.max(np.abs(n1 - n3)) < 1e-11 * np.max(np.abs(n1))
    assert np.max(np.abs(T1 - T3)) < 1e-11 * max(1.0, np.max(np.abs(T1)))


@pytest.mark.parametrize("cfg,kw", [(1, dict(N=30, K_neq=40)),
                                    (2, dict(N=40, K_neq=24, K_eq=8)),
                                    (3, dict(N=16, K_neq=12, K_eq=6)),
                                    (4, dict(C=2, N=14, K_neq=8, K_eq=4))])
def test_p10_dense_vs_paper_recursion_on_shrunk_configs(cfg, kw):
    w = wlmod.make_config(cfg, **kw)
    n1, T1 = od.charge_and_transmission(w)
    n3, T3 = orgf.charge_and_transmission(w)
    assert np.max(np.abs(n1 - n3) / np.abs(n1)) < 1e-11
    tol = 1e-11 * np.maximum(np.abs(T1), 1e-6 * np.max(np.abs(T1)))
    assert np.all(np.abs(T1 - T3) <= tol + 1e-300)


# ------------------------------------------------------------------ P10 for the C++/OpenMP tier O3

@pytest.mark.parametrize("N,n", [(2, 3), (5, 3), (6, 4), (7, 1), (8, 1), (4, 17)])
def test_p10_dense_vs_cpp_recursion_random_complex_blocks(N, n):
    """oracle/negf_rgf_omp.cpp (own Sancho-Rubio, own elimination, Alg.2 + Alg.1) against the dense
    definition on random NON-symmetric complex blocks, both lead parities."""
    rng = np.random.default_rng(100 + 10 * N + n)
    U, ce, co = _random_hermitian_device(rng, N, n)
    if n == 1:
        ce, co = ce.reshape(1), co.reshape(1)
    z_neq = rng.uniform(-3, 3, 6) + 1e-3j
    w_neq = rng.uniform(0.5, 1.5, 6)
    z_eq = rng.uniform(-3, 3, 4) + 1j * rng.uniform(0.1, 2.0, 4)
    w_eq = rng.normal(size=4) + 1j * rng.normal(size=4)
    lead_kind = 0 if n == 1 else 1
    args = (U, ce, co, n, z_eq, w_eq, z_neq, w_neq, 0.1, -0.2, 0.05, lead_kind)
    n1, T1 = od.chain_dense(*args)
    n3, T3 = omp.chain_charge(*args)
    assert np.max(np.abs(n1 - n3)) < 1e-11 * np.max(np.abs(n1))
    assert np.max(np.abs(T1 - T3)) < 1e-11 * max(1.0, np.max(np.abs(T1)))


@pytest.mark.parametrize("cfg,kw", [(1, dict(N=30, K_neq=40)),
                                    (2, dict(N=40, K_neq=24, K_eq=8)),
                                    (3, dict(N=16, K_neq=12, K_eq=6)),
                                    (4, dict(C=2, N=14, K_neq=8, K_eq=4))])
def test_p10_dense_vs_cpp_recursion_on_shrunk_configs(cfg, kw):
    w = wlmod.make_config(cfg, **kw)
    n1, T1 = od.charge_and_transmission(w)
    n3, T3 = omp.charge_and_transmission(w)
    assert np.max(np.abs(n1 - n3) / np.abs(n1)) < 1e-11
    tol = 1e-11 * np.maximum(np.abs(T1), 1e-6 * np.max(np.abs(T1)))
    assert np.all(np.abs(T1 - T3) <= tol + 1e-300)


def test_cpp_tier_is_thread_count_independent_up_to_rounding():
    """One energy per thread; the per-thread partial charges are summed in thread order, so a
    different thread count only reorders a sum (1e-16 relative)."""
    w = wlmod.make_config(3, N=10, K_neq=9, K_eq=3)
    a = omp.charge_and_transmission(w, threads=1)
    b = omp.charge_and_transmission(w, threads=3)
    assert np.max(np.abs(a[0] - b[0]) / np.abs(a[0])) < 1e-14
    assert np.array_equal(a[1], b[1])
