"""Tier O3 (paper's Algorithms 1-2) against an independent library algorithm at
full device length: banded LU (LAPACK zgbsv via scipy) for the first and last
block columns of G^R (SURVEY 8(c) tier O2)."""
import numpy as np
from scipy.linalg import solve_banded

import workloads as wlmod
from oracle import negf_rgf as orgf
from oracle import negf_rgf_omp as omp
from oracle import selfenergy as se


def _banded_columns(U, ce, co, n, z, sL, sR):
    """First and last block columns of [zI - H - Sigma]^-1 by banded LU."""
    N = U.shape[0]
    D = N * n
    kl = ku = 2 * n - 1
    ab = np.zeros((kl + ku + 1, D), dtype=np.complex128)

    def put(r, c, v):
        ab[ku + r - c, c] += v

    for i in range(N):
        for a in range(n):
            put(i * n + a, i * n + a, z - U[i])
        if i + 1 < N:
            B = ce if i % 2 == 0 else co
            for a in range(n):
                for b in range(n):
                    if B[a, b] != 0:
                        put(i * n + a, (i + 1) * n + b, -B[a, b])
                        put((i + 1) * n + b, i * n + a, -np.conj(B[a, b]))
    for a in range(n):
        for b in range(n):
            put(a, b, -sL[a, b])
            put(D - n + a, D - n + b, -sR[a, b])
    rhs = np.zeros((D, 2 * n), dtype=np.complex128)
    rhs[:n, :n] = np.eye(n)
    rhs[D - n:, n:] = np.eye(n)
    X = solve_banded((kl, ku), ab, rhs)
    return X[:, :n], X[:, n:]


def test_o3_vs_banded_lu_full_length_config3():
    w = wlmod.config3()                       # N = 1000, n = 17, full length
    n, N = w.n, w.N
    U = -w.phi[0]
    idx = np.array([5, 700, 1311, 2040])      # in-gap, near band edge, in band
    z = w.z_neq[idx]
    sL, sR, _ = se.sigma_block(z, w.coup_even, w.coup_odd, N, U[0], U[-1])
    _, trAL, trAR, Tm = orgf.chain_rgf(U, w.coup_even, w.coup_odd, n, z, sL, sR)
    for k in range(len(z)):
        GL, GR = _banded_columns(U, w.coup_even, w.coup_odd, n, z[k], sL[k], sR[k])
        gamL = 1j * (sL[k] - sL[k].conj().T)
        gamR = 1j * (sR[k] - sR[k].conj().T)
        AL = np.einsum("ia,ab,ib->i", GL, gamL, GL.conj()).real.reshape(N, n).sum(1)
        AR = np.einsum("ia,ab,ib->i", GR, gamR, GR.conj()).real.reshape(N, n).sum(1)
        G0N = GR[:n]
        T = np.trace(gamL @ G0N @ gamR @ G0N.conj().T).real
        scale = max(AL.max(), AR.max())
        assert np.max(np.abs(AL - trAL[k])) < 1e-10 * scale
        assert np.max(np.abs(AR - trAR[k])) < 1e-10 * scale
        assert abs(T - Tm[k]) < 1e-10 * max(1.0, abs(T))


def test_o3_vs_banded_lu_full_length_config2_mode():
    w = wlmod.config2()
    U = -w.phi[0]
    N = w.N
    j = 6                                      # lowest-gap subband
    ce, co = w.coup_even[j:j + 1], w.coup_odd[j:j + 1]
    idx = np.array([3, 1000, 2500, 4090])
    z = w.z_neq[idx]
    (tauL, t1L), (tauR, t1R) = se.scalar_lead_bonds(ce, co, N)
    sL = se.sigma_scalar(z, U[0], tauL, t1L).reshape(-1, 1, 1)
    sR = se.sigma_scalar(z, U[-1], tauR, t1R).reshape(-1, 1, 1)
    _, trAL, trAR, Tm = orgf.chain_rgf(U, ce, co, 1, z, sL, sR)
    for k in range(len(z)):
        GL, GR = _banded_columns(U, ce.reshape(1, 1), co.reshape(1, 1), 1, z[k], sL[k], sR[k])
        gL, gR = -2 * sL[k, 0, 0].imag, -2 * sR[k, 0, 0].imag
        AL = (np.abs(GL[:, 0]) ** 2) * gL
        AR = (np.abs(GR[:, 0]) ** 2) * gR
        T = gL * gR * abs(GR[0, 0]) ** 2
        scale = max(AL.max(), AR.max())
        assert np.max(np.abs(AL - trAL[k])) < 1e-10 * scale
        assert np.max(np.abs(AR - trAR[k])) < 1e-10 * scale
        assert abs(T - Tm[k]) < 1e-10 * max(1e-6, abs(T))


def test_cpp_o3_vs_banded_lu_and_numpy_tier_full_length_config3():
    """The C++/OpenMP tier at full device length (N = 1000, n = 17) on sampled energies: per-ring
    charge and T(E) against the banded-LU columns (independent library algorithm) with the C++
    tier's own self-energies, and against the numpy tier end to end."""
    w = wlmod.config3()
    n, N = w.n, w.N
    U = -w.phi[0]
    idx = np.array([5, 700, 1311, 2040])
    z = w.z_neq[idx]
    one = np.ones(1)
    for k in range(len(z)):
        # one real-axis point with weight 1, mu far above / far below: f_S = 1, f_D = 0 isolates A_L, and v.v.
        nL, T, sig = omp.chain_charge(U, w.coup_even, w.coup_odd, n, [], [], z[k:k + 1], one,
                                      50.0, -50.0, 0.0259, 1, want_sigma=True)
        nR, _ = omp.chain_charge(U, w.coup_even, w.coup_odd, n, [], [], z[k:k + 1], one,
                                 -50.0, 50.0, 0.0259, 1)
        sL, sR = sig[0, 0], sig[0, 1]
        GL, GR = _banded_columns(U, w.coup_even, w.coup_odd, n, z[k], sL, sR)
        gamL = 1j * (sL - sL.conj().T)
        gamR = 1j * (sR - sR.conj().T)
        AL = np.einsum("ia,ab,ib->i", GL, gamL, GL.conj()).real.reshape(N, n).sum(1)
        AR = np.einsum("ia,ab,ib->i", GR, gamR, GR.conj()).real.reshape(N, n).sum(1)
        G0N = GR[:n]
        Tb = np.trace(gamL @ G0N @ gamR @ G0N.conj().T).real
        scale = max(AL.max(), AR.max())
        assert np.max(np.abs(AL - 2 * np.pi * nL)) < 1e-10 * scale
        assert np.max(np.abs(AR - 2 * np.pi * nR)) < 1e-10 * scale
        assert abs(Tb - T[0]) < 1e-10 * max(1.0, abs(Tb))
        # self-energies of the two tiers agree (both polished to rounding level, reading R10)
        sLn, sRn, _ = se.sigma_block(z[k:k + 1], w.coup_even, w.coup_odd, N, U[0], U[-1])
        assert np.max(np.abs(sLn[0] - sL)) < 1e-11 * np.max(np.abs(sL))
        assert np.max(np.abs(sRn[0] - sR)) < 1e-11 * np.max(np.abs(sR))
    sub = w.subset(neq_idx=idx, eq_idx=[0, 31, 63], channels=[0])
    n_np, T_np = orgf.charge_and_transmission(sub)
    n_cc, T_cc = omp.charge_and_transmission(sub)
    assert np.max(np.abs(n_np - n_cc) / np.abs(n_np)) < 1e-11
    assert np.max(np.abs(T_np - T_cc)) < 1e-11 * max(1.0, np.max(np.abs(T_np)))


def test_cpp_o3_scalar_vs_numpy_tier_full_length_config2_mode():
    w = wlmod.config2()
    sub = w.subset(neq_idx=np.arange(0, 4096, 64), eq_idx=np.arange(0, 64, 4), channels=[0])
    n_np, T_np = orgf.charge_and_transmission(sub)
    n_cc, T_cc = omp.charge_and_transmission(sub)
    assert np.max(np.abs(n_np - n_cc) / np.abs(n_np)) < 1e-12
    tol = 1e-11 * np.maximum(np.abs(T_np), 1e-6 * np.max(np.abs(T_np)))
    assert np.all(np.abs(T_np - T_cc) <= tol)
