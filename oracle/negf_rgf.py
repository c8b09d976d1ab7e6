"""Tier O3 oracle: the paper's block-tridiagonal recursion (Algorithm 2 + Algorithm 1).

TEST INFRASTRUCTURE ONLY (see oracle/__init__.py).  Shares no code with the CUDA
path.  This module follows the paper's own algorithm step by step, in its
notation, so that full-size devices (where the dense definition of
``negf_dense`` cannot go) still have a CPU result.  It is itself required to
match ``negf_dense`` on small devices and a banded LU solve at full N
(tests/test_oracle_rgf.py).

Notation (readings R1, R2, R6):
  alpha_j = z - U_j - [j=0] Sigma_L - [j=N-1] Sigma_R     diagonal of (G^R)^-1
  beta_j  = upper diagonal of (G^R)^-1 = -H_{j,j+1}
  gamma_j = lower diagonal of (G^R)^-1 = -H_{j+1,j} = -H_{j,j+1}^dagger

Algorithm 2, with beta/gamma placed as required for
non-commuting blocks (the printed form has them exchanged, which is immaterial
for the scalar real hoppings the paper ran -- reading R1):
  y_0 = x_{N-1} = 0
  ytilde_n = [alpha_{n-1} - y_{n-1}]^-1 beta_{n-1},   y_n = gamma_{n-1} ytilde_n     n = 1..N-1
  xtilde_n = [alpha_{n+1} - x_{n+1}]^-1 gamma_n,      x_n = beta_n xtilde_n          n = N-2..0

Algorithm 1 (steps 1-4 are lost in the extracted text and are
restored from the prose at :131 and by analogy with steps 6-8 -- reading R2):
  1. G_(T,T)   = [alpha_T - x_T - y_T]^-1
  2. G_(n+1,T) = -xtilde_n G_(n,T)        n >= T
  3. G_(n-1,T) = -ytilde_n G_(n,T)        n <= T
  6-8. A_l,(T,T) = G_(T,k) Gamma_l,(k,k) G_(T,k)^dagger   with G_(T,k) from the
       recursions 2/3 started at the lead block k (k = 0 and k = N-1).
Only the diagonal blocks are kept.
"""
from __future__ import annotations

import numpy as np

from . import selfenergy as se
from .negf_dense import fermi_real


def _inv(a):
    return 1.0 / a if a.shape[-1] == 1 else np.linalg.inv(a)


def _mm(a, b):
    return a * b if (a.shape[-1] == 1 and b.shape[-1] == 1) else a @ b


def _dag(a):
    return np.conj(np.swapaxes(a, -1, -2))


def chain_rgf(U, coup_even, coup_odd, n, z, sigL, sigR):
    """Algorithms 2 and 1 for K energies at once.

    Returns (trG[K, N] complex: Tr_ring G_(T,T);
             trAL[K, N], trAR[K, N] real: Tr_ring A_l,(T,T);
             T[K] real: Tr[Gamma_L G_(0,N-1) Gamma_R G_(0,N-1)^dagger]).
    """
    U = np.asarray(U, dtype=np.float64)
    N = U.shape[0]
    z = np.asarray(z, dtype=np.complex128)
    K = z.shape[0]
    ce = np.asarray(coup_even, dtype=np.complex128).reshape(n, n)
    co = np.asarray(coup_odd, dtype=np.complex128).reshape(n, n)
    eye = np.eye(n, dtype=np.complex128)

    def beta(j):            # -H_{j,j+1}
        return -(ce if j % 2 == 0 else co)

    def gamma(j):           # -H_{j+1,j}
        return -(ce if j % 2 == 0 else co).conj().T

    def alpha(j):
        a = (z - U[j])[:, None, None] * eye
        if j == 0:
            a = a - sigL
        if j == N - 1:
            a = a - sigR
        return a

    # ---------------- Algorithm 2
    ytil = [None] * N
    y = [None] * N
    y[0] = np.zeros((K, n, n), dtype=np.complex128)
    for m in range(1, N):
        ytil[m] = _mm(_inv(alpha(m - 1) - y[m - 1]), beta(m - 1))
        y[m] = _mm(gamma(m - 1), ytil[m])
    xtil = [None] * N
    x = [None] * N
    x[N - 1] = np.zeros((K, n, n), dtype=np.complex128)
    for m in range(N - 2, -1, -1):
        xtil[m] = _mm(_inv(alpha(m + 1) - x[m + 1]), gamma(m))
        x[m] = _mm(beta(m), xtil[m])

    # ---------------- Algorithm 1, diagonal of G^R (step 1)
    trG = np.empty((K, N), dtype=np.complex128)
    G00 = GNN = None
    for T in range(N):
        GTT = _inv(alpha(T) - x[T] - y[T])
        trG[:, T] = np.trace(GTT, axis1=-2, axis2=-1)
        if T == 0:
            G00 = GTT
        if T == N - 1:
            GNN = GTT

    gamL = 1j * (sigL - _dag(sigL))
    gamR = 1j * (sigR - _dag(sigR))

    def tr_A(Gcol, gam):    # Tr[ G_(T,k) Gamma G_(T,k)^dagger ]
        return np.einsum("kab,kbc,kac->k", Gcol, gam, Gcol.conj()).real

    # ---------------- Algorithm 1, lead k = 0 (step 2: downwards from the diagonal)
    trAL = np.empty((K, N))
    Gc = G00
    trAL[:, 0] = tr_A(Gc, gamL)
    for m in range(0, N - 1):
        Gc = -_mm(xtil[m], Gc)
        trAL[:, m + 1] = tr_A(Gc, gamL)
    # ---------------- lead k = N-1 (step 3: upwards from the diagonal)
    trAR = np.empty((K, N))
    Gc = GNN
    trAR[:, N - 1] = tr_A(Gc, gamR)
    for m in range(N - 1, 0, -1):
        Gc = -_mm(ytil[m], Gc)
        trAR[:, m - 1] = tr_A(Gc, gamR)
    G0N = Gc                                   # G_(0,N-1)
    Tm = np.einsum("kab,kbc,kcd,kad->k", gamL, G0N, gamR, G0N.conj()).real
    return trG, trAL, trAR, Tm


def _sigmas(z, U, coup_even, coup_odd, n, lead_kind, sr_tol, sr_maxit):
    N = U.shape[0]
    if lead_kind == 0:
        (tauL, t1L), (tauR, t1R) = se.scalar_lead_bonds(coup_even, coup_odd, N)
        sL = se.sigma_scalar(z, U[0], float(tauL), float(t1L)).reshape(-1, 1, 1)
        sR = se.sigma_scalar(z, U[-1], float(tauR), float(t1R)).reshape(-1, 1, 1)
        return sL, sR
    sL, sR, _ = se.sigma_block(z, np.asarray(coup_even).reshape(n, n),
                               np.asarray(coup_odd).reshape(n, n), N, U[0], U[-1],
                               sr_tol, sr_maxit)
    return sL, sR


def chain_charge(U, coup_even, coup_odd, n, z_eq, w_eq, z_neq, w_neq, mu_s, mu_d, kT,
                 lead_kind=0, sr_tol=1e-12, sr_maxit=200, chunk=64):
    """Per-ring charge (no deg / mode weight) and T(E) of one chain / channel via
    Algorithms 1-2, energies processed ``chunk`` at a time (eq.(4))."""
    U = np.asarray(U, dtype=np.float64)
    N = U.shape[0]
    n_ring = np.zeros(N)
    T = np.zeros(len(z_neq))
    for s in range(0, len(z_eq), chunk):
        zz = z_eq[s:s + chunk]
        sL, sR = _sigmas(zz, U, coup_even, coup_odd, n, lead_kind, sr_tol, sr_maxit)
        trG, _, _, _ = chain_rgf(U, coup_even, coup_odd, n, zz, sL, sR)
        n_ring += (-1.0 / np.pi) * (w_eq[s:s + chunk, None] * trG).imag.sum(axis=0)
    for s in range(0, len(z_neq), chunk):
        zz = z_neq[s:s + chunk]
        sL, sR = _sigmas(zz, U, coup_even, coup_odd, n, lead_kind, sr_tol, sr_maxit)
        _, trAL, trAR, Tm = chain_rgf(U, coup_even, coup_odd, n, zz, sL, sR)
        fS = fermi_real(zz.real, mu_s, kT)[:, None]
        fD = fermi_real(zz.real, mu_d, kT)[:, None]
        w = w_neq[s:s + chunk, None] / (2.0 * np.pi)
        n_ring += (w * (fS * trAL + fD * trAR)).sum(axis=0)
        T[s:s + chunk] = Tm
    return n_ring, T


def charge_and_transmission(wl, channels=None, chunk=64):
    """Tier O3 for a whole workload: returns (n[C, N], T[C, K_neq])."""
    chans = range(wl.C) if channels is None else channels
    n_out = np.zeros((wl.C, wl.N))
    T_out = np.zeros((wl.C, wl.K_neq))
    for c in chans:
        U = -wl.phi[c]
        if wl.kind == "scalar":
            for j in range(wl.n_modes):
                nr, T = chain_charge(U, wl.coup_even[j:j + 1], wl.coup_odd[j:j + 1], 1,
                                     wl.z_eq, wl.w_eq, wl.z_neq, wl.w_neq,
                                     wl.mu_s, wl.mu_d, wl.kT, 0, chunk=max(chunk, 4096))
                n_out[c] += wl.deg * wl.mode_weight[j] * nr
                T_out[c] += wl.mode_weight[j] * T
        else:
            nr, T = chain_charge(U, wl.coup_even, wl.coup_odd, wl.n,
                                 wl.z_eq, wl.w_eq, wl.z_neq, wl.w_neq,
                                 wl.mu_s, wl.mu_d, wl.kT, 1, wl.sr_tol, wl.sr_maxit, chunk)
            n_out[c] += wl.deg * nr
            T_out[c] += T
    return n_out, T_out
