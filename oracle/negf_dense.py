"""Tier O1 oracle: NEGF charge and transmission *by definition* (dense inversion).

TEST INFRASTRUCTURE ONLY (see oracle/__init__.py).  Shares no code with the CUDA
path.  For fixed inputs the recursive Green's function method reaches exactly
the result of a dense inversion, so the oracle is the plain definition:

  G^R(E) = [(E + i eta) I - H - Sigma_L - Sigma_R]^-1               eq.(2)
  Gamma_l = i (Sigma_l - Sigma_l^dagger),  A_l = G^R Gamma_l G^R^dagger
  rho = (1/pi) Im[ int^{E_min} G^R F_min dE ] - (1/2pi) int_{E_min}^{E_max} sum_l A_l F_l dE
                                                                     eq.(4)
  T_pq(E) = Tr[Gamma_p G^R Gamma_q G^R^dagger]                      eq.(5)

Output convention (reading R12): n_i = electrons per ring >= 0, i.e.
minus the paper's rho, times the degeneracy ``deg``:
  n_i = deg * [ -(1/pi) Im sum_k W_k Tr_ring G_ii(z_k)
                + (1/2pi) sum_k w_k ( f_S(E_k) Tr_ring A_L,ii + f_D(E_k) Tr_ring A_R,ii ) ]
summed over modes with ``mode_weight`` (scalar chains).  H has diagonal
U_i = -phi_i and off-diagonal blocks H_{i,i+1} = coup_even / coup_odd
for even / odd i, H_{i+1,i} = H_{i,i+1}^dagger.
"""
from __future__ import annotations

import numpy as np

from . import selfenergy as se


def fermi_real(E, mu, kT):
    """F_l(E) = 1/(1 + exp((E - mu_l)/kT)), real E."""
    x = (np.asarray(E, dtype=np.float64) - mu) / kT
    e = np.exp(-np.abs(x))                       # never overflows
    return np.where(x > 0, e / (1.0 + e), 1.0 / (1.0 + e))


def build_hamiltonian(U, coup_even, coup_odd, n: int):
    """Dense block-tridiagonal H of dimension N*n (Fig.1(a))."""
    N = U.shape[0]
    D = N * n
    H = np.zeros((D, D), dtype=np.complex128)
    ce = np.asarray(coup_even, dtype=np.complex128).reshape(n, n)
    co = np.asarray(coup_odd, dtype=np.complex128).reshape(n, n)
    for i in range(N):
        H[i * n:(i + 1) * n, i * n:(i + 1) * n] = U[i] * np.eye(n)
        if i + 1 < N:
            B = ce if i % 2 == 0 else co
            H[i * n:(i + 1) * n, (i + 1) * n:(i + 2) * n] = B
            H[(i + 1) * n:(i + 2) * n, i * n:(i + 1) * n] = B.conj().T
    return H


def _self_energies(z, U, coup_even, coup_odd, n, lead_kind, sr_tol, sr_maxit):
    """Sigma_L(z), Sigma_R(z) of shape (K, n, n) for one chain / channel."""
    N = U.shape[0]
    z = np.asarray(z, dtype=np.complex128)
    if lead_kind == 0:
        assert n == 1
        (tauL, t1L), (tauR, t1R) = se.scalar_lead_bonds(coup_even, coup_odd, N)
        sL = se.sigma_scalar(z, U[0], float(tauL), float(t1L))
        sR = se.sigma_scalar(z, U[-1], float(tauR), float(t1R))
        return sL.reshape(-1, 1, 1), sR.reshape(-1, 1, 1), np.zeros(z.shape[0], np.int64)
    sL, sR, it = se.sigma_block(z, np.asarray(coup_even).reshape(n, n),
                                np.asarray(coup_odd).reshape(n, n), N, U[0], U[-1],
                                sr_tol, sr_maxit)
    return sL, sR, it


def chain_dense(U, coup_even, coup_odd, n, z_eq, w_eq, z_neq, w_neq,
                mu_s, mu_d, kT, lead_kind=0, sr_tol=1e-12, sr_maxit=200):
    """Charge per ring (without deg / mode weight) and T(E) of ONE chain or ONE
    real-space channel, by dense inversion.  Returns (n_ring (N,), T (K_neq,),
    details dict)."""
    U = np.asarray(U, dtype=np.float64)
    N = U.shape[0]
    D = N * n
    H = build_hamiltonian(U, coup_even, coup_odd, n)
    eye = np.eye(D, dtype=np.complex128)
    n_ring = np.zeros(N)
    T = np.zeros(len(z_neq))

    # ---- contour part: -(1/pi) Im sum_k W_k Tr_ring G_ii(z_k)      (eq.(4), first term)
    if len(z_eq):
        sL, sR, _ = _self_energies(z_eq, U, coup_even, coup_odd, n, lead_kind, sr_tol, sr_maxit)
        for k, z in enumerate(z_eq):
            M = z * eye - H
            M[:n, :n] -= sL[k]
            M[D - n:, D - n:] -= sR[k]
            G = np.linalg.inv(M)
            tr = np.diagonal(G).reshape(N, n).sum(axis=1)
            n_ring += (-1.0 / np.pi) * (w_eq[k] * tr).imag

    # ---- real-axis part: (1/2pi) sum_k w_k (f_S A_L,ii + f_D A_R,ii)   (eq.(4), second term)
    if len(z_neq):
        sL, sR, _ = _self_energies(z_neq, U, coup_even, coup_odd, n, lead_kind, sr_tol, sr_maxit)
        fS = fermi_real(z_neq.real, mu_s, kT)
        fD = fermi_real(z_neq.real, mu_d, kT)
        for k, z in enumerate(z_neq):
            M = z * eye - H
            M[:n, :n] -= sL[k]
            M[D - n:, D - n:] -= sR[k]
            G = np.linalg.inv(M)
            gamL = 1j * (sL[k] - sL[k].conj().T)
            gamR = 1j * (sR[k] - sR[k].conj().T)
            GL = G[:, :n]                 # the only columns Gamma_L (block (0,0)) touches
            GR = G[:, D - n:]             # likewise Gamma_R (block (N-1,N-1))
            AL = np.einsum("ia,ab,ib->i", GL, gamL, GL.conj()).real   # diag(G Gamma_L G^dagger)
            AR = np.einsum("ia,ab,ib->i", GR, gamR, GR.conj()).real
            n_ring += (w_neq[k] / (2.0 * np.pi)) * (
                fS[k] * AL.reshape(N, n).sum(axis=1) + fD[k] * AR.reshape(N, n).sum(axis=1))
            G0N = G[:n, D - n:]
            T[k] = np.trace(gamL @ G0N @ gamR @ G0N.conj().T).real
    return n_ring, T


def charge_and_transmission(wl, channels=None):
    """Tier O1 for a whole workload: returns (n[C, N], T[C, K_neq])."""
    C = wl.C
    chans = range(C) if channels is None else channels
    n_out = np.zeros((C, wl.N))
    T_out = np.zeros((C, wl.K_neq))
    for c in chans:
        U = -wl.phi[c]
        if wl.kind == "scalar":
            for j in range(wl.n_modes):
                nr, T = chain_dense(U, wl.coup_even[j:j + 1], wl.coup_odd[j:j + 1], 1,
                                    wl.z_eq, wl.w_eq, wl.z_neq, wl.w_neq,
                                    wl.mu_s, wl.mu_d, wl.kT, 0)
                n_out[c] += wl.deg * wl.mode_weight[j] * nr
                T_out[c] += wl.mode_weight[j] * T
        else:
            nr, T = chain_dense(U, wl.coup_even, wl.coup_odd, wl.n,
                                wl.z_eq, wl.w_eq, wl.z_neq, wl.w_neq,
                                wl.mu_s, wl.mu_d, wl.kT, 1, wl.sr_tol, wl.sr_maxit)
            n_out[c] += wl.deg * nr
            T_out[c] += T
    return n_out, T_out


def green_dense(U, coup_even, coup_odd, n, z, lead_kind=0, sr_tol=1e-12, sr_maxit=200):
    """Full G^R(z), Sigma_L, Sigma_R at a single z (for identity / invariant tests)."""
    U = np.asarray(U, dtype=np.float64)
    N = U.shape[0]
    D = N * n
    H = build_hamiltonian(U, coup_even, coup_odd, n)
    sL, sR, _ = _self_energies(np.array([z]), U, coup_even, coup_odd, n, lead_kind,
                               sr_tol, sr_maxit)
    M = z * np.eye(D, dtype=np.complex128) - H
    M[:n, :n] -= sL[0]
    M[D - n:, D - n:] -= sR[0]
    return np.linalg.inv(M), sL[0], sR[0]


def landauer_dense(wl, channels=None):
    """Lead currents and zero-bias conductance BY DEFINITION (eq.(5)-(6)), from the
    dense Green's function -- not from T(E):

      I_l = (g_s e/h) int Tr[ F_l Gamma_l A + i Gamma_l G^< ] dE,   A = sum_l A_l,  G^< = i sum_l A_l F_l
      G   = G_0 int T(E) (-dF/dE) dE,   T = Tr[Gamma_S G^R Gamma_D G^R^dagger],  F = F(E - mu_S, kT)

    on the real-axis nodes / weights of the workload.  Returns (I_S[C], I_D[C], G[C]) with the
    currents in eV (multiply by g_s e/h) and G in units of G_0; scalar chains are summed over modes
    with ``mode_weight``.  For two leads the integrand of I_S reduces algebraically to
    T_SD (F_S - F_D); this function does not use that."""
    chans = range(wl.C) if channels is None else channels
    I_S = np.zeros(wl.C)
    I_D = np.zeros(wl.C)
    G = np.zeros(wl.C)
    E = wl.z_neq.real
    fS = fermi_real(E, wl.mu_s, wl.kT)
    fD = fermi_real(E, wl.mu_d, wl.kT)
    dfdE = fS * (1.0 - fS) / wl.kT                      # -dF/dE of the source Fermi function
    for c in chans:
        U = -wl.phi[c]
        units = ([(wl.coup_even[j:j + 1], wl.coup_odd[j:j + 1], 1, 0, wl.mode_weight[j])
                  for j in range(wl.n_modes)] if wl.kind == "scalar"
                 else [(wl.coup_even, wl.coup_odd, wl.n, 1, 1.0)])
        for ce, co, n, lead_kind, wgt in units:
            N = U.shape[0]
            D = N * n
            for k, z in enumerate(wl.z_neq):
                Gr, sL, sR = green_dense(U, ce, co, n, z, lead_kind, wl.sr_tol, wl.sr_maxit)
                gamL = np.zeros((D, D), dtype=np.complex128)
                gamR = np.zeros((D, D), dtype=np.complex128)
                gamL[:n, :n] = 1j * (sL - sL.conj().T)
                gamR[D - n:, D - n:] = 1j * (sR - sR.conj().T)
                AL = Gr @ gamL @ Gr.conj().T
                AR = Gr @ gamR @ Gr.conj().T
                A = AL + AR
                Gless = 1j * (AL * fS[k] + AR * fD[k])
                iS = np.trace(fS[k] * gamL @ A + 1j * gamL @ Gless).real
                iD = np.trace(fD[k] * gamR @ A + 1j * gamR @ Gless).real
                T = np.trace(gamL @ Gr @ gamR @ Gr.conj().T).real
                I_S[c] += wgt * wl.w_neq[k] * iS
                I_D[c] += wgt * wl.w_neq[k] * iD
                G[c] += wgt * wl.w_neq[k] * T * dfdE[k]
    return I_S, I_D, G


def integrand_dense(wl, ring: int, channels=None):
    """The integrand of the second term of eq.(4) at one ring as a function of energy (PAPER.md:353,
    "the integrand A_1 F_1 + A_2 F_2 at the center of the channel"), by the definition:
      I_c(E_k) = sum_modes mode_weight (F_S Tr_ring A_S,(r,r) + F_D Tr_ring A_D,(r,r))(E_k),
    A_l = G^R Gamma_l G^R^dagger from the dense inverse.  Returns I[C, K_neq]."""
    chans = range(wl.C) if channels is None else channels
    out = np.zeros((wl.C, wl.K_neq))
    fS = fermi_real(wl.z_neq.real, wl.mu_s, wl.kT)
    fD = fermi_real(wl.z_neq.real, wl.mu_d, wl.kT)
    for c in chans:
        U = -wl.phi[c]
        units = ([(wl.coup_even[j:j + 1], wl.coup_odd[j:j + 1], 1, 0, wl.mode_weight[j])
                  for j in range(wl.n_modes)] if wl.kind == "scalar"
                 else [(wl.coup_even, wl.coup_odd, wl.n, 1, 1.0)])
        for ce, co, n, lead_kind, wgt in units:
            D = U.shape[0] * n
            rows = slice(ring * n, (ring + 1) * n)
            for k, z in enumerate(wl.z_neq):
                Gr, sL, sR = green_dense(U, ce, co, n, z, lead_kind, wl.sr_tol, wl.sr_maxit)
                gamL = 1j * (sL - sL.conj().T)
                gamR = 1j * (sR - sR.conj().T)
                GL = Gr[rows, :n]
                GR = Gr[rows, D - n:]
                aL = np.trace(GL @ gamL @ GL.conj().T).real
                aR = np.trace(GR @ gamR @ GR.conj().T).real
                out[c, k] += wgt * (fS[k] * aL + fD[k] * aR)
    return out
