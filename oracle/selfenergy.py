"""Lead self-energies, CPU oracle (test infrastructure only -- see oracle/__init__.py).

Sigma_l^R = tau_l^dagger g_l^R tau_l (eq.(2)).  The paper computes
the surface Green's function g either "using a decimation technique [33,34]" or
from "an analytical expression ... (e.g. for CNTs [23])".  The
analytic formula is not printed; it is derived below (reading R8).

Lead geometry (readings R7, R9): each lead is the semi-infinite
continuation of the device's alternating coupling pattern -- the bond between
rings j and j+1 is ``coup_even`` for even j and ``coup_odd`` for odd j, for every
integer j -- with a uniform on-site energy equal to the adjacent end ring's U.
"""
from __future__ import annotations

import numpy as np


# --------------------------------------------------------------------------- scalar chains

def surface_gf_alternating(z, t1, t2):
    """Retarded surface Green's function of a semi-infinite chain with zero
    on-site energy whose bonds alternate t1, t2, t1, ... starting from the surface
    site (t1 = bond from the surface site into the lead).

    Continued fraction:  g = 1/(z - t1^2 g'),  g' = 1/(z - t2^2 g)
      =>  z t2^2 g^2 - (z^2 - t1^2 + t2^2) g + z = 0.
    With X = z^2 - t1^2 + t2^2 the discriminant factorises,
      S^2 = X^2 - 4 z^2 t2^2 = (z-(a+b)) (z-(a-b)) (z-(b-a)) (z+(a+b)),  a=|t1|, b=|t2|,
    and taking the principal square root of each factor gives the branch with
    S -> z^2 for |z| -> infinity in the upper half plane, i.e. the retarded root
      g = (X - S)/(2 z t2^2) = 2 z/(X + S),     Im g <= 0.
    The two forms are algebraically equal; the one that does not cancel is used.
    For t1 = t2 = t this is g = (z - sqrt(z-2|t|) sqrt(z+2|t|))/(2 t^2), the 1D
    closed form quoted in BASELINE.json (north_star).
    """
    z = np.asarray(z, dtype=np.complex128)
    a = abs(t1)
    b = abs(t2)
    X = z * z + (b - a) * (b + a)        # not z*z - a*a + b*b: that cancels when |z| << a ~ b
    S = (np.sqrt(z - (a + b)) * np.sqrt(z - (a - b))
         * np.sqrt(z - (b - a)) * np.sqrt(z + (a + b)))
    same_side = (X.real * S.real + X.imag * S.imag) >= 0.0   # Re(conj(X) S) >= 0
    with np.errstate(divide="ignore", invalid="ignore"):
        g_sum = 2.0 * z / (X + S)
        g_dif = (X - S) / (2.0 * z * b * b)
    return np.where(same_side, g_sum, g_dif)


def scalar_lead_bonds(coup_even, coup_odd, N: int):
    """|bond| magnitudes (tau, t1) for the left and right lead of an N-ring chain.

    Bond (j, j+1) is even-type for even j.  Left lead: rings -1, -2, ...; the
    device-lead bond is (-1, 0) (odd type) and the first bond inside the lead is
    (-2, -1) (even type).  Right lead: rings N, N+1, ...; device-lead bond
    (N-1, N) has the type of N-1, the first interior bond (N, N+1) the type of N.
    Returns ((tauL, t1L), (tauR, t1R)).
    """
    even = float(np.abs(np.asarray(coup_even)).reshape(-1)[0])
    odd = float(np.abs(np.asarray(coup_odd)).reshape(-1)[0])
    left = (odd, even)
    right = (odd, even) if (N - 1) % 2 == 1 else (even, odd)
    return left, right


def sigma_scalar(z, U_end, tau, t1):
    """Sigma(z) = |tau|^2 g(z - U_end) for a scalar chain whose lead has bonds
    t1 (first interior), t2 = tau (by alternation), on-site U_end."""
    g = surface_gf_alternating(np.asarray(z) - U_end, t1, tau)
    return (abs(tau) ** 2) * g


# --------------------------------------------------------------------------- dense blocks

def sancho_rubio(z, H00, H01, tol: float = 1e-12, maxit: int = 200, extra: int = 1,
                 polish: int = 2):
    """Surface Green's function of a semi-infinite stack of principal layers by
    decimation (refs [33,34] of the paper; reading R10).

    Layers p = 0, 1, 2, ... with on-site block H00 and H_{p,p+1} = H01.
      eps_s = eps = H00, a = H01, b = H01^dagger
      repeat: g = (z - eps)^-1
              eps_s += a g b ;  eps += a g b + b g a ;  a <- a g a ;  b <- b g b
      until max|a|, max|b| < tol (then ``extra`` more iterations);
      g_surf = (z - eps_s)^-1.
    ``z`` may be an array of K energies; the result has shape (K, m, m).  Returns
    (g_surf, iterations used per energy).

    The decimation inverts z - eps of isolated 2^k-layer segments, which is ill
    conditioned whenever z lies within rounding-amplified reach of one of their
    real-axis poles: at eta = 1e-6 the raw result carries errors of 1e-13 (typical)
    to 2e-8 (next to a pole of the isolated layer) against the closed form.  Reading
    R10 asks for the converged surface Green's function, so the decimation result is
    then polished with ``polish`` Newton steps on the property that DEFINES it --
    adding one more layer to a semi-infinite stack leaves it unchanged,
        g = [z - H00 - H01 g H01^dagger]^-1
    (see ``polish_surface_gf``), after which the fixed-point residual is at rounding
    level for every z.
    """
    z = np.atleast_1d(np.asarray(z, dtype=np.complex128))
    K = z.shape[0]
    m = H00.shape[0]
    eye = np.eye(m, dtype=np.complex128)
    zI = z[:, None, None] * eye
    eps_s = np.broadcast_to(H00.astype(np.complex128), (K, m, m)).copy()
    eps = eps_s.copy()
    a = np.broadcast_to(H01.astype(np.complex128), (K, m, m)).copy()
    b = np.broadcast_to(H01.conj().T.astype(np.complex128), (K, m, m)).copy()
    iters = np.zeros(K, dtype=np.int64)
    done = np.zeros(K, dtype=bool)
    remaining = np.full(K, -1, dtype=np.int64)   # -1: criterion not met yet; else extra iterations to go
    for _ in range(maxit):
        active = ~done
        if not active.any():
            break
        g = np.linalg.inv(zI[active] - eps[active])
        agb = a[active] @ g @ b[active]
        bga = b[active] @ g @ a[active]
        eps_s[active] += agb
        eps[active] += agb + bga
        a[active] = a[active] @ g @ a[active]
        b[active] = b[active] @ g @ b[active]
        iters[active] += 1
        conv = np.maximum(np.abs(a).max(axis=(1, 2)), np.abs(b).max(axis=(1, 2))) < tol
        # an energy is finished once it has met the criterion and done its extra iterations
        newly = active & (remaining < 0) & conv
        cont = active & (remaining > 0)
        remaining[cont] -= 1
        remaining[newly] = extra
        done |= active & (remaining == 0)
    # energies that never met the criterion are reported through ``iters == maxit``
    g_surf = np.linalg.inv(zI - eps_s)
    for _ in range(polish):
        g_surf = polish_surface_gf(z, H00, H01, g_surf)
    return g_surf, iters


def polish_surface_gf(z, H00, H01, g):
    """One Newton step on  F(g) = [z - H00 - H01 g H01^dagger]^-1 - g = 0,  the defining
    fixed-point property of the surface Green's function of a semi-infinite stack
    (refs [33,34]).

    Only the block X = g[S, S] enters H01 g H01^dagger, S = the columns in which H01 is
    non-zero (the surface ring for the two-ring layers of ``block_lead_layers``), so the
    unknown is X:  with B = H01[:, S],  G(X) = [z - H00 - B X B^dagger]^-1,
        dG[S, S] = P dX Q,   P = G[S, :] B,   Q = B^dagger G[:, S],
    and the Newton correction solves  dX - P dX Q = G[S, S] - X  as a dense
    |S|^2 x |S|^2 linear system (row-major vec: vec(P dX Q) = (P kron Q^T) vec(dX)).
    Returns G(X + dX), the whole layer's surface Green's function.
    """
    z = np.atleast_1d(np.asarray(z, dtype=np.complex128))
    m = H00.shape[0]
    S = np.nonzero(np.abs(H01).sum(axis=0) > 0)[0]
    ns = S.shape[0]
    B = H01[:, S].astype(np.complex128)
    Bd = B.conj().T
    eye = np.eye(m, dtype=np.complex128)
    out = np.empty_like(g)
    for k in range(z.shape[0]):
        X = g[k][np.ix_(S, S)]
        G = np.linalg.inv(z[k] * eye - H00 - B @ X @ Bd)
        P = G[S, :] @ B
        Q = Bd @ G[:, S]
        A = np.eye(ns * ns, dtype=np.complex128) - np.kron(P, Q.T)
        dX = np.linalg.solve(A, (G[np.ix_(S, S)] - X).reshape(-1)).reshape(ns, ns)
        out[k] = np.linalg.inv(z[k] * eye - H00 - B @ (X + dX) @ Bd)
    return out


def block_lead_layers(coup_even, coup_odd, N: int, U_left: float, U_right: float):
    """Principal layers (two rings each) of the left and right lead.

    Left lead, layer p = rings (-1-2p, -2-2p):
        H00 = [[U, H_{-1,-2}], [H_{-2,-1}, U]],  H_{-2,-1} = coup_even (j=-2 even)
        H01 = [[0, 0], [H_{-2,-3}, 0]],          H_{-2,-3} = coup_odd^dagger (j=-3 odd)
        tau = H_{-1,0} = coup_odd;   Sigma_L = tau^dagger g tau        (eq.(2))
    Right lead, layer p = rings (N+2p, N+1+2p):
        H00 = [[U, H_{N,N+1}], [H_{N,N+1}^dagger, U]],  H01 = [[0,0],[H_{N+1,N+2},0]]
        tau' = H_{N,N-1} = H_{N-1,N}^dagger;  Sigma_R = tau'^dagger g tau'
    The surface ring is the first n rows/columns of each layer.
    Returns dict(left=(H00, H01, tau), right=(H00, H01, tau')).
    """
    ce = np.asarray(coup_even, dtype=np.complex128)
    co = np.asarray(coup_odd, dtype=np.complex128)
    n = ce.shape[0]
    Z = np.zeros((n, n), dtype=np.complex128)
    eye = np.eye(n, dtype=np.complex128)

    def bond(j):          # H_{j,j+1}
        return ce if j % 2 == 0 else co

    # left
    H00L = np.block([[U_left * eye, bond(-2).conj().T], [bond(-2), U_left * eye]])
    H01L = np.block([[Z, Z], [bond(-3).conj().T, Z]])
    tauL = bond(-1)                       # H_{-1,0}
    # right
    H00R = np.block([[U_right * eye, bond(N)], [bond(N).conj().T, U_right * eye]])
    H01R = np.block([[Z, Z], [bond(N + 1), Z]])
    tauR = bond(N - 1).conj().T           # H_{N,N-1}
    return {"left": (H00L, H01L, tauL), "right": (H00R, H01R, tauR)}


def sigma_block(z, coup_even, coup_odd, N: int, U_left: float, U_right: float,
                tol: float = 1e-12, maxit: int = 200, extra: int = 1):
    """(Sigma_L, Sigma_R, iterations) for K energies, each Sigma of shape (K, n, n)."""
    layers = block_lead_layers(coup_even, coup_odd, N, U_left, U_right)
    n = np.asarray(coup_even).shape[0]
    out = []
    its = []
    for side in ("left", "right"):
        H00, H01, tau = layers[side]
        g, it = sancho_rubio(z, H00, H01, tol, maxit, extra)
        gs = g[:, :n, :n]
        out.append(tau.conj().T @ gs @ tau)
        its.append(it)
    return out[0], out[1], np.maximum(its[0], its[1])
