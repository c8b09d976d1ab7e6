"""Tier O3 oracle, C++17/OpenMP edition: loader and array marshalling for negf_rgf_omp.cpp.

TEST INFRASTRUCTURE ONLY (see oracle/__init__.py).  The arithmetic lives in
``negf_rgf_omp.cpp`` (the paper's Algorithm 2 + Algorithm 1, one energy point per
thread, with its own Sancho-Rubio / closed-form self-energies); this module compiles
it with g++ for the host it runs on and passes plain arrays.  Nothing here or there is
shared with, or linked into, the CUDA library.

The shared object is built lazily, per host CPU (``-march=native``: the file name
carries a hash of the CPU flags, so an object built in one container is never loaded
on a different CPU), under ``oracle/_build/`` (git-ignored).
"""
from __future__ import annotations

import ctypes as C
import hashlib
import os
import subprocess

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "negf_rgf_omp.cpp")
OUT_DIR = os.path.join(HERE, "_build")
CXXFLAGS = ["-O3", "-march=native", "-std=c++17", "-fopenmp", "-fPIC", "-shared"]

_lib = None


def _host_tag() -> str:
    h = hashlib.sha256()
    try:
        with open("/proc/cpuinfo") as fh:
            for line in fh:
                if line.startswith("flags") or line.startswith("model name"):
                    h.update(line.encode())
                    if line.startswith("flags"):
                        break
    except OSError:
        pass
    with open(SRC, "rb") as fh:
        h.update(fh.read())
    h.update(" ".join(CXXFLAGS).encode())
    return h.hexdigest()[:12]


def build(verbose: bool = False) -> str:
    """Compile negf_rgf_omp.cpp for this host (no-op if already built); returns the path."""
    os.makedirs(OUT_DIR, exist_ok=True)
    path = os.path.join(OUT_DIR, f"libnegf_o3_{_host_tag()}.so")
    if os.path.exists(path):
        return path
    tmp = path + f".tmp{os.getpid()}"
    cmd = ["g++", *CXXFLAGS, SRC, "-o", tmp]
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError(f"g++ failed for {SRC}:\n{r.stdout}\n{r.stderr}")
    os.replace(tmp, path)
    if verbose:
        print("built", path)
    return path


def load() -> C.CDLL:
    global _lib
    if _lib is None:
        lib = C.CDLL(build())
        dp, ip = C.POINTER(C.c_double), C.POINTER(C.c_int)
        lib.o3_chain_charge.restype = C.c_int
        lib.o3_chain_charge.argtypes = [C.c_int, C.c_int, dp, dp, dp, C.c_int, dp, dp, C.c_int, dp, dp,
                                        C.c_double, C.c_double, C.c_double, C.c_int, C.c_double, C.c_int,
                                        C.c_int, dp, dp, ip, dp]
        lib.o3_max_threads.restype = C.c_int
        _lib = lib
    return _lib


def max_threads() -> int:
    return int(load().o3_max_threads())


def _dp(a):
    return a.ctypes.data_as(C.POINTER(C.c_double)) if a is not None and a.size else None


def chain_charge(U, coup_even, coup_odd, n, z_eq, w_eq, z_neq, w_neq, mu_s, mu_d, kT,
                 lead_kind=0, sr_tol=1e-12, sr_maxit=200, threads=0, want_sigma=False):
    """Per-ring charge (no deg / mode weight) and T(E) of one chain / channel.

    Same contract as ``oracle.negf_rgf.chain_charge``.  Returns (n_ring[N], T[K_neq]) and, with
    ``want_sigma``, also Sigma[K_eq + K_neq, 2, n, n] (contour points first).
    """
    lib = load()
    U = np.ascontiguousarray(U, dtype=np.float64)
    N = U.shape[0]
    ce = np.ascontiguousarray(np.asarray(coup_even, dtype=np.complex128).reshape(n, n))
    co = np.ascontiguousarray(np.asarray(coup_odd, dtype=np.complex128).reshape(n, n))
    ze = np.ascontiguousarray(z_eq, dtype=np.complex128).reshape(-1)
    we = np.ascontiguousarray(w_eq, dtype=np.complex128).reshape(-1)
    zn = np.ascontiguousarray(z_neq, dtype=np.complex128).reshape(-1)
    wn = np.ascontiguousarray(w_neq, dtype=np.float64).reshape(-1)
    n_ring = np.zeros(N)
    T = np.zeros(max(len(zn), 1))
    its = C.c_int(0)
    sig = np.zeros((len(ze) + len(zn), 2, n, n), dtype=np.complex128) if want_sigma else None
    rc = lib.o3_chain_charge(N, n, _dp(U), _dp(ce.view(np.float64)), _dp(co.view(np.float64)),
                             len(ze), _dp(ze.view(np.float64)), _dp(we.view(np.float64)),
                             len(zn), _dp(zn.view(np.float64)), _dp(wn),
                             float(mu_s), float(mu_d), float(kT), int(lead_kind), float(sr_tol),
                             int(sr_maxit), int(threads), _dp(n_ring), _dp(T), C.byref(its),
                             _dp(sig.view(np.float64)) if want_sigma else None)
    if rc != 0:
        raise ValueError("o3_chain_charge: bad arguments")
    T = T[:len(zn)]
    if want_sigma:
        return n_ring, T, sig
    return n_ring, T


def charge_and_transmission(wl, channels=None, threads=0):
    """Tier O3 (C++/OpenMP) for a whole workload: returns (n[C, N], T[C, K_neq])."""
    chans = range(wl.C) if channels is None else channels
    n_out = np.zeros((wl.C, wl.N))
    T_out = np.zeros((wl.C, wl.K_neq))
    for c in chans:
        U = -wl.phi[c]
        if wl.kind == "scalar":
            for j in range(wl.n_modes):
                nr, T = chain_charge(U, wl.coup_even[j:j + 1], wl.coup_odd[j:j + 1], 1,
                                     wl.z_eq, wl.w_eq, wl.z_neq, wl.w_neq, wl.mu_s, wl.mu_d, wl.kT,
                                     0, threads=threads)
                n_out[c] += wl.deg * wl.mode_weight[j] * nr
                T_out[c] += wl.mode_weight[j] * T
        else:
            nr, T = chain_charge(U, wl.coup_even, wl.coup_odd, wl.n, wl.z_eq, wl.w_eq, wl.z_neq,
                                 wl.w_neq, wl.mu_s, wl.mu_d, wl.kT, 1, wl.sr_tol, wl.sr_maxit,
                                 threads=threads)
            n_out[c] += wl.deg * nr
            T_out[c] += T
    return n_out, T_out
