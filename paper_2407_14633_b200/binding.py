"""ctypes binding of libnegf_b200.so -- argument marshalling only.

Every function here has the name and the arguments of its C-ABI counterpart in
``include/negf.h``; all arithmetic of the method runs in the CUDA kernels behind
that boundary.  PyTorch appears only as the owner of device memory and of the
CUDA stream.  There is no CPU fallback: if the library is missing, loading
raises; if there is no GPU, ``negf_create`` returns NEGF_ECUDA and this module
raises ``NegfError``.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libnegf_b200.so")

NEGF_OK, NEGF_EINVAL, NEGF_ENOMEM, NEGF_ECUDA, NEGF_ENOCONV, NEGF_ESTATE = range(6)
STATUS_NAMES = {0: "NEGF_OK", 1: "NEGF_EINVAL", 2: "NEGF_ENOMEM", 3: "NEGF_ECUDA",
                4: "NEGF_ENOCONV", 5: "NEGF_ESTATE"}

# every symbol include/negf.h declares (tests check the library exports all of them)
EXPORTED_SYMBOLS = [
    "negf_create", "negf_destroy", "negf_set_potential", "negf_charge", "negf_transmission",
    "negf_self_energy", "negf_current", "negf_set_probe", "negf_integrand_peak", "negf_solve_host", "negf_sync",
    "negf_kernel_stats", "negf_get_plan",
    "broyden_create", "broyden_step", "broyden_reset", "broyden_destroy", "broyden_residual_noalloc",
    "negf_fp64_peak", "negf_last_error", "negf_version",
]


class NegfError(RuntimeError):
    def __init__(self, status: int, where: str, text: str):
        self.status = status
        super().__init__(f"{where}: {STATUS_NAMES.get(status, status)}: {text}")


class negf_c64(C.Structure):
    _fields_ = [("re", C.c_double), ("im", C.c_double)]


class negf_config(C.Structure):
    _fields_ = [
        ("n_channels", C.c_int32), ("n_rings", C.c_int32), ("block", C.c_int32),
        ("n_modes", C.c_int32), ("lead_kind", C.c_int32), ("sr_maxit", C.c_int32),
        ("sr_tol", C.c_double), ("mu_s", C.c_double), ("mu_d", C.c_double), ("kT", C.c_double),
        ("deg", C.c_double),
        ("coup_even", C.c_void_p), ("coup_odd", C.c_void_p), ("mode_weight", C.c_void_p),
        ("n_eq", C.c_int32), ("z_eq", C.c_void_p), ("w_eq", C.c_void_p),
        ("n_neq", C.c_int32), ("z_neq", C.c_void_p), ("w_neq", C.c_void_p),
        ("workspace_bytes", C.c_int64), ("profile", C.c_int32), ("reserved", C.c_int32),
        ("pivot_theta", C.c_double),
    ]


class negf_kernel_stat(C.Structure):
    _fields_ = [("name", C.c_char * 48), ("launches", C.c_int64), ("total_ms", C.c_double)]


class negf_plan_info(C.Structure):
    _fields_ = [("history_bytes", C.c_int64), ("partial_bytes", C.c_int64),
                ("n_batches", C.c_int32), ("sweeps_per_charge", C.c_int32),
                ("max_sr_iterations", C.c_int32), ("kernel_launches", C.c_int32),
                ("sr_passes_total", C.c_int64)]


_lib = None


def load_library(path: Optional[str] = None) -> C.CDLL:
    """dlopen libnegf_b200.so (built in-tree by ``paper_2407_14633_b200.build``)."""
    global _lib
    if _lib is not None and path is None:
        return _lib
    p = path or LIB_PATH
    if not os.path.exists(p):
        raise FileNotFoundError(
            f"{p} not found: build it with `python -m paper_2407_14633_b200.build` "
            "(there is no CPU fallback)")
    lib = C.CDLL(p)
    vp, i32, i64, dbl = C.c_void_p, C.c_int32, C.c_int64, C.c_double
    sig = {
        "negf_create": (C.c_int, [C.POINTER(negf_config), vp, C.POINTER(vp)]),
        "negf_destroy": (C.c_int, [vp]),
        "negf_set_potential": (C.c_int, [vp, vp]),
        "negf_charge": (C.c_int, [vp, vp]),
        "negf_transmission": (C.c_int, [vp, vp]),
        "negf_self_energy": (C.c_int, [vp, vp]),
        "negf_current": (C.c_int, [vp, vp, vp]),
        "negf_set_probe": (C.c_int, [vp, i32]),
        "negf_integrand_peak": (C.c_int, [vp, vp, vp, vp]),
        "negf_solve_host": (C.c_int, [vp, vp, vp, vp]),
        "negf_sync": (C.c_int, [vp]),
        "negf_kernel_stats": (C.c_int, [vp, C.POINTER(negf_kernel_stat), C.POINTER(i32), i32]),
        "negf_get_plan": (C.c_int, [vp, C.POINTER(negf_plan_info)]),
        "broyden_create": (C.c_int, [i64, i32, dbl, vp, C.POINTER(vp)]),
        "broyden_step": (C.c_int, [vp, vp, vp, C.POINTER(dbl)]),
        "broyden_reset": (C.c_int, [vp]),
        "broyden_destroy": (C.c_int, [vp]),
        "broyden_residual_noalloc": (C.c_int, [vp, vp, i64, vp, vp]),
        "negf_fp64_peak": (C.c_int, [C.POINTER(dbl), C.POINTER(dbl)]),
        "negf_last_error": (C.c_char_p, []),
        "negf_version": (C.c_char_p, []),
    }
    for name, (res, args) in sig.items():
        fn = getattr(lib, name)
        fn.restype = res
        fn.argtypes = args
    if path is None:
        _lib = lib
    return lib


def _check(st: int, where: str):
    if st != NEGF_OK:
        raise NegfError(st, where, load_library().negf_last_error().decode(errors="replace"))


def _c128(a) -> np.ndarray:
    return np.ascontiguousarray(np.asarray(a, dtype=np.complex128))


def _f64(a) -> np.ndarray:
    return np.ascontiguousarray(np.asarray(a, dtype=np.float64))


def _ptr(a: Optional[np.ndarray]):
    return None if a is None or a.size == 0 else a.ctypes.data_as(C.c_void_p)


def _dev_ptr(t, n_elems: int, what: str):
    """data_ptr() of a contiguous float64 CUDA tensor with at least n_elems elements."""
    import torch
    if not isinstance(t, torch.Tensor) or not t.is_cuda:
        raise TypeError(f"{what}: expected a CUDA torch.Tensor")
    if t.dtype != torch.float64 or not t.is_contiguous() or t.numel() < n_elems:
        raise ValueError(f"{what}: need a contiguous float64 tensor with >= {n_elems} elements")
    return C.c_void_p(t.data_ptr())


def _stream_ptr(stream) -> C.c_void_p:
    import torch
    s = stream if stream is not None else torch.cuda.current_stream()
    return C.c_void_p(s.cuda_stream)


class Negf:
    """negf_handle: ``negf_create`` .. ``negf_destroy`` (include/negf.h)."""

    def __init__(self, *, n_channels, n_rings, block, n_modes, lead_kind, coup_even, coup_odd,
                 mode_weight=None, z_eq=None, w_eq=None, z_neq=None, w_neq=None,
                 mu_s=0.0, mu_d=0.0, kT=0.0259, deg=2.0, sr_tol=1e-12, sr_maxit=200,
                 workspace_bytes=0, profile=False, pivot_theta=0.0, stream=None):
        self._lib = load_library()
        self._h = C.c_void_p(None)
        keep = []

        def arr(a, conv):
            if a is None:
                return None
            b = conv(a)
            keep.append(b)
            return b

        ce, co = arr(coup_even, _c128), arr(coup_odd, _c128)
        mw = arr(mode_weight, _f64)
        ze, we = arr(z_eq if z_eq is not None else [], _c128), arr(w_eq if w_eq is not None else [], _c128)
        zn, wn = arr(z_neq if z_neq is not None else [], _c128), arr(w_neq if w_neq is not None else [], _f64)
        if ze.shape != we.shape or zn.shape != wn.shape:
            raise ValueError("nodes and weights must have the same length")
        nexp = (n_modes if block == 1 else block * block)
        if ce.size != nexp or co.size != nexp:
            raise ValueError(f"coup_even/coup_odd need {nexp} entries")
        if block == 1 and (mw is None or mw.size != n_modes):
            raise ValueError("mode_weight needs n_modes entries")
        cfg = negf_config(
            n_channels=n_channels, n_rings=n_rings, block=block, n_modes=n_modes,
            lead_kind=lead_kind, sr_maxit=sr_maxit, sr_tol=sr_tol, mu_s=mu_s, mu_d=mu_d, kT=kT,
            deg=deg, coup_even=_ptr(ce), coup_odd=_ptr(co), mode_weight=_ptr(mw),
            n_eq=ze.size, z_eq=_ptr(ze), w_eq=_ptr(we), n_neq=zn.size, z_neq=_ptr(zn),
            w_neq=_ptr(wn), workspace_bytes=int(workspace_bytes), profile=int(bool(profile)),
            reserved=0, pivot_theta=float(pivot_theta))
        self.C, self.N, self.K_neq = int(n_channels), int(n_rings), int(zn.size)
        _check(self._lib.negf_create(C.byref(cfg), _stream_ptr(stream), C.byref(self._h)),
               "negf_create")

    @classmethod
    def from_workload(cls, wl, **kw):
        """Marshal a ``workloads.Workload`` into ``negf_config``."""
        return cls(n_channels=wl.C, n_rings=wl.N, block=wl.n, n_modes=wl.n_modes,
                   lead_kind=wl.lead_kind, coup_even=wl.coup_even, coup_odd=wl.coup_odd,
                   mode_weight=wl.mode_weight if wl.n == 1 else None,
                   z_eq=wl.z_eq, w_eq=wl.w_eq, z_neq=wl.z_neq, w_neq=wl.w_neq,
                   mu_s=wl.mu_s, mu_d=wl.mu_d, kT=wl.kT, deg=wl.deg, sr_tol=wl.sr_tol,
                   sr_maxit=wl.sr_maxit, **kw)

    # ---- the C-ABI calls, same names ----
    def negf_set_potential(self, phi_dev):
        _check(self._lib.negf_set_potential(self._h, _dev_ptr(phi_dev, self.C * self.N, "phi_dev")),
               "negf_set_potential")

    def negf_charge(self, n_dev):
        _check(self._lib.negf_charge(self._h, _dev_ptr(n_dev, self.C * self.N, "n_dev")),
               "negf_charge")

    def negf_transmission(self, T_dev):
        _check(self._lib.negf_transmission(self._h, _dev_ptr(T_dev, self.C * self.K_neq, "T_dev")),
               "negf_transmission")

    def negf_self_energy(self, sigma_dev):
        """sigma_dev: complex128 CUDA tensor [C][K_eq + K_neq][2][n*n]."""
        import torch
        if (not isinstance(sigma_dev, torch.Tensor) or not sigma_dev.is_cuda
                or sigma_dev.dtype != torch.complex128 or not sigma_dev.is_contiguous()):
            raise ValueError("sigma_dev: need a contiguous complex128 CUDA tensor")
        _check(self._lib.negf_self_energy(self._h, C.c_void_p(sigma_dev.data_ptr())), "negf_self_energy")

    def negf_current(self, current_dev=None, conductance_dev=None):
        a = _dev_ptr(current_dev, self.C, "current_dev") if current_dev is not None else None
        b = _dev_ptr(conductance_dev, self.C, "conductance_dev") if conductance_dev is not None else None
        _check(self._lib.negf_current(self._h, a, b), "negf_current")

    def negf_set_probe(self, ring: int):
        _check(self._lib.negf_set_probe(self._h, int(ring)), "negf_set_probe")

    def negf_integrand_peak(self, integrand_dev=None, k_peak_dev=None, E_peak_dev=None):
        """integrand_dev: float64 [C][K_neq]; k_peak_dev: int32 [C]; E_peak_dev: float64 [C] (CUDA tensors or None)."""
        import torch
        a = _dev_ptr(integrand_dev, self.C * self.K_neq, "integrand_dev") if integrand_dev is not None else None
        b = None
        if k_peak_dev is not None:
            if (not isinstance(k_peak_dev, torch.Tensor) or not k_peak_dev.is_cuda or k_peak_dev.dtype != torch.int32
                    or not k_peak_dev.is_contiguous() or k_peak_dev.numel() < self.C):
                raise ValueError("k_peak_dev: need a contiguous int32 CUDA tensor with >= C elements")
            b = C.c_void_p(k_peak_dev.data_ptr())
        c = _dev_ptr(E_peak_dev, self.C, "E_peak_dev") if E_peak_dev is not None else None
        _check(self._lib.negf_integrand_peak(self._h, a, b, c), "negf_integrand_peak")

    def negf_solve_host(self, phi_host: np.ndarray, n_host: np.ndarray, T_host: Optional[np.ndarray] = None):
        """HOST buffers in, HOST buffers out (numpy arrays or pinned torch CPU tensors)."""
        def hp(a, n, what):
            if a is None:
                return None
            if hasattr(a, "data_ptr"):            # torch CPU tensor (e.g. pinned)
                if a.is_cuda or a.numel() < n or not a.is_contiguous():
                    raise ValueError(f"{what}: need a contiguous CPU float64 buffer with >= {n} elements")
                return C.c_void_p(a.data_ptr())
            if a.dtype != np.float64 or not a.flags.c_contiguous or a.size < n:
                raise ValueError(f"{what}: need a C-contiguous float64 array with >= {n} elements")
            return a.ctypes.data_as(C.c_void_p)
        _check(self._lib.negf_solve_host(self._h, hp(phi_host, self.C * self.N, "phi_host"),
                                         hp(n_host, self.C * self.N, "n_host"),
                                         hp(T_host, self.C * self.K_neq, "T_host")),
               "negf_solve_host")

    def negf_sync(self):
        _check(self._lib.negf_sync(self._h), "negf_sync")

    def negf_kernel_stats(self, reset=False):
        cnt = C.c_int32(16)
        buf = (negf_kernel_stat * 16)()
        _check(self._lib.negf_kernel_stats(self._h, buf, C.byref(cnt), int(reset)), "negf_kernel_stats")
        return {buf[i].name.decode(): (int(buf[i].launches), float(buf[i].total_ms))
                for i in range(cnt.value)}

    def negf_get_plan(self):
        info = negf_plan_info()
        _check(self._lib.negf_get_plan(self._h, C.byref(info)), "negf_get_plan")
        return {k: getattr(info, k) for k, _ in negf_plan_info._fields_ if k != "reserved"}

    def negf_destroy(self):
        if getattr(self, "_h", None) is not None and self._h.value:
            self._lib.negf_destroy(self._h)
            self._h = C.c_void_p(None)

    close = negf_destroy

    def __del__(self):
        try:
            self.negf_destroy()
        except Exception:
            pass


class Broyden:
    """broyden_handle: ``broyden_create`` .. ``broyden_destroy`` (include/negf.h)."""

    def __init__(self, length: int, history: int = 8, zeta: float = 0.1, stream=None):
        self._lib = load_library()
        self._h = C.c_void_p(None)
        self.length = int(length)
        _check(self._lib.broyden_create(self.length, int(history), float(zeta), _stream_ptr(stream),
                                        C.byref(self._h)), "broyden_create")

    def broyden_step(self, x_in_dev, x_out_dev, want_eps: bool = True):
        eps = C.c_double(0.0)
        _check(self._lib.broyden_step(self._h, _dev_ptr(x_in_dev, self.length, "x_in_dev"),
                                      _dev_ptr(x_out_dev, self.length, "x_out_dev"),
                                      C.byref(eps) if want_eps else None), "broyden_step")
        return eps.value if want_eps else None

    def broyden_reset(self):
        _check(self._lib.broyden_reset(self._h), "broyden_reset")

    def broyden_destroy(self):
        if getattr(self, "_h", None) is not None and self._h.value:
            self._lib.broyden_destroy(self._h)
            self._h = C.c_void_p(None)

    close = broyden_destroy

    def __del__(self):
        try:
            self.broyden_destroy()
        except Exception:
            pass


NEGF_NOALLOC_MAX_LEN = 1 << 26      # include/negf.h


def broyden_residual_noalloc(x_in_dev, x_out_dev, eps_max_dev, length: Optional[int] = None, stream=None):
    """``broyden_residual_noalloc`` (include/negf.h): eps_max of Alg.3 steps 4-7 into the one-element
    device tensor ``eps_max_dev``; launches on ``stream``, allocates nothing, does not synchronise."""
    n = int(x_in_dev.numel() if length is None else length)
    need = n if 1 <= n <= NEGF_NOALLOC_MAX_LEN else 0       # out-of-range lengths are refused by the library
    _check(load_library().broyden_residual_noalloc(
        _dev_ptr(x_in_dev, need, "x_in_dev"), _dev_ptr(x_out_dev, need, "x_out_dev"), n,
        _dev_ptr(eps_max_dev, 1, "eps_max_dev"), _stream_ptr(stream)), "broyden_residual_noalloc")


def negf_fp64_peak():
    """(DFMA TFLOP/s, DMMA TFLOP/s) measured on the current device."""
    a, b = C.c_double(0.0), C.c_double(0.0)
    _check(load_library().negf_fp64_peak(C.byref(a), C.byref(b)), "negf_fp64_peak")
    return a.value, b.value


def negf_version() -> str:
    return load_library().negf_version().decode()
