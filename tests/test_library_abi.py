"""The C-ABI shared library builds, loads and exports every symbol include/negf.h
declares; argument validation works without a GPU (no compute calls here)."""
import ctypes as C
import os
import re
import shutil

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

pytestmark = pytest.mark.skipif(
    shutil.which("nvcc") is None and not os.path.exists("/usr/local/cuda/bin/nvcc")
    and not os.path.exists(os.path.join(ROOT, "paper_2407_14633_b200", "libnegf_b200.so")),
    reason="neither nvcc nor a prebuilt libnegf_b200.so")


@pytest.fixture(scope="module")
def lib():
    from paper_2407_14633_b200 import build, binding
    if shutil.which("nvcc") or os.path.exists("/usr/local/cuda/bin/nvcc"):
        build.build()
    return binding.load_library()


def _declared_functions():
    text = open(os.path.join(ROOT, "include", "negf.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    names = re.findall(r"NEGF_API\s+(?:negf_status|const char\*)\s+((?:negf|broyden)_\w+)\s*\(", text)
    return sorted(set(names))


def test_exports_every_declared_symbol(lib):
    from paper_2407_14633_b200 import binding
    declared = _declared_functions()
    assert len(declared) >= 14
    assert sorted(binding.EXPORTED_SYMBOLS) == declared
    for name in declared:
        assert hasattr(lib, name), name


def test_version_and_error_string(lib):
    assert b"sm_100a" in lib.negf_version()
    assert isinstance(lib.negf_last_error(), bytes)


def test_argument_validation_without_gpu(lib):
    from paper_2407_14633_b200 import binding as b
    h = C.c_void_p(None)
    assert lib.negf_create(None, None, C.byref(h)) == b.NEGF_EINVAL
    cfg = b.negf_config()
    cfg.n_channels, cfg.n_rings, cfg.block = 1, 1, 1        # N < 2
    assert lib.negf_create(C.byref(cfg), None, C.byref(h)) == b.NEGF_EINVAL
    assert b"n_rings" in lib.negf_last_error()
    cfg.n_rings, cfg.kT, cfg.deg = 10, -1.0, 2.0             # kT <= 0
    assert lib.negf_create(C.byref(cfg), None, C.byref(h)) == b.NEGF_EINVAL
    cfg.kT = 0.0259
    cfg.reserved = 1                                         # reserved fields must be 0
    assert lib.negf_create(C.byref(cfg), None, C.byref(h)) == b.NEGF_EINVAL
    assert b"reserved" in lib.negf_last_error()
    cfg.reserved, cfg.pivot_theta = 0, -1.0
    assert lib.negf_create(C.byref(cfg), None, C.byref(h)) == b.NEGF_EINVAL
    assert lib.negf_set_probe(None, 0) == b.NEGF_EINVAL
    assert lib.negf_integrand_peak(None, None, None, None) == b.NEGF_EINVAL
    assert lib.negf_set_potential(None, None) == b.NEGF_EINVAL
    assert lib.negf_charge(None, None) == b.NEGF_EINVAL
    assert lib.negf_transmission(None, None) == b.NEGF_EINVAL
    bh = C.c_void_p(None)
    assert lib.broyden_create(0, 8, 0.1, None, C.byref(bh)) == b.NEGF_EINVAL
    assert lib.broyden_step(None, None, None, None) == b.NEGF_EINVAL
    assert lib.negf_destroy(None) == b.NEGF_OK and lib.broyden_destroy(None) == b.NEGF_OK


def test_no_cpu_fallback_without_device(lib):
    """Without a CUDA device a well-formed negf_create must fail with NEGF_ECUDA."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    from paper_2407_14633_b200 import binding as b
    import workloads
    w = workloads.config1(N=10, K_neq=4)
    ce = np.ascontiguousarray(w.coup_even)
    co = np.ascontiguousarray(w.coup_odd)
    mw = np.ascontiguousarray(w.mode_weight)
    zn = np.ascontiguousarray(w.z_neq)
    wn = np.ascontiguousarray(w.w_neq)
    cfg = b.negf_config(n_channels=1, n_rings=10, block=1, n_modes=1, lead_kind=0, sr_maxit=200,
                        sr_tol=1e-12, mu_s=0.0, mu_d=-0.1, kT=0.0259, deg=2.0,
                        coup_even=ce.ctypes.data, coup_odd=co.ctypes.data, mode_weight=mw.ctypes.data,
                        n_eq=0, z_eq=None, w_eq=None, n_neq=4, z_neq=zn.ctypes.data,
                        w_neq=wn.ctypes.data, workspace_bytes=0, profile=0, reserved=0)
    h = C.c_void_p(None)
    assert lib.negf_create(C.byref(cfg), None, C.byref(h)) == b.NEGF_ECUDA
    assert not h.value
