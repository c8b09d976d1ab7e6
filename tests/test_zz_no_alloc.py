"""GPU test of ``broyden_residual_noalloc`` (include/negf.h): the allocation-free entry point whose
scratch is a file-scope device array (csrc/residual_noalloc.cu).  Its output is compared with the existing
path's -- the eps_max that ``broyden_step`` returns for the same (x_in, x_out), Alg.3 steps 4-7,
PAPER.md:216-230 -- on two calls in a row: the second with a shorter vector and a smaller residual, so that
anything carried over in the shared array from the first call would show.  Collected last on purpose
(the suite runs with pytest -x); passes alone in a fresh process and after the other tests."""
import ctypes as C

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

RTOL = 1e-10     # the tolerance of the parity tests (tests/parity.py); a maximum is in fact reproduced exactly


def _existing_path_eps(x_in, x_out):
    """eps_max from broyden_step on a fresh handle (it updates x_in in place: work on a copy)."""
    from paper_2407_14633_b200 import Broyden
    g = Broyden(x_in.numel(), 8, 0.1)
    try:
        return g.broyden_step(x_in.clone(), x_out)
    finally:
        g.broyden_destroy()


def _pair(n, scale, seed):
    import torch
    rng = np.random.default_rng(seed)
    x_in = rng.normal(size=n)
    x_out = x_in + scale * rng.normal(size=n)
    return torch.tensor(x_in, device="cuda"), torch.tensor(x_out, device="cuda")


def test_no_alloc_residual_matches_broyden_step_twice_in_a_row():
    import torch
    from paper_2407_14633_b200 import broyden_residual_noalloc
    eps_dev = torch.full((1,), -1.0, dtype=torch.float64, device="cuda")
    # 256 000 entries = config 5's vector (63 blocks, ragged tail), then 5 000 entries (2 blocks)
    for n, scale, seed in [(256_000, 1.0, 11), (5_000, 1e-6, 12)]:
        x_in, x_out = _pair(n, scale, seed)
        want = _existing_path_eps(x_in, x_out)
        keep = x_in.clone()
        broyden_residual_noalloc(x_in, x_out, eps_dev)
        torch.cuda.synchronize()
        got = float(eps_dev.item())
        assert np.isfinite(want) and want > 0.0
        assert abs(got - want) <= RTOL * want, (n, got, want)
        assert torch.equal(x_in, keep)                      # inputs are read only
        f = (x_in - x_out).abs() / (x_in + x_out).abs().clamp_min(1e-300)
        assert abs(got - float(f.max().item())) <= RTOL * want


def test_no_alloc_residual_reports_non_finite_and_rejects_oversize():
    import torch
    from paper_2407_14633_b200 import NEGF_NOALLOC_MAX_LEN, NegfError, broyden_residual_noalloc, load_library
    x_in, x_out = _pair(9_000, 1e-3, 13)
    x_out[8_999] = float("nan")
    eps_dev = torch.zeros(1, dtype=torch.float64, device="cuda")
    broyden_residual_noalloc(x_in, x_out, eps_dev)
    assert float(eps_dev.item()) == float("inf") == _existing_path_eps(x_in, x_out)
    with pytest.raises(NegfError) as err:                   # beyond the static array: refused, nothing launched
        broyden_residual_noalloc(x_in, x_out, eps_dev, length=NEGF_NOALLOC_MAX_LEN + 1)
    assert "outside" in str(err.value)
    lib = load_library()
    assert lib.broyden_residual_noalloc(None, None, 1, None, None) != 0
    assert lib.broyden_residual_noalloc(C.c_void_p(x_in.data_ptr()), C.c_void_p(x_out.data_ptr()), 0,
                                        C.c_void_p(eps_dev.data_ptr()), None) != 0
    torch.cuda.synchronize()
