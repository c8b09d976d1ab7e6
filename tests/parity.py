"""Tolerance rule shared by the GPU parity tests.

north_star: relative 1e-10 in FP64.  Per output array y: pass iff for every element
|y_gpu - y_ref| <= rtol * max(|y_ref|, floor * max|y_ref|).  The floor (1e-6) only
matters for T(E), which spans ~1e-130..15 inside one sweep; charge per ring is O(1-10).
"""
import numpy as np

RTOL = 1e-10
FLOOR = 1e-6


def max_rel_err(got, ref, floor=FLOOR):
    got = np.asarray(got, dtype=np.float64)
    ref = np.asarray(ref, dtype=np.float64)
    scale = np.maximum(np.abs(ref), floor * np.max(np.abs(ref)))
    scale = np.maximum(scale, 1e-300)
    return float(np.max(np.abs(got - ref) / scale))


def assert_parity(got, ref, what, rtol=RTOL, floor=FLOOR):
    assert np.all(np.isfinite(np.asarray(got))), f"{what}: non-finite GPU values"
    err = max_rel_err(got, ref, floor)
    assert err <= rtol, f"{what}: max relative error {err:.3e} > {rtol:.1e}"
    return err
