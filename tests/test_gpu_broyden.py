"""GPU parity, Broyden's modified second method (Algorithm 3; step a6 of
SURVEY 8(a)) through the C-ABI against oracle/broyden.py: per step with identical state on both
sides, over a trajectory, at the config-5 vector length (256 000 entries), and inside the
self-consistent loop of a shrunk config 5 (20 iterations, history 8, mixing 0.1)."""
from dataclasses import replace

import numpy as np
import pytest

import workloads as wlmod
from oracle import broyden as obroyden
from oracle import negf_dense as od
from tests.parity import assert_parity, max_rel_err

pytestmark = pytest.mark.gpu


def _contractive_map(dim, seed):
    rng = np.random.default_rng(seed)
    A = rng.normal(size=(dim, dim)) / np.sqrt(dim)
    A *= 0.6 / np.linalg.norm(A, 2)
    b = rng.normal(size=dim)
    return lambda x: np.tanh(A @ x) + b


def test_first_step_is_linear_mixing_and_eps():
    import torch
    from paper_2407_14633_b200 import Broyden
    rng = np.random.default_rng(1)
    x0, y0 = rng.normal(size=777), rng.normal(size=777)
    g = Broyden(777, 8, 0.1)
    x = torch.tensor(x0, device="cuda")
    eps = g.broyden_step(x, torch.tensor(y0, device="cuda"))
    f = x0 - y0
    np.testing.assert_allclose(x.cpu().numpy(), x0 - 0.1 * f, rtol=0, atol=1e-15)   # Alg.3 step 18, s = 0
    assert abs(eps - np.max(np.abs(f) / np.abs(x0 + y0))) <= 1e-12 * eps           # steps 4-7
    g.broyden_destroy()


@pytest.mark.parametrize("dim,steps,history", [(12, 25, 8), (1, 10, 8), (1000, 14, 3), (33, 30, 1)])
def test_trajectory_matches_algorithm3(dim, steps, history):
    """Same map iterated on both sides; every iterate must agree (window eviction included:
    steps > history)."""
    import torch
    from paper_2407_14633_b200 import Broyden
    F = _contractive_map(dim, 5 + dim)
    ob = obroyden.Broyden(dim, history, 0.1)
    gb = Broyden(dim, history, 0.1)
    x_ref = np.zeros(dim)
    x = torch.zeros(dim, dtype=torch.float64, device="cuda")
    for it in range(steps):
        y_ref = F(x_ref)
        y_gpu = F(x.cpu().numpy())
        x_ref, eps_ref = ob.step(x_ref, y_ref)
        eps = gb.broyden_step(x, torch.tensor(y_gpu, device="cuda"))
        assert_parity(x.cpu().numpy(), x_ref, f"iterate {it}", rtol=1e-10)
        assert abs(eps - eps_ref) <= 1e-9 * eps_ref + 1e-14       # f is a difference of O(1) numbers
    gb.broyden_destroy()


def test_per_step_parity_with_identical_state_at_config5_length():
    """len = 64 * 4000: each step feeds both sides the SAME (x_in, x_out) pair (the oracle's), so
    differences cannot accumulate; 11 steps wrap the 8-pair window."""
    import torch
    from paper_2407_14633_b200 import Broyden
    n = 64 * 4000
    rng = np.random.default_rng(11)
    ob = obroyden.Broyden(n, 8, 0.1)
    gb = Broyden(n, 8, 0.1)
    x_ref = rng.normal(size=n)
    d = 0.3 + 0.5 * rng.uniform(size=n)
    b = rng.normal(size=n)
    for it in range(11):
        y = d * np.roll(x_ref, 1) * 0.5 + 0.2 * np.sin(x_ref) + b
        x = torch.tensor(x_ref, device="cuda")
        x_next, _ = ob.step(x_ref, y)
        gb.broyden_step(x, torch.tensor(y, device="cuda"), want_eps=False)
        assert_parity(x.cpu().numpy(), x_next, f"step {it}", rtol=1e-10)
        x_ref = x_next
    gb.broyden_destroy()


def test_non_finite_residual_gives_non_finite_eps_max():
    """A NaN (or infinite) entry of F(x) -- e.g. a singular pivot upstream -- must not be reported
    as convergence: eps_max comes back non-finite (the oracle's np.max returns NaN; the device
    returns +infinity, fmax would have dropped the NaN).  PAPER.md:216 loops on eps_max >= 1e-5."""
    import torch
    from paper_2407_14633_b200 import Broyden
    rng = np.random.default_rng(3)
    for bad, pos in ((np.nan, 4321), (np.inf, 0), (-np.inf, 99999)):
        x0, y0 = rng.normal(size=100000), rng.normal(size=100000)
        y0[pos] = bad
        gb = Broyden(100000, 8, 0.1)
        eps = gb.broyden_step(torch.tensor(x0, device="cuda"), torch.tensor(y0, device="cuda"))
        _, eps_ref = obroyden.Broyden(100000, 8, 0.1).step(x0, y0)
        assert not np.isfinite(eps) and not np.isfinite(eps_ref)
        gb.broyden_destroy()


@pytest.mark.parametrize("history,steps", [(3, 9), (1, 5), (8, 14)])
def test_device_window_keeps_the_secant_equation(history, steps):
    """R17 on the device alone: x_{m+2} - x_{m+1} + G_{m+1} f_{m+1} = 0 defines G_{m+1} on f_{m+1}
    only, so the secant equation is checked through linearity: for the affine map F(x) = A x + b
    (f is affine, df = (I - A) dx) a method that satisfies G_{m+1} df_m = dx_m for the newest pair
    with history >= 1 reproduces the oracle trajectory, and the oracle is pinned on the secant
    equation (tests/test_oracle_broyden.py::test_r17_*).  Here: trajectory parity past eviction
    with history 1, 3, 8 on an affine map (no tanh saturation hiding a wrong term)."""
    import torch
    from paper_2407_14633_b200 import Broyden
    dim = 40
    rng = np.random.default_rng(100 + history)
    A = rng.normal(size=(dim, dim))
    A *= 0.7 / np.linalg.norm(A, 2)
    b = rng.normal(size=dim)
    ob = obroyden.Broyden(dim, history, 0.1)
    gb = Broyden(dim, history, 0.1)
    x_ref = np.zeros(dim)
    x = torch.zeros(dim, dtype=torch.float64, device="cuda")
    for it in range(steps):
        x_ref, _ = ob.step(x_ref, A @ x_ref + b)
        xg = x.cpu().numpy()
        gb.broyden_step(x, torch.tensor(A @ xg + b, device="cuda"), want_eps=False)
        assert_parity(x.cpu().numpy(), x_ref, f"iterate {it}", rtol=1e-9)
    gb.broyden_destroy()


def test_repeated_pair_adds_no_history_and_reset():
    """R18: d = ||df||^2 = 0 skips steps 9-13; broyden_reset restarts at plain mixing."""
    import torch
    from paper_2407_14633_b200 import Broyden
    rng = np.random.default_rng(2)
    x0, y0 = rng.normal(size=50), rng.normal(size=50)
    ob = obroyden.Broyden(50, 8, 0.1)
    gb = Broyden(50, 8, 0.1)
    x_ref = x0.copy()
    x = torch.tensor(x0, device="cuda")
    for y in (y0, y0 + 0.1, None, y0 * 0.5):
        if y is None:                                  # feed the same (x, F(x)) pair again, bit for bit
            x_ref = prev_x.copy()
            x = prev_x_gpu.clone()
            y = prev_y
        prev_x, prev_x_gpu, prev_y = x_ref.copy(), x.clone(), y
        x_ref, _ = ob.step(x_ref, y)
        gb.broyden_step(x, torch.tensor(y, device="cuda"))
        assert_parity(x.cpu().numpy(), x_ref, "repeated pair", rtol=1e-10)
    gb.broyden_reset()
    x = torch.tensor(x0, device="cuda")
    gb.broyden_step(x, torch.tensor(y0, device="cuda"))
    np.testing.assert_allclose(x.cpu().numpy(), x0 - 0.1 * (x0 - y0), rtol=0, atol=1e-15)
    gb.broyden_destroy()


def test_config5_shrunk_self_consistent_loop():
    """BASELINE.json configs[4] on a shrunk array (3 channels x 12 rings): 20 Broyden iterations on
    the per-ring potential with the Poisson stand-in; GPU (negf_charge + broyden_step) against the
    oracle (dense definition + Algorithm 3), per iteration, and the residual must fall."""
    import torch
    from paper_2407_14633_b200 import Broyden, Negf
    wl = wlmod.make_config(5, C=3, N=12, K_neq=24, K_eq=8)
    poisson = wl.extra["poisson"]
    iters = wl.extra["broyden_iters"]
    # oracle trajectory
    ob = obroyden.Broyden(wl.C * wl.N, wl.extra["broyden_history"], wl.extra["broyden_zeta"])
    phi_ref = wl.phi.copy()
    traj, resid = [], []
    for it in range(iters):
        w = replace(wl, phi=phi_ref)
        n_ref, _ = od.charge_and_transmission(w)
        phi_out = poisson.phi_out(wl.phi, n_ref)
        resid.append(np.max(np.abs(phi_ref - phi_out)))
        x, _ = ob.step(phi_ref.reshape(-1), phi_out.reshape(-1))
        phi_ref = x.reshape(wl.C, wl.N)
        traj.append(phi_ref.copy())
    assert resid[-1] < 1e-2 * resid[0]
    # GPU trajectory
    h = Negf.from_workload(wl)
    gb = Broyden(wl.C * wl.N, wl.extra["broyden_history"], wl.extra["broyden_zeta"])
    phi_ext = torch.tensor(wl.phi, dtype=torch.float64, device="cuda")
    r_dev = torch.tensor(poisson.r, dtype=torch.float64, device="cuda")
    phi = phi_ext.clone()
    n = torch.empty((wl.C, wl.N), dtype=torch.float64, device="cuda")
    worst = 0.0
    for it in range(iters):
        h.negf_set_potential(phi)
        h.negf_charge(n)
        phi_out = poisson.phi_out(phi_ext, n, r_dev)
        gb.broyden_step(phi.view(-1), phi_out.view(-1), want_eps=False)
        err = max_rel_err(phi.cpu().numpy(), traj[it])
        worst = max(worst, err)
        # 20 iterations of a secant method amplify last-bit differences of the charge: the
        # trajectory tolerance is looser than the per-step one
        assert err < 1e-8, (it, err)
    h.negf_destroy()
    gb.broyden_destroy()
    print("config5-shrunk trajectory: worst relative error", worst)
