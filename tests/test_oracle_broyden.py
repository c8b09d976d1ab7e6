"""Pins of the Broyden oracle (Algorithm 3): textbook special
cases and the dense-matrix method it must equal (DESIGN.md pins P11, P12)."""
import numpy as np

from oracle.broyden import Broyden, DenseBadBroyden


def _contractive_map(dim, seed):
    rng = np.random.default_rng(seed)
    A = rng.normal(size=(dim, dim))
    A = 0.9 * A / np.linalg.norm(A, 2)
    b = rng.normal(size=dim)

    def F(x):
        return A @ np.tanh(x) + b
    return F


def test_p11_first_step_is_linear_mixing():
    """m = 0: x_1 = x_0 - zeta f (Alg.3 step 18 with s = 0)."""
    rng = np.random.default_rng(0)
    x, y = rng.normal(size=9), rng.normal(size=9)
    b = Broyden(9, history=8, zeta=0.1)
    x1, eps = b.step(x, y)
    assert np.array_equal(x1, x - 0.1 * (x - y))
    assert eps == np.max(np.abs(x - y) / np.abs(x + y))


def test_p11_length_one_is_secant_method():
    """For a scalar unknown, steps m >= 1 are the secant method on f(x) = x - F(x)."""
    F = lambda x: np.cos(x)
    b = Broyden(1, history=50, zeta=0.3)
    xs = [np.array([0.2])]
    for _ in range(6):
        xn, _ = b.step(xs[-1], F(xs[-1]))
        xs.append(xn)
    f = lambda x: x - F(x)
    for m in range(1, 6):
        x0, x1 = xs[m - 1][0], xs[m][0]
        secant = x1 - f(x1) * (x1 - x0) / (f(x1) - f(x0))
        assert abs(xs[m + 1][0] - secant) < 1e-13
    assert abs(f(xs[-1][0])) < 1e-6


def test_p11_equals_dense_bad_broyden_full_history():
    dim = 12
    F = _contractive_map(dim, 3)
    a, d = Broyden(dim, history=100, zeta=0.1), DenseBadBroyden(dim, zeta=0.1)
    xa = xd = np.zeros(dim)
    for _ in range(15):
        xa, _ = a.step(xa, F(xa))
        xd = d.step(xd, F(xd))
        assert np.max(np.abs(xa - xd)) < 1e-11 * max(1.0, np.max(np.abs(xd)))


def test_p11_secant_condition_on_stored_pairs():
    """G_m df_j = dx_j for the newest stored pair: with G = zeta I + sum w_j v_j^T."""
    dim = 10
    F = _contractive_map(dim, 4)
    b = Broyden(dim, history=100, zeta=0.1)
    x = np.zeros(dim)
    xs, fs = [], []
    for _ in range(8):
        xs.append(x.copy())
        fs.append(x - F(x))
        x, _ = b.step(x, F(x))
    G = 0.1 * np.eye(dim) + sum(np.outer(w, v) for v, w in zip(b.V, b.W))
    dx, df = xs[-1] - xs[-2], fs[-1] - fs[-2]
    assert np.max(np.abs(G @ df - dx)) < 1e-12


def test_p12_window_converges_and_beats_plain_mixing():
    dim = 12
    F = _contractive_map(dim, 7)
    x = np.zeros(dim)
    for _ in range(25):
        x = x - 0.1 * (x - F(x))
    plain = np.max(np.abs(x - F(x)))
    b = Broyden(dim, history=8, zeta=0.1)
    x = np.zeros(dim)
    for _ in range(25):
        x, _ = b.step(x, F(x))
    assert np.max(np.abs(x - F(x))) < 1e-3 * plain


def test_window_eviction_and_zero_df():
    """History never exceeds h; a repeated (x, F) pair (d = 0) adds no pair (R18)."""
    dim = 6
    F = _contractive_map(dim, 9)
    b = Broyden(dim, history=3, zeta=0.1)
    x = np.zeros(dim)
    for _ in range(7):
        x, _ = b.step(x, F(x))
    assert len(b.V) == 3 and len(b.W) == 3
    b2 = Broyden(dim, history=3, zeta=0.1)
    x0 = np.ones(dim)
    b2.step(x0, F(x0))
    nV = len(b2.V)
    x1, _ = b2.step(x0, F(x0))            # same input again: df = 0
    assert len(b2.V) == nV and np.all(np.isfinite(x1))
