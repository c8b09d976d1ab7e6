"""Broyden's modified second method, CPU oracle (test infrastructure only).

Algorithm 3 of the paper, single rank (the MPI_Allreduce
steps 7, 8, 10, 15 are identities on one rank), written step by step with the
paper's step numbers.  Readings (R15-R19):
  R15  step 13 prints "-eta Delta f"; the mixing fraction is zeta.
  R16  the library performs ONE iteration per call and returns eps_max.
  R17  history window h: only the most recent h (v, w) pairs are kept; sums run
       over stored pairs oldest first.  The paper keeps all M pairs;
       the window is BASELINE.json's ("history 8").  When the window is full, the
       oldest pair leaves *before* steps 9-11, so that w_m = dx - G df is formed
       with the same G = zeta I + sum_kept w v^T that the new pair is then added
       to: only this order keeps the secant equation G_{m+1} df_m = dx_m that
       defines the method (pinned by tests/test_oracle_broyden.py::test_r17_*).
  R18  d = ||Delta f||^2 = 0: steps 9-13 are skipped (no new pair).
  R19  eps_t = |f_t| / max(|x_in,t + x_out,t|, 1e-300).

``DenseBadBroyden`` is the textbook method with an explicit inverse-Jacobian
matrix G (len x len):  G <- G + (dx - G df) df^T / (df^T df),  x <- x - G f,
G_0 = zeta I, which Algorithm 3 with unlimited history must reproduce.
"""
from __future__ import annotations

import numpy as np


class Broyden:
    """State of Algorithm 3 for a vector of length ``length``."""

    def __init__(self, length: int, history: int = 8, zeta: float = 0.1):
        self.length = int(length)
        self.history = int(history)
        self.zeta = float(zeta)
        self.reset()

    def reset(self):
        self.m = 0
        self.f_old = np.zeros(self.length)
        self.x_old = np.zeros(self.length)
        self.V = []          # rows of V^T  (v_j), oldest first
        self.W = []          # columns of W (w_j), oldest first

    def step(self, x_in: np.ndarray, x_out: np.ndarray):
        """One pass of the loop body; returns (x_next, eps_max)."""
        x_in = np.asarray(x_in, dtype=np.float64)
        x_out = np.asarray(x_out, dtype=np.float64)
        f = x_in - x_out                                             # step 2
        df = f - self.f_old                                          # step 3
        eps = np.abs(f) / np.maximum(np.abs(x_in + x_out), 1e-300)   # step 4
        eps_max = float(eps.max()) if eps.size else 0.0              # steps 5, 7
        d = float(np.dot(df, df))                                    # steps 6, 8
        if self.m > 0 and d != 0.0:
            if len(self.V) == self.history:                          # R17: full window ->
                self.V.pop(0)                                        # the oldest pair leaves
                self.W.pop(0)                                        # before steps 9-11
            s = np.zeros(self.length)
            for v, w in zip(self.V, self.W):                         # steps 9-11 (m > 1)
                s += w * float(np.dot(v, df))
            v_new = df / d                                           # step 12
            w_new = -self.zeta * df + (x_in - self.x_old) - s        # step 13
            self.V.append(v_new)
            self.W.append(w_new)
        s = np.zeros(self.length)
        for v, w in zip(self.V, self.W):                             # steps 14-16
            s += w * float(np.dot(v, f))
        self.x_old = x_in.copy()                                     # step 17
        x_next = self.x_old - self.zeta * f - s                      # step 18
        self.f_old = f
        self.m += 1                                                  # step 19
        return x_next, eps_max


class DenseBadBroyden:
    """Broyden's second ("bad") method with the inverse Jacobian as a dense matrix."""

    def __init__(self, length: int, zeta: float = 0.1):
        self.G = zeta * np.eye(length)
        self.have_old = False
        self.x_old = None
        self.f_old = None

    def step(self, x_in, x_out):
        x_in = np.asarray(x_in, dtype=np.float64)
        f = x_in - np.asarray(x_out, dtype=np.float64)
        if self.have_old:
            dx = x_in - self.x_old
            df = f - self.f_old
            d = float(df @ df)
            if d != 0.0:
                self.G = self.G + np.outer(dx - self.G @ df, df) / d
        self.x_old = x_in.copy()
        self.f_old = f.copy()
        self.have_old = True
        return x_in - self.G @ f
