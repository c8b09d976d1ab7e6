"""CPU oracle for the NEGF charge / transmission / Broyden hot path.

TEST INFRASTRUCTURE ONLY.  This package is the slow, plain, obviously-correct
statement of what the CUDA path must compute, written from the paper
(/root/reference/PAPER.md, arXiv 2407.14633) and from the readings listed in
DESIGN.md.  Only ``tests/``, ``__graft_entry__.smoke()`` and the
``cpu_baseline`` / ``--impl reference`` legs of ``bench.py`` may import it.  It
shares no code with ``paper_2407_14633_b200/`` and never imports it; both sides
receive their inputs as plain arrays from ``workloads/``.

Modules
  selfenergy  closed-form surface Green's function of the alternating chain and
              Sancho-Rubio decimation
  negf_dense  tier O1: the definition -- dense inversion of
              (E+i eta)I - H - Sigma_L - Sigma_R        (eq.(2),(4),(5))
  negf_rgf    tier O3: the paper's Algorithm 2 + Algorithm 1 (block-tridiagonal
              recursion), step by step
  negf_rgf_omp(.cpp/.py)  tier O3 again in plain C++17 + OpenMP (one energy point per
              thread, own Sancho-Rubio): full-size block devices in minutes; the timed
              CPU baseline of bench.py.  Pinned to negf_dense and to banded LU.
  broyden     Algorithm 3 (modified second Broyden) and the dense-matrix
              "bad Broyden" it must equal

Parity pins (tests/, -m "not gpu"): see DESIGN.md "Pins".  Every function here
is pinned by at least one closed form / invariant / brute-force case; none is
"parity unpinned".
"""
