"""Seeded synthetic inputs for the five BASELINE.json configs.

This module is the only code shared by the CPU oracle (``oracle/``) and the CUDA
path (``paper_2407_14633_b200/``).  It holds none of the method's arithmetic
(no Green's functions, no self-energies, no recursions, no Broyden): it only
produces the *inputs* of the C-ABI of ``include/negf.h`` -- potentials,
coupling blocks, quadrature nodes/weights, the Poisson stand-in map -- as plain
numpy arrays.  See DESIGN.md "Input recipe".
"""
from .configs import (  # noqa: F401
    Workload,
    PoissonStandIn,
    config1,
    config2,
    config3,
    config4,
    config5,
    table2,
    make_config,
    scalar_twin,
    cnt_mode_couplings,
    cnt_realspace_couplings,
    barrier_profile,
    contour_semicircle,
    contour_equilibrium,
    contour_neutral,
    real_axis_three_segment,
    refine_segment_limits,
    equilibrium_variant,
    two_part_equilibrium_variant,
    neutral_variant,
    real_axis_gauss_legendre,
    real_axis_uniform,
    fermi,
    CNT_N,
    T_HOP,
    ETA,
    KT,
    MU_S,
    MU_D,
    DEG,
    E_B,
    F_TAIL,
)
