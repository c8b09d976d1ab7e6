"""GPU parity, scalar (mode-space) path: configs[0] and configs[1] of BASELINE.json through the
C-ABI against the CPU oracle, element by element (north_star: 1e-10 relative)."""
import numpy as np
import pytest

import workloads as wlmod
from oracle import negf_dense as od
from oracle import negf_rgf as orgf
from tests.parity import assert_parity

pytestmark = pytest.mark.gpu


def _gpu_run(wl, **kw):
    import torch
    from paper_2407_14633_b200 import Negf
    h = Negf.from_workload(wl, **kw)
    phi = torch.tensor(wl.phi, dtype=torch.float64, device="cuda")
    n = torch.empty((wl.C, wl.N), dtype=torch.float64, device="cuda")
    T = torch.empty((wl.C, max(wl.K_neq, 1)), dtype=torch.float64, device="cuda")
    h.negf_set_potential(phi)
    h.negf_charge(n)
    h.negf_transmission(T)
    h.negf_sync()
    out = n.cpu().numpy(), T.cpu().numpy()[:, :wl.K_neq]
    h.negf_destroy()
    return out


def test_config1_full_vs_dense_definition():
    wl = wlmod.config1()
    n_ref, T_ref = od.charge_and_transmission(wl)
    n, T = _gpu_run(wl)
    assert_parity(n, n_ref, "config1 charge")
    assert_parity(T, T_ref, "config1 T(E)")


@pytest.mark.parametrize("N,K_neq,K_eq", [(40, 37, 9), (33, 64, 16), (2, 5, 3), (17, 1, 0), (50, 0, 7)])
def test_config2_shrunk_vs_dense_definition(N, K_neq, K_eq):
    """Several tiles (N > 16) and ragged tails (N % 16 != 0, K % 32 != 0), both lead parities,
    the degenerate N = 2, contour-only and real-axis-only handles."""
    wl = wlmod.make_config(2, N=N, K_neq=max(K_neq, 1), K_eq=K_eq)
    if K_neq == 0:
        wl = wl.subset(neq_idx=[])
    n_ref, T_ref = od.charge_and_transmission(wl)
    n, T = _gpu_run(wl)
    assert_parity(n, n_ref, "config2-shrunk charge")
    if K_neq:
        assert_parity(T, T_ref, "config2-shrunk T(E)")


def test_config2_full_vs_paper_recursion():
    """Full configs[1] (the bench workload, same launch configuration) against tier O3."""
    wl = wlmod.config2()
    n_ref, T_ref = orgf.charge_and_transmission(wl)
    n, T = _gpu_run(wl)
    assert_parity(n, n_ref, "config2 charge")
    assert_parity(T, T_ref, "config2 T(E)")


def test_config2_full_sampled_vs_dense_definition():
    """Sampled energies of the full-size device against the dense definition (tier O1)."""
    wl = wlmod.config2()
    rng = np.random.default_rng(7)
    sub = wl.subset(neq_idx=np.sort(rng.choice(wl.K_neq, 3, replace=False)),
                    eq_idx=np.sort(rng.choice(wl.K_eq, 2, replace=False)))
    n_ref, T_ref = od.charge_and_transmission(sub)
    n, T = _gpu_run(sub)
    assert_parity(n, n_ref, "config2 sampled charge")
    assert_parity(T, T_ref, "config2 sampled T(E)")


def test_workspace_tiling_gives_identical_results():
    """A small workspace cap forces several sweep launches; results must not change."""
    wl = wlmod.make_config(2, N=64, K_neq=96, K_eq=16)
    n1, T1 = _gpu_run(wl)
    n2, T2 = _gpu_run(wl, workspace_bytes=64 * 32 * 16 * 5)
    assert np.array_equal(n1, n2) and np.array_equal(T1, T2)


def test_multi_channel_scalar_and_host_path():
    import torch
    from paper_2407_14633_b200 import Negf
    wl = wlmod.make_config(2, N=48, K_neq=40, K_eq=8)
    rng = np.random.default_rng(3)
    wl.C = 3
    wl.phi = np.stack([wl.phi[0], wl.phi[0] + 0.05 * rng.normal(size=wl.N), -wl.phi[0]])
    n_ref, T_ref = od.charge_and_transmission(wl)
    n, T = _gpu_run(wl)
    assert_parity(n, n_ref, "3-channel charge")
    assert_parity(T, T_ref, "3-channel T(E)")
    h = Negf.from_workload(wl)
    n_host = np.empty((wl.C, wl.N))
    T_host = np.empty((wl.C, wl.K_neq))
    h.negf_solve_host(np.ascontiguousarray(wl.phi), n_host, T_host)
    assert np.array_equal(n_host, n) and np.array_equal(T_host, T)
    h.negf_destroy()


def test_state_errors_and_rerun():
    import torch
    from paper_2407_14633_b200 import Negf, NegfError
    wl = wlmod.make_config(2, N=20, K_neq=8, K_eq=4)
    h = Negf.from_workload(wl)
    n = torch.empty((1, wl.N), dtype=torch.float64, device="cuda")
    with pytest.raises(NegfError) as ei:
        h.negf_charge(n)
    assert ei.value.status == 5                      # NEGF_ESTATE
    phi = torch.tensor(wl.phi, dtype=torch.float64, device="cuda")
    h.negf_set_potential(phi)
    h.negf_charge(n)
    a = n.cpu().numpy().copy()
    h.negf_set_potential(phi * 0.5)
    h.negf_charge(n)
    b = n.cpu().numpy().copy()
    h.negf_set_potential(phi)
    h.negf_charge(n)
    assert np.array_equal(a, n.cpu().numpy()) and not np.array_equal(a, b)   # deterministic
    h.negf_destroy()


def test_landauer_reductions():
    """eq.(5)-(6): current and zero-bias conductance from T(E); ideal tube at low kT gives
    G = G_0 * (number of open modes)."""
    import torch
    from paper_2407_14633_b200 import Negf
    wl = wlmod.make_config(2, N=24, K_neq=64, K_eq=0)
    wl.phi[:] = 0.0
    wl.mu_s = wl.mu_d = 0.6
    wl.kT = 0.002
    wl.z_neq, wl.w_neq = wlmod.real_axis_gauss_legendre(0.6 - 0.05, 0.6 + 0.05, 64, eta=1e-9)
    h = Negf.from_workload(wl)
    h.negf_set_potential(torch.tensor(wl.phi, dtype=torch.float64, device="cuda"))
    cur = torch.empty(1, dtype=torch.float64, device="cuda")
    cond = torch.empty(1, dtype=torch.float64, device="cuda")
    h.negf_current(cur, cond)
    h.negf_sync()
    assert abs(cond.item() - 4.0) < 1e-4             # 4 open subbands at E = 0.6 eV
    assert abs(cur.item()) < 1e-12                   # mu_s == mu_d
    h.negf_destroy()


@pytest.mark.parametrize("cfg,kw", [(2, dict(N=18, K_neq=21, K_eq=0)), (1, dict(N=30, K_neq=40)),
                                    (3, dict(N=9, K_neq=10, K_eq=0)), (4, dict(C=3, N=8, K_neq=9, K_eq=0))])
def test_current_and_conductance_vs_definition(cfg, kw):
    """negf_current against the oracle's currents by the definition of eq.(5)
    (Tr[F_l Gamma_l A + i Gamma_l G^<] from the dense Green's function) and the
    conductance of eq.(6), at mu_S != mu_D, scalar and block handles, several channels."""
    import torch
    from paper_2407_14633_b200 import Negf
    wl = wlmod.make_config(cfg, **kw)
    assert wl.mu_s != wl.mu_d
    I_ref, I_D, G_ref = od.landauer_dense(wl)
    assert np.all(np.abs(I_ref + I_D) < 1e-9 * np.abs(I_ref))          # conservation (P6) in the oracle
    h = Negf.from_workload(wl)
    h.negf_set_potential(torch.tensor(wl.phi, dtype=torch.float64, device="cuda"))
    cur = torch.empty(wl.C, dtype=torch.float64, device="cuda")
    cond = torch.empty(wl.C, dtype=torch.float64, device="cuda")
    h.negf_current(cur, cond)
    h.negf_sync()
    assert_parity(cur.cpu().numpy(), I_ref, f"config{cfg} current")
    assert_parity(cond.cpu().numpy(), G_ref, f"config{cfg} conductance")
    h.negf_destroy()


def test_current_of_ideal_tube_on_gpu():
    """Pin on the CUDA path alone: I = (g_s e/h) M (mu_S - mu_D) with M = 2 open modes (library units:
    eV), both chemical potentials inside the first plateau of the ideal (17,0) tube."""
    import torch
    from paper_2407_14633_b200 import Negf
    mu_s, mu_d, kT = 0.42, 0.36, 0.004
    wl = wlmod.make_config(2, N=16, K_neq=160, K_eq=0)
    wl.phi[:] = 0.0
    wl.mu_s, wl.mu_d, wl.kT = mu_s, mu_d, kT
    wl.z_neq, wl.w_neq = wlmod.real_axis_gauss_legendre(mu_d - 14 * kT, mu_s + 14 * kT, 160, eta=1e-9)
    h = Negf.from_workload(wl)
    h.negf_set_potential(torch.tensor(wl.phi, dtype=torch.float64, device="cuda"))
    cur = torch.empty(1, dtype=torch.float64, device="cuda")
    h.negf_current(cur, None)
    h.negf_sync()
    assert abs(cur.item() - 2.0 * (mu_s - mu_d)) < 1e-6
    h.negf_destroy()


@pytest.mark.parametrize("cfg,kw", [(2, dict(N=21, K_neq=8, K_eq=8)), (3, dict(N=10, K_neq=8, K_eq=8)),
                                    (4, dict(C=2, N=9, K_neq=8, K_eq=8))])
def test_equilibrium_only_and_neutral_contours_vs_definition(cfg, kw):
    """the equilibrium-only contour (two arcs + the enclosed Fermi poles
    z_p = mu + i pi kT (2p+1) as extra (z, W) points, no real-axis points) and the neutral-charge
    contour run through the same kernels; charge per ring against the dense definition."""
    base = wlmod.make_config(cfg, **kw)
    for wl in (wlmod.equilibrium_variant(base, mu=-0.03, K_eq=24), wlmod.neutral_variant(base, K_eq=24)):
        assert wl.K_neq == 0
        n_ref, _ = od.charge_and_transmission(wl)
        import torch
        from paper_2407_14633_b200 import Negf
        h = Negf.from_workload(wl)
        n = torch.empty((wl.C, wl.N), dtype=torch.float64, device="cuda")
        h.negf_set_potential(torch.tensor(wl.phi, dtype=torch.float64, device="cuda"))
        h.negf_charge(n)
        h.negf_sync()
        assert_parity(n.cpu().numpy(), n_ref, f"{wl.name} charge")
        h.negf_destroy()


def test_equilibrium_only_equals_two_part_on_gpu():
    """The 8(f)-3 pin on the CUDA path alone: equilibrium-only contour == two-part path at mu_S = mu_D
    (to the 2 eta G G^dagger term, ~1e-7) on a chain whose band edges are far from the Fermi window."""
    import torch
    from paper_2407_14633_b200 import Negf
    base = wlmod.make_config(1, N=40, K_neq=8)
    mu, e_b = 0.3, -6.0
    weq = wlmod.equilibrium_variant(base, mu=mu, K_eq=48, e_b=e_b)
    w2 = wlmod.two_part_equilibrium_variant(base, mu=mu, K_eq=48, K_neq=160)
    w2.z_eq, w2.w_eq = wlmod.contour_semicircle(e_b, mu - wlmod.F_TAIL * base.kT, 48, mu, base.kT)
    out = []
    for wl in (weq, w2):
        h = Negf.from_workload(wl)
        n = torch.empty((wl.C, wl.N), dtype=torch.float64, device="cuda")
        h.negf_set_potential(torch.tensor(wl.phi, dtype=torch.float64, device="cuda"))
        h.negf_charge(n)
        h.negf_sync()
        out.append(n.cpu().numpy())
        h.negf_destroy()
    assert np.max(np.abs(out[0] - out[1]) / out[1]) < 2e-6


def test_table2_long_channel_workload():
    """SURVEY 8(f)-4 workload (Table 2): N = 524 288 rings, 90 contour points
    (equilibrium contour with the Fermi poles), 8 doubly-degenerate modes.  Shrunk (N = 300) against the
    dense definition in full; at FULL length in the launch configuration bench.py times, the charge of
    sampled (mode, contour point) subsets against the C++ tier O3 oracle, every ring."""
    import torch
    from paper_2407_14633_b200 import Negf
    from oracle import negf_rgf_omp as omp

    def gpu_charge(wl):
        h = Negf.from_workload(wl)
        n = torch.empty((wl.C, wl.N), dtype=torch.float64, device="cuda")
        h.negf_set_potential(torch.tensor(wl.phi, dtype=torch.float64, device="cuda"))
        h.negf_charge(n)
        h.negf_sync()
        h.negf_destroy()
        return n.cpu().numpy()

    small = wlmod.table2(N=300)
    assert small.K_eq == 90 and small.K_neq == 0 and small.n_modes == 8
    n_ref, _ = od.charge_and_transmission(small)
    assert_parity(gpu_charge(small), n_ref, "table2 shrunk charge")
    full = wlmod.table2()
    assert full.N == 524288
    n_full = gpu_charge(full)                      # the full launch configuration: all 720 chains
    assert np.all(np.isfinite(n_full)) and np.all(n_full > 0)
    # linear in the contour points: the sampled subsets are themselves valid workloads
    sub = full.subset(eq_idx=[0, 11, 22, 23, 55, 86, 87, 89])
    sub.coup_even, sub.coup_odd, sub.mode_weight, sub.n_modes = (full.coup_even[[0, 7]], full.coup_odd[[0, 7]],
                                                                 full.mode_weight[[0, 7]], 2)
    n_sub = gpu_charge(sub)
    n_ref, _ = omp.charge_and_transmission(sub)
    assert_parity(n_sub, n_ref, "table2 full-length charge of sampled chains, every ring")


@pytest.mark.parametrize("cfg,kw,ring", [(2, dict(N=37, K_neq=45, K_eq=4), 18), (2, dict(N=37, K_neq=45, K_eq=4), 0),
                                         (1, dict(N=30, K_neq=33), 29), (3, dict(N=9, K_neq=10, K_eq=2), 4),
                                         (4, dict(C=2, N=8, K_neq=9, K_eq=2), 7)])
def test_integrand_probe_and_peak_vs_definition(cfg, kw, ring):
    """SURVEY 8(f)-2, device side: the integrand A_1 F_1 + A_2 F_2 at a probe ring as a function
    of energy and the position of its peak, against the dense definition; the charge must not depend on
    the probe; the host-side refresh then puts the dense segment around the peak."""
    import torch
    from paper_2407_14633_b200 import Negf
    wl = wlmod.make_config(cfg, **kw)
    I_ref = od.integrand_dense(wl, ring)
    h = Negf.from_workload(wl)
    phi = torch.tensor(wl.phi, dtype=torch.float64, device="cuda")
    n0 = torch.empty((wl.C, wl.N), dtype=torch.float64, device="cuda")
    n1 = torch.empty_like(n0)
    h.negf_set_potential(phi)
    h.negf_charge(n0)
    h.negf_set_probe(ring)
    h.negf_charge(n1)
    I = torch.empty((wl.C, wl.K_neq), dtype=torch.float64, device="cuda")
    kp = torch.empty(wl.C, dtype=torch.int32, device="cuda")
    Ep = torch.empty(wl.C, dtype=torch.float64, device="cuda")
    h.negf_integrand_peak(I, kp, Ep)
    h.negf_sync()
    assert torch.equal(n0, n1)                                        # the probe does not touch the charge
    assert_parity(I.cpu().numpy(), I_ref, f"config{cfg} integrand at ring {ring}")
    assert np.array_equal(kp.cpu().numpy(), np.argmax(I_ref, axis=1))
    assert np.array_equal(Ep.cpu().numpy(), wl.z_neq.real[np.argmax(I_ref, axis=1)])
    e_s, l1, l2 = wlmod.refine_segment_limits(wl.z_neq.real, I.cpu().numpy()[0], wl.kT)
    assert e_s == Ep.cpu().numpy()[0] and l1 < e_s < l2
    h.negf_set_probe(-1)
    with pytest.raises(Exception):
        h.negf_integrand_peak(I, kp, Ep)
    h.negf_destroy()


def _charge_with_env(wl, env):
    import os
    import torch
    from paper_2407_14633_b200 import Negf
    old = {k: os.environ.get(k) for k in env}
    os.environ.update(env)
    try:
        h = Negf.from_workload(wl)
    finally:
        for k, v in old.items():
            if v is None:
                os.environ.pop(k, None)
            else:
                os.environ[k] = v
    n = torch.empty((wl.C, wl.N), dtype=torch.float64, device="cuda")
    h.negf_set_potential(torch.tensor(wl.phi, dtype=torch.float64, device="cuda"))
    h.negf_charge(n)
    h.negf_sync()
    plan = h.negf_get_plan()
    h.negf_destroy()
    return n.cpu().numpy(), plan


@pytest.mark.parametrize("N,seg_len", [(300, 7), (257, 256), (64, 1), (2, 5), (3, 1), (1000, 33)])
def test_parallel_in_N_contour_path_vs_definition_and_serial(N, seg_len):
    """the segmented (parallel-in-N) contour half-sweeps -- segment transfer products, serial
    pass over the segment starts, parallel re-run of every segment -- against the dense definition
    (N <= 300) and against the serial pass of the same library: several segments, a ragged last segment,
    one-step segments, N = 2 and 3, both contour directions, config 2's mix of real-axis and contour tasks."""
    wl = wlmod.table2(N=N) if N != 1000 else wlmod.make_config(2, N=1000, K_neq=64, K_eq=24)
    n_seg, plan_seg = _charge_with_env(wl, {"NEGF_SEG_MIN_RINGS": "2", "NEGF_SEG_LEN": str(seg_len)})
    n_ser, plan_ser = _charge_with_env(wl, {"NEGF_SEG_MIN_RINGS": "1000000000"})
    if N >= 3:
        assert plan_seg["kernel_launches"] == plan_ser["kernel_launches"] + 2      # 3 contour kernels instead of 1
    assert_parity(n_seg, n_ser, f"segmented vs serial contour pass, N={N}", rtol=1e-12)
    if N <= 300:
        n_ref, _ = od.charge_and_transmission(wl)
        assert_parity(n_seg, n_ref, f"segmented contour pass vs dense definition, N={N}")
