"""GPU parity, block (real-space, n x n) path: shrunk and sampled versions of BASELINE.json
configs[2..4] through the C-ABI against the CPU oracle, element by element (north_star: 1e-10
relative).  Dense inversion (tier O1) on shrunk devices, the paper's recursion (tier O3) at full
device length, random non-symmetric complex blocks to catch dagger / transpose / ordering mistakes,
and the forced column-search path of the in-register Gauss-Jordan."""
import numpy as np
import pytest

import workloads as wlmod
from oracle import negf_dense as od
from oracle import negf_rgf as orgf
from oracle import negf_rgf_omp as omp
from tests.parity import assert_parity

pytestmark = pytest.mark.gpu


def _gpu_run(wl, want_plan=False, **kw):
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
    plan = h.negf_get_plan()
    h.negf_destroy()
    return out + (plan,) if want_plan else out


def _random_block_workload(n, N, K_neq, K_eq, seed, C=1, sparse=False, eta=1e-3):
    """Device with random complex non-Hermitian coupling blocks (not a CNT): every dagger,
    transpose and left/right ordering in the recursion matters.  Such a random chain has
    localised states inside the window whose only broadening is eta, i.e. G ~ 1/(i eta) and a
    condition number ~ 1/eta for T(E) with respect to rounding in Sigma (measured: 1e-15 relative
    noise on Sigma moves T by 4e-8 at eta = 1e-6).  This is a structure test, so it runs at
    eta = 1e-3, where both sides can deliver 1e-10."""
    rng = np.random.default_rng(seed)
    base = wlmod.make_config(3, N=N, K_neq=max(K_neq, 1), K_eq=K_eq)
    if K_neq == 0:
        base = base.subset(neq_idx=[])

    def blockmat():
        m = rng.normal(size=(n, n)) + 1j * rng.normal(size=(n, n))
        if sparse:
            m = m * (rng.uniform(size=(n, n)) < 0.4)
            m[0, n - 1] = 1.0 + 0.5j            # keep it connected
        return (0.9 * m).astype(np.complex128)

    phi = 0.3 * rng.normal(size=(C, N))
    z_neq = (base.z_neq.real + 1j * eta).astype(np.complex128)
    return wlmod.Workload(
        name=f"random_n{n}", kind="block", C=C, N=N, n=n, n_modes=1,
        coup_even=blockmat(), coup_odd=blockmat(), mode_weight=np.ones(1), phi=phi,
        z_eq=base.z_eq, w_eq=base.w_eq, z_neq=z_neq, w_neq=base.w_neq, lead_kind=1, seed=seed,
        eta=eta)


@pytest.mark.parametrize("N,K_neq,K_eq", [(12, 8, 4), (33, 37, 17), (2, 5, 3), (7, 16, 0), (9, 0, 6)])
def test_config3_shrunk_vs_dense_definition(N, K_neq, K_eq):
    """17 x 17 blocks; several CTAs per direction (K > 15) with ragged tails, even and odd N (both
    parities of the right lead), the degenerate N = 2, contour-only and real-axis-only handles."""
    wl = wlmod.make_config(3, N=N, K_neq=max(K_neq, 1), K_eq=K_eq)
    if K_neq == 0:
        wl = wl.subset(neq_idx=[])
    n_ref, T_ref = od.charge_and_transmission(wl)
    n, T = _gpu_run(wl)
    assert_parity(n, n_ref, "config3-shrunk charge")
    if K_neq:
        assert_parity(T, T_ref, "config3-shrunk T(E)")


@pytest.mark.parametrize("n,sparse", [(2, False), (3, False), (4, True), (5, False), (8, True), (17, False),
                                      (17, True)])
def test_random_complex_blocks_vs_dense_definition(n, sparse):
    # n = 17 takes the eight-lanes-per-task forward kernel and the warp-level Sancho-Rubio inversions with dense
    # (padded-row width 17: three CTAs per SM) and sparse random complex couplings, two channels
    # (n = 17: 26 rings of random 17 x 17 blocks are worse conditioned than the small cases -- at eta = 1e-3 this
    # round's kernels give T(E) to 1.5e-10 and round 1's to 5.2e-10 -- so the structure test runs at eta = 1e-2)
    wl = _random_block_workload(n, N=9 + n, K_neq=40, K_eq=11, seed=100 + n, C=2, sparse=sparse,
                                eta=1e-2 if n == 17 else 1e-3)
    n_ref, T_ref = od.charge_and_transmission(wl)
    n_gpu, T_gpu = _gpu_run(wl)
    assert_parity(n_gpu, n_ref, f"random n={n} charge")
    assert_parity(T_gpu, T_ref, f"random n={n} T(E)")


def test_forced_column_search_matches():
    """negf_config.pivot_theta = 1e150 rejects every diagonal candidate, so every elimination step
    takes the partial-pivoting search path; the results must still match the dense definition."""
    wl3 = wlmod.make_config(3, N=10, K_neq=20, K_eq=5)
    wlr = _random_block_workload(5, N=11, K_neq=17, K_eq=4, seed=77)
    wl17 = _random_block_workload(17, N=7, K_neq=11, K_eq=3, seed=78, sparse=True)
    for w in (wl3, wlr, wl17):
        n_ref, T_ref = od.charge_and_transmission(w)
        n, T = _gpu_run(w, pivot_theta=1e150)
        assert_parity(n, n_ref, f"{w.name} forced-search charge")
        assert_parity(T, T_ref, f"{w.name} forced-search T(E)")


@pytest.mark.parametrize("theta", [0.05, 0.25, 0.6])
def test_threshold_pivoting_paths_of_the_n17_forward_kernel(theta):
    """block_fwd17.cu at n = 17 has three pivoting paths: diagonal candidates, the in-register column search
    (candidate rejected by the row-norm test) and the shared-memory slow path (corner d rejected as first
    pivot; pivot_theta = 1e150 above sends every ring there).  Large but finite thresholds reject a good share
    of the diagonal candidates while the corner still passes for part of the warps, so the column search, the
    permutation through shared memory and mixed warps (tasks on different paths) all run; results must match
    the dense definition.  Real-space tube and random sparse non-symmetric complex couplings."""
    wl3 = wlmod.make_config(3, N=12, K_neq=37, K_eq=5)
    wl17 = _random_block_workload(17, N=9, K_neq=21, K_eq=3, seed=178, sparse=True)
    for w in (wl3, wl17):
        n_ref, T_ref = od.charge_and_transmission(w)
        n, T = _gpu_run(w, pivot_theta=theta)
        assert_parity(n, n_ref, f"{w.name} theta={theta} charge")
        assert_parity(T, T_ref, f"{w.name} theta={theta} T(E)")


def test_integrand_probe_generic_block_sizes():
    """SURVEY 8(f)-2 on the SIMT way back of the generic block sizes (n != 17): integrand at a probe ring
    and its peak against the dense definition, random non-symmetric complex blocks."""
    import torch
    from paper_2407_14633_b200 import Negf
    for n, ring in ((5, 3), (3, 0), (8, 6)):
        wl = _random_block_workload(n, N=7, K_neq=12, K_eq=2, seed=90 + n, C=2)
        I_ref = od.integrand_dense(wl, ring)
        h = Negf.from_workload(wl)
        h.negf_set_potential(torch.tensor(wl.phi, dtype=torch.float64, device="cuda"))
        h.negf_set_probe(ring)
        I = torch.empty((wl.C, wl.K_neq), dtype=torch.float64, device="cuda")
        kp = torch.empty(wl.C, dtype=torch.int32, device="cuda")
        h.negf_integrand_peak(I, kp, None)
        h.negf_sync()
        assert_parity(I.cpu().numpy(), I_ref, f"random n={n} integrand at ring {ring}")
        assert np.array_equal(kp.cpu().numpy(), np.argmax(I_ref, axis=1))
        h.negf_destroy()


def test_config4_shrunk_multi_channel():
    wl = wlmod.make_config(4, C=3, N=14, K_neq=19, K_eq=5)
    n_ref, T_ref = od.charge_and_transmission(wl)
    n, T = _gpu_run(wl)
    assert_parity(n, n_ref, "config4-shrunk charge")
    assert_parity(T, T_ref, "config4-shrunk T(E)")


def test_real_space_equals_sum_of_modes_on_gpu():
    """Pin P7 on the GPU: the block path on the (17,0) real-space tube reproduces the scalar path
    on its 17 mode chains (ring-uniform potential => block-circulant tube)."""
    wl = wlmod.make_config(3, N=40, K_neq=48, K_eq=8)
    twin = wlmod.scalar_twin(wl)
    n_b, T_b = _gpu_run(wl)
    n_s, T_s = _gpu_run(twin)
    assert_parity(n_b, n_s, "block vs modes charge")
    assert_parity(T_b, T_s, "block vs modes T(E)", rtol=2e-10)   # both sides SR/closed-form limited


def test_workspace_tiling_gives_identical_results(monkeypatch):
    """A small workspace cap forces several sweep launches (contour pairs and real-axis CTAs in
    different launches); results must be bit-identical.  (The overlap plan is switched off on both sides:
    it groups the Sancho-Rubio tasks differently, which moves results by ~1e-12 -- the next test.)"""
    monkeypatch.setenv("NEGF_FORCE_OVERLAP", "0")
    wl = wlmod.make_config(3, N=16, K_neq=50, K_eq=20)
    n1, T1, plan1 = _gpu_run(wl, want_plan=True)
    slot = 16 * 17 * 256 * 16
    n2, T2, plan2 = _gpu_run(wl, want_plan=True, workspace_bytes=4 * slot)
    assert plan2["n_batches"] > plan1["n_batches"] >= 1
    assert np.array_equal(n1, n2) and np.array_equal(T1, T2)


def test_overlap_plan_gives_identical_results():
    """The overlap plan of config 3 (contour half-sweeps on a side stream beside the self-energies of the
    real-axis energies, real-axis CTAs in their own launch) forced on a small device: same results as the
    single-launch plan (to rounding: the two Sancho-Rubio launches group the tasks into CTAs differently, and
    a task polishes as long as its CTA-mates do), also when negf_set_potential is called twice before
    negf_charge and when the sweep is re-run for a probe."""
    import os
    import torch
    from paper_2407_14633_b200 import Negf
    wl = wlmod.make_config(3, N=14, K_neq=30, K_eq=9)
    out = {}
    for mode in ("0", "1"):
        os.environ["NEGF_FORCE_OVERLAP"] = mode
        try:
            h = Negf.from_workload(wl)
        finally:
            del os.environ["NEGF_FORCE_OVERLAP"]
        phi = torch.tensor(wl.phi, dtype=torch.float64, device="cuda")
        n = torch.empty((wl.C, wl.N), dtype=torch.float64, device="cuda")
        T = torch.empty((wl.C, wl.K_neq), dtype=torch.float64, device="cuda")
        h.negf_set_potential(phi * 0.5)            # overwritten before any charge: the stale contour sweep must be joined
        h.negf_set_potential(phi)
        h.negf_charge(n)
        h.negf_transmission(T)
        h.negf_sync()
        a = (n.cpu().numpy().copy(), T.cpu().numpy().copy())
        h.negf_set_probe(3)                         # re-runs the sweep for the same potential
        h.negf_charge(n)
        h.negf_sync()
        assert np.array_equal(a[0], n.cpu().numpy())
        plan = h.negf_get_plan()
        h.negf_destroy()
        out[mode] = a + (plan["kernel_launches"],)
    assert out["1"][2] == out["0"][2] + 2
    assert_parity(out["1"][0], out["0"][0], "overlap vs single-launch charge", rtol=1e-12)
    assert_parity(out["1"][1], out["0"][1], "overlap vs single-launch T(E)", rtol=1e-10)
    n_ref, T_ref = od.charge_and_transmission(wl)
    assert_parity(out["1"][0], n_ref, "overlap plan charge")
    assert_parity(out["1"][1], T_ref, "overlap plan T(E)")


def test_config3_full_length_sampled_vs_paper_recursion():
    """Full device length (N = 1000, the bench launch geometry: 256-thread CTAs, 15 tasks each) on a
    sample of configs[2]'s energies against tier O3."""
    wl = wlmod.config3()
    rng = np.random.default_rng(11)
    sub = wl.subset(neq_idx=np.sort(rng.choice(wl.K_neq, 20, replace=False)),
                    eq_idx=np.sort(rng.choice(wl.K_eq, 4, replace=False)))
    n_ref, T_ref = orgf.charge_and_transmission(sub, chunk=24)
    n, T = _gpu_run(sub)
    assert_parity(n, n_ref, "config3 sampled charge")
    assert_parity(T, T_ref, "config3 sampled T(E)")


def test_sancho_rubio_iterations_and_nonconvergence():
    import torch
    from paper_2407_14633_b200 import Negf, NegfError
    wl = wlmod.make_config(3, N=8, K_neq=8, K_eq=2)
    h = Negf.from_workload(wl)
    phi = torch.tensor(wl.phi, dtype=torch.float64, device="cuda")
    h.negf_set_potential(phi)
    h.negf_sync()
    its = h.negf_get_plan()["max_sr_iterations"]
    assert 5 <= its <= 60          # eta = 1e-6: ~20 doublings, + 2 extra passes
    h.negf_destroy()
    wl.sr_maxit = 3
    h = Negf.from_workload(wl)
    h.negf_set_potential(phi)
    with pytest.raises(NegfError) as ei:
        h.negf_sync()
    assert ei.value.status == 4    # NEGF_ENOCONV
    h.negf_destroy()


def test_unsupported_block_size_fails_loudly():
    from paper_2407_14633_b200 import NegfError
    wl = _random_block_workload(7, N=6, K_neq=4, K_eq=2, seed=5)
    with pytest.raises(NegfError) as ei:
        _gpu_run(wl)
    assert ei.value.status == 1    # NEGF_EINVAL, no silent fallback


def test_self_energy_kernel_vs_oracle():
    """Step a1b in isolation: Sigma_L, Sigma_R of the Sancho-Rubio kernel against the oracle's
    decimation for every energy (contour first), both lead parities and both ends' potentials."""
    import torch
    from oracle import selfenergy as se
    from paper_2407_14633_b200 import Negf
    for N in (8, 9):
        wl = wlmod.make_config(4, C=2, N=N, K_neq=33, K_eq=6)
        h = Negf.from_workload(wl)
        h.negf_set_potential(torch.tensor(wl.phi, dtype=torch.float64, device="cuda"))
        K = wl.K_eq + wl.K_neq
        sig = torch.empty((wl.C, K, 2, wl.n * wl.n), dtype=torch.complex128, device="cuda")
        h.negf_self_energy(sig)
        h.negf_sync()
        sig = sig.cpu().numpy().reshape(wl.C, K, 2, wl.n, wl.n)
        zall = np.concatenate([wl.z_eq, wl.z_neq])
        for c in range(wl.C):
            U = -wl.phi[c]
            sL, sR, _ = se.sigma_block(zall, wl.coup_even, wl.coup_odd, wl.N, U[0], U[-1])
            for lead, ref in ((0, sL), (1, sR)):
                scale = np.abs(ref).max(axis=(1, 2))
                err = np.abs(sig[c, :, lead] - ref).max(axis=(1, 2)) / scale
                assert err.max() < 1e-12, (N, c, lead, err.max())
        h.negf_destroy()


@pytest.mark.parametrize("cfg", [4, 5])
def test_config4_and_5_full_length_sampled_vs_paper_recursion(cfg):
    """configs[3] / configs[4] at their full device length (N = 2000 / 4000) and channel potentials, on
    sampled channels and energies the oracle (tier O3) can do in seconds."""
    wl = wlmod.make_config(cfg)
    rng = np.random.default_rng(40 + cfg)
    sub = wl.subset(neq_idx=np.sort(rng.choice(wl.K_neq, 5, replace=False)),
                    eq_idx=np.sort(rng.choice(wl.K_eq, 3, replace=False)),
                    channels=np.sort(rng.choice(wl.C, 2, replace=False)))
    n_ref, T_ref = orgf.charge_and_transmission(sub, chunk=8)
    n, T = _gpu_run(sub)
    assert_parity(n, n_ref, f"config{cfg} sampled charge")
    assert_parity(T, T_ref, f"config{cfg} sampled T(E)")


def test_self_energy_next_to_a_segment_pole_regression():
    """z - U_end = -0.33765527 + 1e-6 i sits ~1e-9 from a pole of an isolated 2^k-cell segment of the
    decimation: the raw result is off by ~4e-7 and the Newton doubling sum used to diverge (NaN
    self-energy in the config 4 loop).  The kernel must redo such a task and still match the oracle."""
    import torch
    from oracle import selfenergy as se
    from paper_2407_14633_b200 import Negf
    z0 = -0.3386878743069309 + 1e-6j
    U0 = -0.001032601892690806
    # second case (config 5 loop, right lead): the decimation itself breaks down to NaN, which fmax-based
    # convergence tests used to swallow
    z1 = 0.33736573920690816 + 1e-6j
    U1 = -0.0002902289467536259
    wl = wlmod.make_config(3, N=4, K_neq=4, K_eq=0)
    wl.z_neq = np.array([z0, z0 + 1e-9, z0 - 1e-7, z1])
    wl.w_neq = np.ones(4)
    wl.phi = np.array([[-U0, -U0, -U1, -U1]])
    h = Negf.from_workload(wl)
    h.negf_set_potential(torch.tensor(wl.phi, dtype=torch.float64, device="cuda"))
    sig = torch.empty((1, 4, 2, wl.n * wl.n), dtype=torch.complex128, device="cuda")
    h.negf_self_energy(sig)
    h.negf_sync()
    sig = sig.cpu().numpy().reshape(4, 2, wl.n, wl.n)
    assert np.all(np.isfinite(sig.view(np.float64)))
    sL, sR, _ = se.sigma_block(wl.z_neq, wl.coup_even, wl.coup_odd, wl.N, U0, U1)
    for lead, ref in ((0, sL), (1, sR)):
        err = np.abs(sig[:, lead] - ref).max() / np.abs(ref).max()
        assert err < 1e-11, (lead, err)
    h.negf_destroy()


@pytest.mark.parametrize("N,K_neq,K_eq", [(2, 9, 3), (3, 8, 0), (5, 0, 6), (31, 15, 2)])
def test_config3_degenerate_shapes(N, K_neq, K_eq):
    """Shortest devices (N = 2, 3: both leads on adjacent rings; odd N flips the right lead's bond),
    real-axis-only and contour-only handles, one more task than a CTA holds (15 = 2 x 7 + 1)."""
    wl = wlmod.make_config(3, N=N, K_neq=max(K_neq, 1), K_eq=K_eq)
    if K_neq == 0:
        wl = wl.subset(neq_idx=[])
    n_ref, T_ref = od.charge_and_transmission(wl)
    n, T = _gpu_run(wl)
    assert_parity(n, n_ref, "config3-degenerate charge")
    if K_neq:
        assert_parity(T, T_ref, "config3-degenerate T(E)")


def test_ideal_tube_integer_transmission_and_reciprocity_on_gpu():
    """Pins P4 / P6 on the CUDA block path itself (no oracle involved): an ideal (17,0) tube has
    T(E) = number of open subbands, |t| |1 - 2 cos(pi q/17)| < |E| < |t| |1 + 2 cos(pi q/17)|, to O(N eta);
    (eta = 1e-6 as in every config)
    and for real H the left-to-right and right-to-left columns give the same transmission, which here
    shows as T being independent of which end the potential step sits on (mirror device)."""
    import torch
    from paper_2407_14633_b200 import Negf
    E = np.array([0.2, 0.3, 0.6, 1.2, 3.0])
    q = np.arange(17)
    lo = 2.5 * np.abs(1.0 - 2.0 * np.abs(np.cos(np.pi * q / 17)))
    hi = 2.5 * np.abs(1.0 + 2.0 * np.abs(np.cos(np.pi * q / 17)))
    expected = np.array([np.sum((lo < e) & (e < hi)) for e in E], dtype=float)
    wl = wlmod.make_config(3, N=24, K_neq=len(E), K_eq=0)
    wl.z_neq = (E + 1e-6j).astype(np.complex128)
    wl.w_neq = np.ones(len(E))
    wl.phi[:] = 0.0
    _, T = _gpu_run(wl)
    assert np.allclose(T[0], expected, rtol=0, atol=1e-3), (T[0], expected)     # O(N eta / |t|) per mode
    # mirror symmetry: a potential profile and its mirror image transmit equally (real symmetric H)
    rng = np.random.default_rng(5)
    wl.phi[0] = 0.2 * rng.normal(size=wl.N)
    wl.z_neq = (E + 1e-6j).astype(np.complex128)
    _, T1 = _gpu_run(wl)
    wl.phi[0] = wl.phi[0][::-1].copy()
    _, T2 = _gpu_run(wl)
    assert_parity(T1, T2, "mirror device T(E)", rtol=1e-9)


def test_config3_full_launch_configuration():
    """configs[2] at FULL size in the launch configuration bench.py times (2112 energies x 1000 rings):
    every element of the per-ring charge and of T(E) against the C++/OpenMP tier O3 oracle
    (oracle/negf_rgf_omp.cpp: Algorithm 2 + Algorithm 1 with its own Sancho-Rubio, pinned to the dense
    definition and to banded LU in the CPU suite).  Passage: Alg.1-2; eq.(4), (5)."""
    wl = wlmod.config3()
    n, T = _gpu_run(wl)
    n_ref, T_ref = omp.charge_and_transmission(wl)
    assert_parity(n, n_ref, "config3 full-size charge, every ring")
    assert_parity(T, T_ref, "config3 full-size T(E), every energy")


def test_config4_full_launch_configuration():
    """configs[3] at full size (16 channels x 2000 rings x 4160 energies, batched sweep launches): ONE WHOLE
    CHANNEL -- all 4160 energies, every ring, every T(E) -- of the full 16-channel run against the C++
    tier O3 oracle; for the other channels T(E) at sampled energies, and bounds on the charge."""
    wl = wlmod.config4()
    n, T = _gpu_run(wl)
    assert np.all(np.isfinite(n)) and np.all(np.isfinite(T))
    assert np.all(n > 0.0) and np.all(n < 2.0 * wl.n)            # 0 .. deg * 17 electrons per ring
    c = 11                                                       # a channel in the middle of the batch order
    n_ref, T_ref = omp.charge_and_transmission(wl, channels=[c])
    assert_parity(n[c], n_ref[c], f"config4 full-size charge of channel {c}, every ring")
    assert_parity(T[c], T_ref[c], f"config4 full-size T(E) of channel {c}, every energy")
    rng = np.random.default_rng(44)
    ks = np.sort(rng.choice(wl.K_neq, 4, replace=False))
    cs = np.array([0, 15])                                       # first and last channel of the batch order
    sub = wl.subset(neq_idx=ks, eq_idx=[], channels=cs)
    _, T_s = omp.charge_and_transmission(sub)
    assert_parity(T[np.ix_(cs, ks)], T_s, "config4 full-run T(E) at sampled channels / energies")


def test_config5_full_launch_configuration():
    """configs[4] at full size (64 channels x 4000 rings x 8320 energies, one negf_charge of the loop):
    sampled T(E) against the oracle, bounds."""
    wl = wlmod.config5()
    n, T = _gpu_run(wl)
    assert np.all(np.isfinite(n)) and np.all(np.isfinite(T))
    assert np.all(n > 0.0) and np.all(n < 2.0 * wl.n)
    rng = np.random.default_rng(55)
    ks = np.sort(rng.choice(wl.K_neq, 3, replace=False))
    cs = np.sort(rng.choice(wl.C, 2, replace=False))
    sub = wl.subset(neq_idx=ks, eq_idx=[], channels=cs)
    _, T_ref = omp.charge_and_transmission(sub)
    assert_parity(T[np.ix_(cs, ks)], T_ref, "config5 full-run T(E) at sampled channels / energies")
