"""Host-side logic of the N > 1 bench path with
world_size 2 on the gloo backend: rendezvous from the torchrun environment, max-over-ranks time
and sum-over-ranks units, and the reference arm running on rank 0 only."""
import json
import os
import socket
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import json, os, sys
sys.path.insert(0, os.environ["NEGF_ROOT"])
import bench
rank, world, local = bench.dist_setup(2, backend="gloo")
assert world == 2 and rank == int(os.environ["RANK"])
bench.dist_barrier(world)
ms, units = bench.dist_max_sum(10.0 * (rank + 1), 7.0 + rank, world)
print(json.dumps({"rank": rank, "ms": ms, "units": units}), flush=True)
import torch.distributed as dist
dist.destroy_process_group()
"""


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _launch(code_or_args, port, extra_env=None):
    procs = []
    for rank in range(2):
        env = dict(os.environ, RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE="2",
                   MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), NEGF_ROOT=ROOT,
                   CUDA_VISIBLE_DEVICES="")
        env.update(extra_env or {})
        procs.append(subprocess.Popen([sys.executable, *code_or_args], env=env, cwd=ROOT,
                                      stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True))
    outs = [p.communicate(timeout=600) for p in procs]
    for p, (o, e) in zip(procs, outs):
        assert p.returncode == 0, e[-2000:]
    return [o for o, _ in outs]


def test_max_over_ranks_and_sum_of_units_gloo():
    outs = _launch(["-c", WORKER], _free_port())
    for o in outs:
        d = json.loads(o.strip().splitlines()[-1])
        assert d["ms"] == 20.0 and d["units"] == 15.0


def test_reference_arm_runs_on_rank0_only():
    outs = _launch(["bench.py", "--impl", "reference", "--gpus", "2", "--steps", "1", "--warmup", "0",
                    "--config", "1"], _free_port())
    lines = [json.loads(l) for o in outs for l in o.strip().splitlines() if l.startswith("{")]
    assert len(lines) == 1
    line = lines[0]
    assert line["impl"] == "reference" and line["n_gpus"] == 2 and line["value"] > 0
    assert line["cpu_baseline"]["kind"] == "oracle" and line["e2e"]["h2d_bytes_per_step"] == 0


def test_poisson_stand_in_as_one_sparse_matrix():
    """bench.py applies the Poisson stand-in of config 5 (harness code) as one SpMV; the CSR matrix must
    be the very map of workloads.PoissonStandIn.apply_K, for one and for several channels."""
    import numpy as np
    import torch
    sys.path.insert(0, ROOT)
    import bench
    import workloads as wlmod
    rng = np.random.default_rng(3)
    for C, N in ((1, 23), (4, 17)):
        p = wlmod.PoissonStandIn(kappa=0.2, r=rng.uniform(0.5, 1.0, (max(C - 1, 0), N)), n0=17.0)
        rowptr, cols, vals = p.as_csr(C, N)
        assert rowptr[-1] == len(cols) == len(vals) and np.all(np.diff(rowptr) >= 4)
        # diagonally dominant, off-diagonal row sum <= 0.9 kappa (BASELINE.json configs[4])
        dense = np.zeros((C * N, C * N))
        for i in range(C * N):
            dense[i, cols[rowptr[i]:rowptr[i + 1]]] = vals[rowptr[i]:rowptr[i + 1]]
        assert np.allclose(np.diag(dense), 0.2) and np.all(dense.sum(1) - 0.2 <= 0.9 * 0.2 + 1e-15)
        q = rng.normal(size=(C, N))
        assert np.max(np.abs(dense @ q.ravel() - p.apply_K(q.copy()).ravel())) < 1e-15
        pd = bench.PoissonOnDevice(p, C, N, "cpu")
        phi_ext = torch.tensor(rng.normal(size=(C, N)))
        n = torch.tensor(q + 17.0)
        assert np.max(np.abs(pd.phi_out(phi_ext, n).numpy() - p.phi_out(phi_ext.numpy(), n.numpy()))) < 1e-15
