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
