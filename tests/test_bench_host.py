"""Host-side logic of bench.py that needs no GPU: the N>1 aggregation (replicas only) over a
world_size-2 gloo group, and the --impl reference contract under a multi-rank launch."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

_WORKER = r"""
import os, sys, json
sys.path.insert(0, {root!r})
import torch.distributed as dist
import bench
rank = int(os.environ["RANK"])
dist.init_process_group("gloo", rank=rank, world_size=2)
# rank 0 took 10 ms for 1000 particles, rank 1 took 14 ms for 1500
ms, n = bench.reduce_over_ranks(10.0 if rank == 0 else 14.0, 1000 if rank == 0 else 1500, 2, "cpu")
print(json.dumps({{"rank": rank, "ms": ms, "n": n}}))
dist.destroy_process_group()
"""


def _spawn(code, extra_env=None, args=()):
    procs = []
    for rank in range(2):
        env = dict(os.environ, RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1",
                   MASTER_PORT="29617", **(extra_env or {}))
        procs.append(subprocess.Popen([sys.executable, *code, *args], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.PIPE, text=True, cwd=ROOT))
    outs = [p.communicate(timeout=300) for p in procs]
    for p, (o, e) in zip(procs, outs):
        assert p.returncode == 0, e
    return [o for o, _ in outs]


def test_replica_aggregation_over_gloo_world_size_2():
    outs = _spawn(["-c", _WORKER.format(root=ROOT)])
    for o in outs:
        r = json.loads(o.strip().splitlines()[-1])
        assert r["ms"] == 14.0 and r["n"] == 2500.0           # max over ranks, sum over ranks


def test_reference_arm_prints_one_line_on_rank0_only():
    outs = _spawn([os.path.join(ROOT, "bench.py")], args=("--impl", "reference", "--gpus", "2", "--steps", "1",
                                                          "--warmup", "0", "--ref-side", "12"))
    assert outs[1].strip() == ""
    line = json.loads(outs[0].strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["cpu_baseline"]["kind"] == "oracle" and line["value"] > 0
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["unit"] == "particle-updates/s"
