"""The N > 1 plumbing of bench.py on CPU: world_size 2 over gloo (the path has no exchange step — "replicas only",
DESIGN.md §9 — so the only collective is the max-over-ranks time / sum-over-ranks units of the report)."""
import json
import os
import socket
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import os, sys, json
sys.path.insert(0, os.environ["BS_ROOT"])
import torch.distributed as dist
import bench
rank, local_rank, world = bench.dist_env()
dist.init_process_group("gloo")
ms, units = bench.aggregate(10.0 + 5.0 * rank, 100.0 * (rank + 1), world, device="cpu", backend_ready=True)
solo = bench.aggregate(3.0, 7.0, 1, device="cpu", backend_ready=True)
print(json.dumps({"rank": rank, "local_rank": local_rank, "world": world, "ms": ms, "units": units, "solo": solo}))
dist.destroy_process_group()
"""


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _env(rank, world, port):
    env = dict(os.environ, RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE=str(world), MASTER_ADDR="127.0.0.1",
               MASTER_PORT=str(port), BS_ROOT=ROOT)
    return env


def test_aggregate_takes_max_time_and_sum_of_units_over_two_ranks():
    port = _free_port()
    procs = [subprocess.Popen([sys.executable, "-c", WORKER], env=_env(r, 2, port), stdout=subprocess.PIPE,
                              stderr=subprocess.PIPE, text=True) for r in range(2)]
    outs = [p.communicate(timeout=180) for p in procs]
    for p, (so, se) in zip(procs, outs):
        assert p.returncode == 0, se[-2000:]
    rows = [json.loads(so.strip().splitlines()[-1]) for so, _ in outs]
    for r, row in enumerate(rows):
        assert (row["rank"], row["local_rank"], row["world"]) == (r, r, 2)
        assert row["ms"] == 15.0 and row["units"] == 300.0       # max over ranks, sum over ranks
        assert row["solo"] == [3.0, 7.0]


def test_reference_arm_runs_on_rank0_only():
    port = _free_port()
    cmd = [sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1", "--warmup", "0",
           "--workload", "2", "--sample-mb", "4"]
    procs = [subprocess.Popen(cmd, env=_env(r, 2, port), stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True)
             for r in range(2)]
    outs = [p.communicate(timeout=300) for p in procs]
    for p, (so, se) in zip(procs, outs):
        assert p.returncode == 0, se[-2000:]
    assert outs[1][0].strip() == ""                               # the other rank exits 0 without work
    line = json.loads(outs[0][0].strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["n_gpus"] == 2 and line["value"] > 0
    assert line["cpu_baseline"]["kind"] == "oracle" and line["e2e"]["h2d_bytes_per_step"] == 0
