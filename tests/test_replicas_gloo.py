"""-m "not gpu": the multi-GPU path of bench.py ("replicas only") on CPU: two gloo
ranks join a 127.0.0.1 rendezvous, each reports a different step time, and the job's value must come
from the slowest one; --impl reference prints on rank 0 only."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
torch = pytest.importorskip("torch")

WORKER = r"""
import os, sys, json
sys.path.insert(0, %(root)r)
import bench
dist, rank, world = bench.init_replicas("gloo")
assert world == 2 and dist is not None
dist.barrier()
ms = bench.max_over_ranks(dist, 4.0 if rank == 0 else 10.0)
dist.barrier()
print(json.dumps({"rank": rank, "ms": ms, "value": bench.replicas_value(world, ms)}))
dist.destroy_process_group()
"""


def _run_ranks(code, port):
    procs = []
    for r in range(2):
        env = dict(os.environ, RANK=str(r), LOCAL_RANK=str(r), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port), OMP_NUM_THREADS="1")
        procs.append(subprocess.Popen([sys.executable, "-c", code], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.PIPE, text=True))
    outs = []
    for p in procs:
        o, e = p.communicate(timeout=240)
        assert p.returncode == 0, e
        outs.append(o)
    return outs


def test_two_gloo_ranks_take_the_slowest_time():
    outs = _run_ranks(WORKER % {"root": ROOT}, 29611)
    recs = [json.loads(o.strip().splitlines()[-1]) for o in outs]
    for rec in recs:
        assert rec["ms"] == 10.0                       # max over ranks, on every rank
        assert rec["value"] == pytest.approx(200.0)     # 2 replicas x (1000 / 10 ms) solves/s
    assert bench_single_rank_value() == pytest.approx(250.0)


def bench_single_rank_value():
    sys.path.insert(0, ROOT)
    import bench
    return bench.replicas_value(1, bench.max_over_ranks(None, 4.0))


def test_reference_arm_prints_on_rank_zero_only():
    """`bench.py --impl reference` under a 2-rank launch: rank 1 exits 0 without output."""
    env = dict(os.environ, RANK="1", LOCAL_RANK="1", WORLD_SIZE="2", MASTER_ADDR="127.0.0.1", MASTER_PORT="29612")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                        "--steps", "1", "--warmup", "0"], env=env, capture_output=True, text=True, timeout=240)
    assert r.returncode == 0 and r.stdout.strip() == ""
