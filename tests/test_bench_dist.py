"""N>1 path of bench.py on CPU: world_size-2 gloo.  The path is 'replicas only' (no data-path collective):
only the barrier and the max-over-ranks of the device time cross ranks."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import os, sys, json
sys.path.insert(0, %r)
import bench
rank, world = bench.dist_init("gloo")
bench.dist_barrier()
ms = bench.dist_max(10.0 + 5.0 * rank)            # slowest rank sets the time
val = bench.aggregate(ms, 1.0, world)             # replicas: units of all ranks / max time
bench.dist_barrier()
if rank == 0:
    print(json.dumps({"ms": ms, "value": val, "world": world}))
""" % ROOT


def test_two_rank_gloo_max_and_aggregate(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER)
    env = dict(os.environ, MASTER_ADDR="127.0.0.1", MASTER_PORT="29533", WORLD_SIZE="2")
    procs = []
    for r in range(2):
        e = dict(env, RANK=str(r), LOCAL_RANK=str(r))
        procs.append(subprocess.Popen([sys.executable, str(script)], env=e, stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True))
    outs = [p.communicate(timeout=240) for p in procs]
    assert all(p.returncode == 0 for p in procs), outs
    line = json.loads(outs[0][0].strip().splitlines()[-1])
    assert line["world"] == 2 and line["ms"] == 15.0
    assert abs(line["value"] - 2 * 1.0 / 15e-3) < 1e-9


def test_reference_arm_non_zero_ranks_exit_without_work():
    env = dict(os.environ, RANK="1", LOCAL_RANK="1", WORLD_SIZE="2")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2"],
                       env=env, capture_output=True, text=True, timeout=120)
    assert r.returncode == 0 and r.stdout.strip() == ""


def test_work_ratio():
    sys.path.insert(0, ROOT)
    import bench
    assert abs(bench.work_ratio(512, 256) - 9.0) < 1e-12
    assert bench.aggregate(20.0, 1.0, 1) == 50.0
