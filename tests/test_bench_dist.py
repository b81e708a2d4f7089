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


AGREE = r"""
import os, sys, json
sys.path.insert(0, %r)
import bench
rank, world = bench.dist_init("gloo")
a = bench.dist_all_ok(True)                       # every rank fine
b = bench.dist_all_ok(rank != 1)                  # rank 1 failed its set-up: EVERY rank must learn it and skip
c = bench.dist_all_ok(rank == 1)                  # rank 0 failed
bench.dist_barrier()                              # nobody is left behind in a collective
print(json.dumps({"rank": rank, "a": a, "b": b, "c": c}))
""" % ROOT


def test_ranks_agree_to_skip_a_collective_path_when_one_failed_its_setup(tmp_path):
    """bench.slab_multi enters its all-to-all only if dist_all_ok says every rank has its plan and buffers."""
    script = tmp_path / "agree.py"
    script.write_text(AGREE)
    env = dict(os.environ, MASTER_ADDR="127.0.0.1", MASTER_PORT="29537", WORLD_SIZE="2")
    procs = []
    for r in range(2):
        e = dict(env, RANK=str(r), LOCAL_RANK=str(r))
        procs.append(subprocess.Popen([sys.executable, str(script)], env=e, stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True))
    outs = [p.communicate(timeout=240) for p in procs]
    assert all(p.returncode == 0 for p in procs), outs
    for r, (out, _) in enumerate(outs):
        got = json.loads(out.strip().splitlines()[-1])
        assert got == {"rank": r, "a": True, "b": False, "c": False}
    sys.path.insert(0, ROOT)
    import bench
    assert bench.dist_all_ok(True) is True and bench.dist_all_ok(False) is False      # no process group: own flag


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


def test_headline_line_survives_slab_rows_that_hang_or_fail(tmp_path):
    """bench.print_line_with_guarded_rows: the N > 1 slab rows are added to the one JSON line when they come back, and
    the line is printed without them (exit code 0, `slab_multi_failed` set) when they never do."""
    sys.path.insert(0, ROOT)
    import io
    from contextlib import redirect_stdout
    import bench
    buf = io.StringIO()
    with redirect_stdout(buf):
        bench.print_line_with_guarded_rows({"value": 1.0}, 0, lambda: {"ms_r2c": 2.0}, 30.0)
        bench.print_line_with_guarded_rows({"value": 1.0}, 1, lambda: {"ms_r2c": 2.0}, 30.0)      # rank 1 prints nothing
        bench.print_line_with_guarded_rows({"value": 1.0}, 0, lambda: {"failed": "RuntimeError: x"}, 30.0)
    lines = [json.loads(l) for l in buf.getvalue().strip().splitlines()]
    assert lines == [{"value": 1.0, "slab_multi_gpu": {"ms_r2c": 2.0}, "slab_multi_failed": None},
                     {"value": 1.0, "slab_multi_gpu": {"failed": "RuntimeError: x"}, "slab_multi_failed": "RuntimeError: x"}]
    hang = tmp_path / "hang.py"
    hang.write_text("import sys, time\nsys.path.insert(0, %r)\nimport bench\n"
                    "bench.print_line_with_guarded_rows({'value': 1.0}, 0, lambda: time.sleep(600), 1.0)\n" % ROOT)
    r = subprocess.run([sys.executable, str(hang)], capture_output=True, text=True, timeout=120)
    assert r.returncode == 0
    out = r.stdout.strip().splitlines()
    assert len(out) == 1
    got = json.loads(out[0])
    assert got["value"] == 1.0 and "no result after 1 s" in got["slab_multi_failed"]


def test_gpus_2_without_a_launcher_starts_two_ranks(tmp_path):
    """`bench.py --gpus 2 --impl reference` with NO rank variables in the environment: bench.py launches its two ranks
    itself (torch.distributed.run on 127.0.0.1); rank 0 runs the oracle arm and prints the one JSON line with n_gpus 2,
    rank 1 starts, sees it has no work in this arm and exits 0."""
    env = {k: v for k, v in os.environ.items()
           if k not in ("RANK", "LOCAL_RANK", "WORLD_SIZE", "MASTER_ADDR", "MASTER_PORT", "TORCHELASTIC_RUN_ID")}
    env["TORCHELASTIC_ERROR_FILE"] = str(tmp_path / "err.json")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--impl", "reference", "--N", "16",
                        "--steps", "1", "--warmup", "0"], env=env, capture_output=True, text=True, timeout=600)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.strip().splitlines() if l.startswith("{")]
    assert len(lines) == 1                                   # one line: rank 1 printed nothing
    got = json.loads(lines[0])
    assert got["impl"] == "reference" and got["n_gpus"] == 2 and got["value"] > 0
