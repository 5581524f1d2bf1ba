"""N > 1 host logic on CPU (gloo, world_size 2): max-over-ranks timing, whole-job value, and the reference arm
under torchrun (rank 0 alone prints its line, the other ranks exit 0 without work)."""
from __future__ import annotations

import json
import os
import socket
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def torchrun(args, env=None, timeout=300):
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr",
           "127.0.0.1", "--master-port", str(free_port())] + args
    e = dict(os.environ)
    e.update(env or {})
    return subprocess.run(cmd, cwd=ROOT, env=e, capture_output=True, text=True, timeout=timeout)


def test_max_over_ranks_and_whole_job_value_gloo(tmp_path):
    r = torchrun([os.path.join(ROOT, "tests", "dist_worker.py")], env={"DIST_OUT": str(tmp_path)})
    assert r.returncode == 0, r.stderr[-2000:]
    outs = [json.load(open(tmp_path / ("rank%d.json" % k))) for k in range(2)]
    for o in outs:
        assert o["world"] == 2
        assert o["ms"] == 15.0                                  # the slower rank decides
        assert abs(o["value"] - 2 * 1000.0 * 4 / 15e-3 / 1e9) < 1e-15   # both replicas' points over the max time


def test_reference_arm_under_torchrun_prints_one_line():
    r = torchrun([os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1", "--warmup", "0",
                  "--grid", "128"])
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [ln for ln in r.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["value"] > 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["e2e"]["h2d_bytes_per_step"] == 0
    assert d["config"]["grid"] == [128, 128] and d["steps_timed"] == 1


def test_gpus_flag_without_torchrun_relaunches_itself():
    """`python bench.py --gpus 2` outside torchrun must not silently time one process: it re-executes under
    torch.distributed.run (checked with the CPU-only reference arm)"""
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "2",
                        "--warmup", "1", "--n", "96"], cwd=ROOT, capture_output=True, text=True, timeout=300)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [ln for ln in r.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1 and json.loads(lines[0])["n_gpus"] == 2


def test_reference_arm_runs_the_cuda_arms_grid_and_caps_its_steps():
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--steps", "100000",
                        "--warmup", "3", "--n", "512", "--ref-seconds", "3"], cwd=ROOT, capture_output=True, text=True,
                       timeout=300)
    assert r.returncode == 0, r.stderr[-2000:]
    d = json.loads([ln for ln in r.stdout.splitlines() if ln.startswith("{")][0])
    assert d["config"]["grid"] == [512, 512] and d["steps"] == 100000 and 1 <= d["steps_timed"] < 100000
    assert d["wall_s"] < 30
