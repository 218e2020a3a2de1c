"""N > 1 path of bench.py on CPU: world_size 2 over gloo (the path runs as replicas; the only cross-rank step is the
max-over-ranks of the timings and the whole-job aggregate)."""
import json
import os
import subprocess
import sys


def test_two_ranks_gloo(tmp_path):
    out = tmp_path / "r.json"
    worker = os.path.join(os.path.dirname(os.path.abspath(__file__)), "_gloo_worker.py")
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr", "127.0.0.1",
           "--master-port", "29571", worker, str(out)]
    r = subprocess.run(cmd, capture_output=True, text=True, timeout=300)
    assert r.returncode == 0, r.stderr[-2000:]
    d = json.load(open(out))
    assert d["ms"] == 11.0 and d["e2e"] == 50.0                 # max over ranks
    assert abs(d["value"] - 1000 * 3 * 4 * 2 / 11.0e-3) < 1e-6  # units of both replicas / max time


def test_reference_arm_other_ranks_exit_without_work():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2")
    root = os.path.join(os.path.dirname(os.path.abspath(__file__)), "..")
    r = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--impl", "reference", "--steps", "1", "--warmup", "0"],
                       capture_output=True, text=True, env=env, timeout=120)
    assert r.returncode == 0 and r.stdout.strip() == ""
