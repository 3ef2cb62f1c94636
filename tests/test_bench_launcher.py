"""bench.py --gpus N must start N ranks itself when it is not already under torchrun (VERDICT round 1,
weak #9: it used to burn on one GPU and print n_gpus = 1).  CPU test of that path: the launcher, the
127.0.0.1 rendezvous, the barrier, the max-over-ranks reduction and the single JSON line, with the gloo
backend and a stub step (bench.py --stub) at world_size 2."""
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
BENCH = os.path.join(ROOT, "bench.py")


def _run(args, env=None):
    e = dict(os.environ)
    for k in ("WORLD_SIZE", "RANK", "LOCAL_RANK", "MASTER_ADDR", "MASTER_PORT"):
        e.pop(k, None)
    e.update(env or {})
    return subprocess.run([sys.executable, BENCH, *args], capture_output=True, text=True, env=e, timeout=300)


def test_gpus_2_launches_two_ranks_and_prints_one_line():
    p = _run(["--gpus", "2", "--steps", "3", "--warmup", "1", "--stub"])
    assert p.returncode == 0, p.stderr[-2000:]
    lines = [l for l in p.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1, p.stdout
    out = json.loads(lines[0])
    assert out["n_gpus"] == 2 and out["steps"] == 3 and out["stub"] is True
    # rank 1 sleeps 20 ms per step, rank 0 10 ms: the reported time is the slower rank's
    assert 19.0 <= out["ms_per_step"] <= 60.0, out
    assert abs(out["value"] - 2 * 1000 / (out["ms_per_step"] * 1e-3)) < 1e-6 * out["value"]


def test_single_rank_stub_and_mismatch_is_refused():
    p = _run(["--gpus", "1", "--steps", "2", "--warmup", "1", "--stub"])
    assert p.returncode == 0 and json.loads(p.stdout.strip().splitlines()[-1])["n_gpus"] == 1
    p = _run(["--gpus", "4", "--stub"], env={"WORLD_SIZE": "2", "RANK": "0"})
    assert p.returncode != 0 and "WORLD_SIZE=2" in (p.stderr + p.stdout)
