"""bench.py's N > 1 plumbing on CPU: `--gpus N` without a torchrun environment must itself start N ranks (one per GPU),
rank 0 alone prints ONE JSON line with n_gpus = N, and a WORLD_SIZE that disagrees with --gpus is refused.  The GPU work
is replaced by fixed numbers (`--control-plane-only`, gloo, 127.0.0.1): nothing is measured here."""
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def run_bench(argv, env_extra=None, drop=("RANK", "LOCAL_RANK", "WORLD_SIZE", "MASTER_ADDR", "MASTER_PORT")):
    env = {k: v for k, v in os.environ.items() if k not in drop}
    env.update(env_extra or {})
    return subprocess.run([sys.executable, os.path.join(ROOT, "bench.py")] + argv, capture_output=True, text=True, env=env, timeout=300)


def test_gpus_2_starts_two_ranks_and_prints_one_line():
    r = run_bench(["--gpus", "2", "--steps", "3", "--warmup", "1", "--control-plane-only"])
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1, r.stdout
    d = json.loads(lines[0])
    assert d["n_gpus"] == 2 and d["control_plane_only"] is True and d["value"] is None
    assert d["units_all_ranks"] == 2 * 3000.0 and d["max_seconds"] == 2.0      # sum of units, max of times (rank 1 is slower)
    assert d["replica_seeds"] == [1, 2]


def test_single_rank_needs_no_launcher():
    r = run_bench(["--gpus", "1", "--steps", "2", "--control-plane-only"])
    assert r.returncode == 0, r.stderr[-2000:]
    d = json.loads([l for l in r.stdout.splitlines() if l.startswith("{")][0])
    assert d["n_gpus"] == 1 and d["units_all_ranks"] == 2000.0


def test_world_size_mismatch_is_refused():
    r = run_bench(["--gpus", "4", "--control-plane-only"], env_extra={"WORLD_SIZE": "2", "RANK": "0", "LOCAL_RANK": "0"})
    assert r.returncode != 0 and "refusing" in (r.stderr + r.stdout)
