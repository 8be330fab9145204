"""GPU test (-m gpu) of bench.py's launch contract: `python bench.py --gpus N` run plainly must become N
ranks by itself.  Only one GPU is available to the tests, so this drives the same re-exec path with N = 1
(`--torchrun`): bench.py replaces itself by `python -m torch.distributed.run --nproc-per-node 1 ... bench.py`, the rank
initialises NCCL, runs its id-range share and the 24-byte exchange, and prints the one JSON line."""
import json, os, subprocess, sys
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _run(extra, env=None):
    cmd = [sys.executable, os.path.join(ROOT, "bench.py"), "--steps", "2", "--warmup", "3", "--batch-log2", "22",
           "--no-configs", "--no-alg1", "--no-cpu-baseline"] + extra
    e = dict(os.environ); e.pop("WORLD_SIZE", None); e.pop("RANK", None); e.pop("LOCAL_RANK", None)
    e.update(env or {})
    return subprocess.run(cmd, capture_output=True, text=True, timeout=600, env=e, cwd=ROOT)


def _line(r):
    rows = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert r.returncode == 0 and len(rows) == 1, r.stderr[-2000:]
    return json.loads(rows[0])


def test_bench_reexecs_itself_under_torchrun():
    plain = _line(_run(["--gpus", "1"]))
    spawned = _line(_run(["--gpus", "1", "--torchrun"]))
    assert plain["launcher"].startswith("none") and spawned["launcher"] == "bench.py -> torch.distributed.run"
    assert spawned["n_gpus"] == 1 and len(spawned["rank_ms_per_step"]) == 1
    assert spawned["best"] == plain["best"]                       # same ids, same ordered minimum through the exchange
    assert spawned["gpu_launches"] == plain["gpu_launches"] > 0


def test_bench_refuses_a_world_size_that_contradicts_gpus():
    r = _run(["--gpus", "2"], env={"WORLD_SIZE": "1", "RANK": "0", "LOCAL_RANK": "0"})
    assert r.returncode != 0 and "must agree" in r.stderr
