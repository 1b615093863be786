"""bench.py contract on CPU: the oracle arm (--impl reference) prints one JSON line with the agreed
keys, and under a 2-rank launch (gloo is not even needed: the path is "replicas only")
rank 0 alone prints it while rank 1 exits 0 without work."""
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
KEYS = {"impl", "metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better",
        "scaling", "vs_baseline", "dtype", "data", "config", "cpu_baseline", "e2e"}


def _run(cmd, env=None):
    e = dict(os.environ)
    e.update(env or {})
    return subprocess.run(cmd, cwd=ROOT, env=e, capture_output=True, text=True, timeout=600)


def test_reference_arm_single_process():
    res = _run([sys.executable, "bench.py", "--impl", "reference", "--config", "1", "--steps", "1", "--warmup", "0",
                "--cpu-sample", "400"])
    assert res.returncode == 0, res.stderr
    lines = [l for l in res.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert KEYS <= set(d) and d["impl"] == "reference" and d["higher_is_better"] is False
    assert d["cpu_baseline"]["kind"] == "oracle" and d["value"] > 0
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["vs_baseline"] is None


def test_reference_arm_two_ranks():
    res = _run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
                "--master-addr", "127.0.0.1", "--master-port", "29591", "bench.py", "--gpus", "2", "--impl",
                "reference", "--config", "1", "--steps", "1", "--warmup", "0", "--cpu-sample", "300"])
    assert res.returncode == 0, res.stderr[-2000:]
    lines = [l for l in res.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1 and json.loads(lines[0])["n_gpus"] == 2


def test_b200_arm_fails_loudly_without_a_gpu():
    import torch
    if torch.cuda.is_available():
        return
    res = _run([sys.executable, "bench.py", "--steps", "1", "--warmup", "0", "--config", "1"])
    assert res.returncode != 0 and "no CPU fallback" in (res.stderr + res.stdout)
