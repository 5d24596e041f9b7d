"""bench.py's reference arm (the oracle on host cores) prints one JSON line with the contract's keys; runs on CPU."""
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_reference_arm_prints_the_contract_line():
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--cfg", "2", "--steps", "1",
                          "--warmup", "0", "--ref-freqs", "16"], capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert out.returncode == 0, out.stderr
    lines = [ln for ln in out.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    for key in ("impl", "metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
                "vs_baseline", "dtype", "data", "config", "cpu_baseline", "e2e"):
        assert key in d, key
    assert d["impl"] == "reference" and d["unit"] == "pairs/s" and d["higher_is_better"] is True and d["value"] > 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["cores"] >= 1 and d["cpu_baseline"]["value"] == d["value"]
    assert d["e2e"] == {"value": d["value"], "unit": d["unit"], "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}
    assert d["config"]["workload"].startswith("cfg2") and d["vs_baseline"] is None


def test_non_zero_ranks_of_the_reference_arm_exit_quietly():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2")
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2"], capture_output=True,
                         text=True, timeout=120, cwd=ROOT, env=env)
    assert out.returncode == 0 and out.stdout.strip() == ""


def test_our_arm_fails_loudly_without_cuda_or_without_its_ranks():
    """No CUDA device here: the product arm must refuse (no CPU fallback, no JSON line) -- at one rank, and as rank 0 of a
    two-rank launch (the x-slab leg); --gpus 2 outside torchrun is refused before anything runs."""
    import torch
    if torch.cuda.is_available():
        import pytest
        pytest.skip("a CUDA device is present")
    bench = os.path.join(ROOT, "bench.py")
    base = {k: v for k, v in os.environ.items() if k not in ("RANK", "WORLD_SIZE", "LOCAL_RANK")}
    for extra_env, argv in (({}, ["--steps", "1", "--warmup", "0"]),
                            ({"RANK": "0", "WORLD_SIZE": "2", "LOCAL_RANK": "0", "MASTER_ADDR": "127.0.0.1", "MASTER_PORT": "29999"},
                             ["--gpus", "2", "--steps", "1", "--warmup", "0"]),
                            ({}, ["--gpus", "2"])):
        out = subprocess.run([sys.executable, bench] + argv, capture_output=True, text=True, timeout=300, cwd=ROOT,
                             env=dict(base, **extra_env))
        assert out.returncode != 0, (argv, out.stdout)
        assert not [ln for ln in out.stdout.splitlines() if ln.startswith("{")], out.stdout
        assert "CUDA" in out.stderr or "one process per GPU" in out.stderr, out.stderr[-400:]
