"""bench.py --impl reference (the oracle as the reference arm) runs without a GPU: one JSON line with the contract's
keys, describing what it really timed; under torchrun only rank 0 works and prints."""
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _run(env_extra):
    env = dict(os.environ, **env_extra)
    return subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--steps", "1",
                           "--warmup", "0"], cwd=ROOT, env=env, capture_output=True, text=True, timeout=600)


def test_reference_arm_prints_one_contract_line():
    r = _run({"RANK": "0", "WORLD_SIZE": "1"})
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.strip()]
    assert len(lines) == 1
    line = json.loads(lines[0])
    assert line["impl"] == "reference" and line["higher_is_better"] is False and line["vs_baseline"] is None
    assert line["unit"] == "us/step/layer" and line["value"] > 0 and line["dtype"] == "f64"
    assert line["config"]["workload"] == "c2_llama31_8b_32k" and line["config"]["layers_per_step"] == 1
    assert line["steps"] == 1 and line["warmup"] == 0                 # what was timed, not what was asked for
    assert abs(line["ms_per_step"] * 1000.0 - line["value"]) < 1e-6 * line["value"]
    cb = line["cpu_baseline"]
    assert cb["kind"] == "oracle" and cb["cores"] == 1 and cb["value"] == line["value"] and cb["sample"]
    assert line["e2e"] == {"value": line["value"], "unit": line["unit"], "h2d_bytes_per_step": 0,
                           "d2h_bytes_per_step": 0}
    assert line["gpu_launches"] == 0


def test_reference_arm_other_ranks_exit_quietly():
    r = _run({"RANK": "1", "WORLD_SIZE": "2"})
    assert r.returncode == 0 and r.stdout.strip() == ""


def test_our_arm_fails_loudly_without_a_cuda_device():
    """No CPU fallback: on a box without a GPU the product arm stops with a clear message, it does not time anything."""
    import pytest
    import torch
    if torch.cuda.is_available():
        pytest.skip("this box has a GPU: the arm would run the real benchmark")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--steps", "1", "--warmup", "1"], cwd=ROOT,
                       capture_output=True, text=True, timeout=600)
    assert r.returncode != 0
    assert "needs a CUDA device" in r.stderr
    assert r.stdout.strip() == ""
