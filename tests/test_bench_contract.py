"""bench.py's contract that can be checked without a GPU: the reference arm (the oracle on the host cores) prints one JSON
line with the agreed keys; under torchrun only rank 0 prints; the CUDA arm refuses to run without a device (no fallback)."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _run(args, env=None):
    e = dict(os.environ)
    e.update(env or {})
    return subprocess.run([sys.executable, os.path.join(ROOT, "bench.py")] + args, capture_output=True, text=True, cwd=ROOT, env=e, timeout=600)


def test_reference_arm_prints_one_json_line_with_the_contract_keys():
    r = _run(["--impl", "reference", "--config", "1", "--steps", "2", "--warmup", "1"])
    assert r.returncode == 0, r.stderr
    lines = [l for l in r.stdout.splitlines() if l.strip()]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["metric"] == "pooled_kv_retrieve_gbps_128k" and d["unit"] == "GB/s"
    assert d["steps"] == 2 and d["warmup"] == 1 and d["n_gpus"] == 1 and d["higher_is_better"] is True and d["vs_baseline"] is None
    assert d["value"] > 0 and d["ms_per_step"] > 0 and d["dtype"] == "u8" and d["data"] == "synthetic"
    assert d["config"]["workload"].startswith("llama3.1-8b") and "sample" in d["config"]
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["cores"] >= 1 and d["cpu_baseline"]["value"] == d["value"]
    assert d["e2e"] == {"value": d["value"], "unit": "GB/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}


def test_reference_arm_other_ranks_exit_silently():
    r = _run(["--impl", "reference", "--config", "1", "--steps", "1", "--warmup", "0", "--gpus", "2"], env={"RANK": "1", "WORLD_SIZE": "2", "LOCAL_RANK": "1"})
    assert r.returncode == 0 and r.stdout.strip() == ""


def test_cuda_arm_refuses_to_run_without_a_gpu():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    r = _run(["--steps", "1", "--warmup", "0"])
    assert r.returncode != 0 and "no CPU fallback" in r.stderr and r.stdout.strip() == ""


def test_gpus_n_starts_n_ranks_by_itself():
    """`python bench.py --gpus 2` with no torchrun around it starts two ranks that find each other (--launch-only: they meet
    over gloo and rank 0 reports how many there were), and only rank 0 prints."""
    e = {k: v for k, v in os.environ.items() if k not in ("RANK", "LOCAL_RANK", "WORLD_SIZE", "MASTER_ADDR", "MASTER_PORT")}
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--launch-only"], capture_output=True, text=True, cwd=ROOT,
                       env=e, timeout=600)
    assert r.returncode == 0, r.stderr
    lines = [l for l in r.stdout.splitlines() if l.strip()]
    assert len(lines) == 1 and json.loads(lines[0]) == {"launched_ranks": 2, "n_gpus": 2}
    assert "started 2 ranks" in r.stderr


def test_gpus_n_refuses_when_fewer_gpus_are_visible():
    """The CUDA arm never runs fewer ranks than asked for: with fewer than N visible GPUs it exits non-zero and says so."""
    import torch
    n = (torch.cuda.device_count() if torch.cuda.is_available() else 0) + 1
    e = {k: v for k, v in os.environ.items() if k not in ("RANK", "LOCAL_RANK", "WORLD_SIZE", "MASTER_ADDR", "MASTER_PORT")}
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", str(max(n, 2)), "--steps", "1", "--warmup", "1"], capture_output=True,
                       text=True, cwd=ROOT, env=e, timeout=600)
    assert r.returncode != 0 and r.stdout.strip() == "" and "CUDA device(s) visible" in r.stderr


def test_a_launcher_that_started_another_world_size_is_refused():
    r = _run(["--gpus", "4", "--launch-only"], env={"RANK": "0", "WORLD_SIZE": "2", "LOCAL_RANK": "0"})
    assert r.returncode != 0 and "WORLD_SIZE=2" in r.stderr
