"""bench.py contract pieces that need no GPU: the reference arm (the oracle on host cores) prints
one JSON line with the agreed keys; the GPU arm refuses to run without a CUDA device (no CPU
fallback); the algorithmic-bytes arithmetic matches SURVEY.md 8(d)."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def run_bench(*args, env=None):
    e = dict(os.environ)
    e.update(env or {})
    return subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), *args], capture_output=True, text=True,
                          cwd=ROOT, env=e, timeout=600)


def test_reference_arm_prints_the_contract_line():
    r = run_bench("--impl", "reference", "--steps", "2", "--warmup", "1", "--cpu-sample-elems", "8192")
    assert r.returncode == 0, r.stderr
    lines = [l for l in r.stdout.splitlines() if l.strip()]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["metric"] == "learner_params_updated_per_sec" and d["unit"] == "learner-params/s"
    assert d["higher_is_better"] is True and d["steps"] == 2 and d["warmup"] == 1 and d["vs_baseline"] is None
    assert d["config"]["workload"] == "swb2000" and d["config"]["S"] == 16 and d["config"]["G"] == 4
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["cores"] == 1 and d["cpu_baseline"]["value"] == d["value"]
    assert d["e2e"] == {"value": d["value"], "unit": d["unit"], "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}
    assert d["value"] > 0


def test_reference_arm_other_ranks_do_no_work():
    r = run_bench("--impl", "reference", "--gpus", "2", "--steps", "1", "--warmup", "1", env={"RANK": "1", "WORLD_SIZE": "2"})
    assert r.returncode == 0 and r.stdout.strip() == ""


def test_gpu_arm_fails_loudly_without_a_gpu():
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    r = run_bench("--steps", "1", "--warmup", "1")
    assert r.returncode != 0 and "no CPU fallback" in (r.stderr + r.stdout)


def test_algorithmic_bytes_match_survey():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.algorithmic_bytes(bench.workload("swb2000")) == 16 * 145_145_344 * 32 == 74_314_416_128
    assert bench.algorithmic_bytes(bench.workload("swb300")) == 16 * 94_797_312 * 32
    assert bench.algorithmic_bytes(bench.workload("swb2000_ragged_bf16")) == 8 * 145_145_344 * 32
    assert bench.algorithmic_bytes(bench.workload("tiny")) == 2 * 1_000_000 * 24
    cfg = bench.workload("swb2000"); cfg["emit"] = True
    assert bench.algorithmic_bytes(cfg) == 16 * 145_145_344 * 34
