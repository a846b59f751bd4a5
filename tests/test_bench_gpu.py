"""bench.py on a real B200 (-m gpu): the GPU arm prints exactly one JSON line carrying the contract's
keys, on the small workload so that it finishes in seconds."""
import json
import os
import subprocess
import sys

import pytest

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def run(*args):
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), *args], capture_output=True, text=True, cwd=ROOT, timeout=900)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.strip()]
    assert len(lines) == 1, r.stdout[:2000]
    return json.loads(lines[0])


def test_gpu_arm_line_has_the_contract_keys():
    d = run("--workload", "tiny", "--steps", "4", "--warmup", "3", "--e2e-steps", "2", "--cpu-sample-elems", "65536",
            "--cpu-sample-steps", "2", "--cpu-repeats", "2")
    assert d["metric"] == "learner_params_updated_per_sec" and d["unit"] == "learner-params/s" and d["n_gpus"] == 1
    assert d["steps"] == 4 and d["warmup"] == 3 and d["higher_is_better"] is True and d["vs_baseline"] is None
    assert d["dtype"] == "f32" and d["data"] == "synthetic" and d["config"]["workload"] == "tiny"
    assert d["gpu_launches"] == 4                                          # one fused kernel per step
    assert d["value"] == pytest.approx(2 * 2 * 1_000_000 / (d["ms_per_step"] * 1e-3), rel=1e-9)
    r = d["roofline"]
    assert r["bound"] == "hbm" and r["unit"] == "GB/s" and r["frac"] == pytest.approx(r["achieved"] / r["peak"])
    assert r["algorithmic_bytes_per_launch"] == 2 * 1_000_000 * 24
    assert r["traffic"] is None and r["traffic_source"]                    # no ncu capture of this workload: never a guess
    assert r["reference_mix"]["read_gbs"] > 1000 and r["reference_mix"]["write_gbs"] > 1000
    e = d["e2e"]
    assert e["h2d_bytes_per_step"] == 2 * 2 * 1_000_000 * 4 and e["d2h_bytes_per_step"] > 0 and 0 < e["value"] < d["value"]
    c = d["cpu_baseline"]
    assert c["kind"] == "oracle" and c["cores"] == 1 and len(c["repeats"]) == 2 and c["value"] == max(c["repeats"])
    assert c["all_cores"]["cores"] == (os.cpu_count() or 1)
    assert set(d["clocks"]) >= {"sm_mhz", "sm_max_mhz", "reasons"}
    assert d["share_pair_weights"]["ms_per_step"] > 0


def test_emulated_partition_line():
    d = run("--workload", "tiny", "--emulate-ranks", "2", "--steps", "4", "--warmup", "2")
    assert d["config"]["partition"] == "superlearner (emulated)" and d["config"]["emulated_ranks"] == 2
    assert d["scaling"] == "strong" and d["gpu_launches"] >= 8 and d["value"] > 0
