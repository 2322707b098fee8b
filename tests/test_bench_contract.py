"""bench.py prints ONE JSON line with the keys the driver reads.  CPU: the reference arm (the oracle on the host cores).
GPU: our arm on a small workload (every leg: device-resident throughput, kernel timing, roofline, streamed end-to-end step)."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
BASE_KEYS = {"metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling", "vs_baseline",
             "dtype", "data", "config", "e2e", "gpu_launches"}


def run_bench(*args, timeout=600):
    res = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), *args], capture_output=True, text=True, timeout=timeout,
                         cwd=ROOT)
    assert res.returncode == 0, res.stderr[-2000:]
    lines = [l for l in res.stdout.splitlines() if l.strip()]
    assert len(lines) == 1, res.stdout[-2000:]
    return json.loads(lines[0])


def test_reference_arm_prints_the_contract_line():
    d = run_bench("--impl", "reference", "--steps", "1", "--warmup", "0")
    assert BASE_KEYS <= set(d) and d["impl"] == "reference"
    assert d["value"] > 0 and d["unit"] == "cell-updates/s" and d["higher_is_better"] is True
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["cores"] >= 1 and d["cpu_baseline"]["value"] == d["value"]
    assert d["e2e"] == {"value": d["value"], "unit": d["unit"], "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}
    assert d["gpu_launches"] == 0 and "workload" in d["config"]


@pytest.mark.gpu
def test_our_arm_prints_the_contract_line():
    d = run_bench("--workload", "C5-128", "--steps", "4", "--warmup", "3", "--no-cpu-baseline")
    assert BASE_KEYS | {"roofline", "kernels", "clocks", "hbm_roofline_frac_step", "kernel_timing"} <= set(d)
    n = 128 ** 3
    assert d["n_gpus"] == 1 and d["steps"] == 4 and d["warmup"] == 3 and d["config"]["grid"] == [128, 128, 128]
    assert d["value"] == pytest.approx(n * 4 / (d["ms_per_step"] * 4e-3), rel=1e-9)
    r = d["roofline"]
    assert r["bound"] == "hbm" and r["unit"] == "GB/s" and r["frac"] == pytest.approx(r["achieved"] / r["peak"])
    assert r["kernel"].startswith("stage_tma") and r["bytes_per_cell"] in (80.0, 120.0)
    k = d["kernels"]
    assert k["stage1"]["launches"] >= 1 and k["stage2"]["launches"] >= 1          # (sampled: every 4th step on small grids)
    assert k["stage1"]["avg_ms"] + k["stage2"]["avg_ms"] <= d["ms_per_step"] * 1.05
    assert d["gpu_launches"] >= 2 * 4
    e = d["e2e"]
    assert e["value"] > 0 and e["d2h_bytes_per_step"] == 40 * n and e["h2d_bytes_per_step"] >= 40 * n and "streamed" in e["mode"]
    assert e["value"] < d["value"]                                                # PCIe-bound
    assert set(d["clocks"]) >= {"sm_mhz", "sm_max_mhz", "reasons"}
    assert d["config"]["floor_hits"] == 0
