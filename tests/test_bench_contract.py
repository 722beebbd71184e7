"""bench.py --impl reference on the CPU (the oracle arm): one JSON line with the keys the driver reads.  Config 1 (one
32769-bin spectrum) keeps it to a second; the GPU arm's line is produced and checked by the gpu-marked test below."""
import json
import subprocess
import sys
from pathlib import Path

import pytest

ROOT = Path(__file__).resolve().parent.parent


def test_reference_arm_prints_one_json_line_with_the_contract_keys():
    res = subprocess.run([sys.executable, str(ROOT / "bench.py"), "--impl", "reference", "--config", "1", "--steps", "2",
                          "--warmup", "1"], capture_output=True, text=True, timeout=600, cwd=str(ROOT))
    assert res.returncode == 0, res.stderr[-2000:]
    lines = [l for l in res.stdout.splitlines() if l.strip()]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["metric"] == "fourier_bins_searched_per_sec_at_zmax" and d["unit"] == "bins/s"
    assert d["higher_is_better"] is True and d["steps"] == 2 and d["warmup"] == 1 and d["vs_baseline"] is None
    assert d["value"] > 0 and d["ms_per_step"] > 0 and d["dtype"] == "f64" and d["data"] == "synthetic"
    assert "cfg1" in d["config"]["workload"] and d["config"]["zmax"] == 32
    cb = d["cpu_baseline"]
    assert cb["kind"] == "oracle" and cb["cores"] >= 1 and cb["value"] == d["value"] and cb["sample"]
    assert d["e2e"] == {"value": d["value"], "unit": "bins/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}
    assert d["gpu_launches"] == 0


@pytest.mark.gpu
def test_gpu_arm_prints_one_json_line_with_the_contract_keys():
    """bench.py's own arm on the GPU, config 1 (one 32769-bin spectrum, seconds): the line it prints carries roofline,
    cpu_baseline, e2e, clocks and the launch count, and they are consistent with each other."""
    res = subprocess.run([sys.executable, str(ROOT / "bench.py"), "--config", "1", "--steps", "5", "--warmup", "3", "--e2e-steps", "1"],
                         capture_output=True, text=True, timeout=900, cwd=str(ROOT))
    assert res.returncode == 0, res.stderr[-2000:]
    lines = [l for l in res.stdout.splitlines() if l.strip()]
    assert len(lines) == 1
    d = json.loads(lines[0])
    for key in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling", "dtype",
                "data", "config", "roofline", "cpu_baseline", "e2e", "clocks", "gpu_launches"):
        assert key in d, key
    assert "impl" not in d and d["metric"] == "fourier_bins_searched_per_sec_at_zmax" and d["steps"] == 5 and d["n_gpus"] == 1
    assert abs(d["value"] - d["config"]["n_bins"] * d["config"]["batch_per_gpu"] / (d["ms_per_step"] * 1e-3)) <= 1e-6 * d["value"]
    r = d["roofline"]
    assert r["bound"] == "hbm" and abs(r["frac"] - r["achieved"] / r["peak"]) < 1e-9 and r["unit"] == "GB/s"
    assert r["algorithmic_bytes_per_bin"] == 8 and 0 < r["frac"] < 1 and 0 < r["path_frac"] <= r["frac"]
    assert sum(r["kernel_ms_all"].values()) <= d["ms_per_step"] * 1.02
    assert 0 < r["sweep_frac"] <= r["sweep_algorithmic_frac"]
    assert d["gpu_launches"] >= 3 * d["steps"]
    assert d["e2e"]["h2d_bytes_per_step"] == d["config"]["input_bytes_per_gpu"] and d["e2e"]["d2h_bytes_per_step"] >= 4
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["value"] > 0
    assert not set(d["clocks"]["reasons"]) & {"hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown"}
