"""bench.py --impl reference on the CPU (the oracle arm): one JSON line with the keys the driver reads.  Config 1 (one
32769-bin spectrum) keeps it to a second; the GPU arm's line is produced on the GPU box and archived under profiles/."""
import json
import subprocess
import sys
from pathlib import Path

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


def test_archived_gpu_bench_line_has_the_contract_keys():
    """The newest headline line measured on the B200 (profiles/) carries roofline, cpu_baseline, e2e, clocks and launch count."""
    files = sorted((ROOT / "profiles").glob("r*_bench_cfg3.json"))
    assert files, "no archived bench line"
    d = json.loads(files[-1].read_text())
    for key in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling", "dtype",
                "data", "config", "roofline", "cpu_baseline", "e2e", "clocks", "gpu_launches"):
        assert key in d, key
    r = d["roofline"]
    assert r["bound"] == "hbm" and abs(r["frac"] - r["achieved"] / r["peak"]) < 1e-9 and r["unit"] == "GB/s"
    assert r["algorithmic_bytes_per_bin"] == 8 and r["traffic"] and d["gpu_launches"] > 0
    assert d["e2e"]["h2d_bytes_per_step"] == d["config"]["input_bytes_per_gpu"] and d["e2e"]["d2h_bytes_per_step"] > 0
    assert not set(d["clocks"]["reasons"]) & {"hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown"}
