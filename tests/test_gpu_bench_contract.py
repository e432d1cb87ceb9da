"""bench.py on the GPU: one JSON line with the contract's keys (metric, value, e2e, roofline, cpu_baseline, clocks ...).
The default line (configs[3], 400M particles) is exercised by the driver; here the same code runs on the small configs."""
import json
import os
import subprocess
import sys

import pytest

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def run_bench(*extra):
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--steps", "200", "--warmup", "3",
                        "--cpu-sample", "200000", *extra], capture_output=True, text=True, timeout=900)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.strip().splitlines() if l.startswith("{")]
    assert len(lines) == 1
    return json.loads(lines[0])


def check_common(d):
    for k in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
              "vs_baseline", "dtype", "data", "config", "clocks", "e2e", "gpu_launches", "roofline", "cpu_baseline",
              "cpu_baseline_all_cores", "host_cores", "peaks"):
        assert k in d, k
    assert d["unit"] == "particles/s" and d["higher_is_better"] is True and d["scaling"] == "weak"
    assert d["vs_baseline"] is None and d["dtype"] == "f32" and d["data"] == "synthetic" and d["warmup"] >= 3
    assert abs(d["value"] - d["config"]["particles"] / (d["ms_per_step"] * 1e-3)) <= 1e-6 * d["value"]
    assert d["gpu_launches"] > 0
    e = d["e2e"]
    assert e["h2d_bytes_per_step"] == 24 * d["config"]["particles"] and e["d2h_bytes_per_step"] > 0
    assert 0 < e["value"] < d["value"]                      # copies are inside the timed region
    rf = d["roofline"]
    assert rf["bound"] in ("hbm", "alu") and 0 < rf["frac"] < 1.5 and abs(rf["frac"] - rf["achieved"] / rf["peak"]) < 1e-9
    c = d["cpu_baseline"]
    assert c["kind"] == "oracle" and c["cores"] == 1 and c["value"] > 0 and "sample" in c
    ca = d["cpu_baseline_all_cores"]
    assert ca["kind"] == "oracle" and ca["cores"] == d["host_cores"] >= 1 and ca["value"] > 0
    assert not set(d["clocks"]["reasons"]) & {"hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown"}
    assert d["clocks"]["samples"] >= 5
    # the measured ALU peaks are near the nominal 148 SM x 128 lanes x clock and 148 x 16 x clock
    assert 25.0 < d["peaks"]["fma_lane_Tops"] < 40.0 and 3.0 < d["peaks"]["mufu_ex2_Tops"] < 5.0


def test_config_1_additive_line():
    d = run_bench("--config", "1", "--no-per-config")
    check_common(d)
    assert d["config"]["workload"] == "cfg1_halos_10M" and d["config"]["mode"] == "additive"
    assert d["gpu_launches"] == 7 * d["steps"]      # count, scan, layout, scatter, splat, large, compose
    assert set(d["stages"]) == {"count", "scan", "scatter", "splat", "large", "compose"}
    assert "per_config" not in d


def test_ordered_mode_line_on_the_small_config():
    d = run_bench("--config", "0", "--mode", "ordered", "--no-per-config")
    check_common(d)
    assert d["config"]["mode"] == "ordered" and "256 MB written between frames" in d["config"]["l2"]
    assert set(d["stages"]) == {"count", "scan", "pairs", "sort", "bounds", "render", "combine"}


def test_default_workload_is_the_largest_single_gpu_config():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.DEFAULT_CONFIG == 3 and bench.tile_for(3) == 32
