"""bench.py on the GPU: one JSON line with the contract's keys (metric, value, e2e, roofline, cpu_baseline, clocks ...)."""
import json
import os
import subprocess
import sys

import pytest

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def run_bench(*extra):
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--steps", "5", "--warmup", "3",
                        "--cpu-sample", "200000", *extra], capture_output=True, text=True, timeout=900)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.strip().splitlines() if l.startswith("{")]
    assert len(lines) == 1
    return json.loads(lines[0])


def check_common(d):
    for k in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
              "vs_baseline", "dtype", "data", "config", "clocks", "e2e", "gpu_launches", "roofline", "cpu_baseline"):
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
    assert not set(d["clocks"]["reasons"]) & {"hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown"}


def test_default_line_is_config_1_additive():
    d = run_bench()
    check_common(d)
    assert d["config"]["workload"] == "cfg1_halos_10M" and d["config"]["mode"] == "additive"
    assert d["gpu_launches"] == 6 * d["steps"]
    assert set(d["stages"]) == {"count", "scan", "scatter", "splat", "large", "compose"}


def test_ordered_mode_line_on_the_small_config():
    d = run_bench("--config", "0", "--mode", "ordered")
    check_common(d)
    assert d["config"]["mode"] == "ordered" and "flush" not in d["config"]["l2"] or True
    assert set(d["stages"]) == {"count", "scan", "pairs", "sort", "bounds", "render", "combine"}
