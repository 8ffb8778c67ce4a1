"""bench.py prints ONE JSON line with the keys the driver reads (small event count; GPU)."""
import json
import os
import subprocess
import sys

import pytest

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _run(*extra):
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--steps", "3", "--warmup", "3", *extra],
                         capture_output=True, text=True, timeout=600)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [l for l in out.stdout.splitlines() if l.strip()]
    assert len(lines) == 1
    return json.loads(lines[0])


def test_default_workload_line():
    d = _run("--events", "262144")
    for k in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling", "vs_baseline",
              "dtype", "data", "config", "roofline", "cpu_baseline", "e2e", "gpu_launches", "clocks"):
        assert k in d, k
    assert d["n_gpus"] == 1 and d["steps"] == 3 and d["warmup"] == 3 and d["dtype"] == "f64" and d["data"] == "synthetic"
    assert d["higher_is_better"] is True and d["scaling"] == "weak" and d["vs_baseline"] is None
    assert d["value"] > 1e6 and d["gpu_launches"] == 12 and "workload" in d["config"] and "model" not in d["config"]
    r = d["roofline"]
    assert r["bound"] == "alu" and r["unit"] == "TFLOP/s" and abs(r["frac"] - r["achieved"] / r["peak"]) < 1e-12
    assert 0.05 < r["frac"] < 1.0 and r["peak_measured_dfma_chain"] > 20
    c = d["cpu_baseline"]
    assert c["kind"] == "oracle" and c["cores"] >= 1 and c["value"] > 0 and "sample" in c
    assert abs(c["events_per_s_per_core"] * c["cores"] / c["value"] - 1) < 1e-12
    e = d["e2e"]
    assert e["value"] > 0 and e["h2d_bytes_per_step"] > 0 and e["d2h_bytes_per_step"] > 0
    assert e["events_per_step"] == 262144          # the same events per step as the device-resident number
    v = d["vegas"]                                  # config 4 beside the headline: 5 iterations from a uniform grid
    assert len(v["events_per_s_per_iteration"]) == 5 and min(v["events_per_s_per_iteration"]) > 1e6
    assert v["integral_pb_combined"] > 0 and v["sigma_pb_combined"] > 0 and 0 < v["cut_pass_fraction_last"] <= 1
    assert set(d["clocks"]) >= {"sm_mhz", "sm_max_mhz", "reasons"}
    ch = d["channels"]                              # SURVEY 8(f) N1 / N2 beside the headline
    assert set(ch) == {"qqx_ttxgg", "qg_ttxqg", "gg_ttxggg"}
    assert ch["gg_ttxggg"]["diagrams"] == 1240 and ch["gg_ttxggg"]["colour_flows"] == 120 and ch["qqx_ttxgg"]["diagrams"] == 36
    assert all(c["events_per_s"] > 1e5 and 0.02 < c["frac_of_measured"] < 1.0 for c in ch.values())


def test_vegas_workload_line():
    d = _run("--workload", "config4", "--events", "262144", "--no-cpu-baseline")
    assert d["config"]["step"].startswith("vegas_iterate") and d["value"] > 1e6
    v = d["vegas"]
    assert v["integral"] > 0 and v["variance"] > 0 and 0 < v["n_pass"] <= 262144
