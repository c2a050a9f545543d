"""The bench.py contract on a GPU box: one JSON line with every key the driver reads, on the smallest config."""
import json
import os
import subprocess
import sys

import pytest

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_bench_prints_one_contract_line():
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--config", "1", "--steps", "3", "--warmup", "3",
                        "--cpu-seconds", "0.5"], capture_output=True, text=True, timeout=600)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    j = json.loads(lines[0])
    for key in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
                "vs_baseline", "dtype", "data", "config", "e2e", "gpu_launches", "roofline", "cpu_baseline", "clocks"):
        assert key in j, key
    assert j["n_gpus"] == 1 and j["steps"] == 3 and j["warmup"] >= 3 and j["higher_is_better"] is True
    assert j["scaling"] == "weak" and j["vs_baseline"] is None and j["data"] == "synthetic"
    assert j["value"] > 0 and j["ms_per_step"] > 0 and j["gpu_launches"] >= 3 * 5
    assert "workload" in j["config"] and "configs[0]" in j["config"]["workload"]
    e = j["e2e"]
    assert e["value"] > 0 and e["value"] <= j["value"] * 1.05 and e["h2d_bytes_per_step"] > 0 and e["d2h_bytes_per_step"] > 0
    rf = j["roofline"]
    assert rf["bound"] == "alu" and 0 < rf["frac"] < 1.2 and abs(rf["frac"] - rf["achieved"] / rf["peak"]) < 1e-12
    assert "traffic" in rf and rf["hbm"]["bound"] == "hbm" and rf["hbm"]["peak"] > 1000
    cb = j["cpu_baseline"]
    assert cb["kind"] == "oracle" and cb["cores"] >= 1 and cb["value"] > 0 and cb["unit"] == j["unit"]
    assert set(j["clocks"]) >= {"sm_mhz", "sm_max_mhz", "reasons"}
    mb = rf["microbench"]
    assert 15.0 <= mb["mufu_ex2_per_clk_per_sm"] <= 16.5 and rf["build_id"]


def test_microbench_measures_the_roofline_denominators():
    """nd_microbench (include/nd.h "Diagnostics"; "measure both ... before quoting any roofline fraction"): the
    exp pipe issues 16 MUFU.EX2 per clock per SM, so n_SM x 16 x clock bounds the sweep; the FP64 RED rates frame the flush."""
    import paper_2607_01591_b200 as nd
    r = nd.nd_microbench()
    assert 15.0 <= r["mufu_ex2_per_clk_per_sm"] <= 16.5, r
    assert r["n_sm"] >= 100 and 1000.0 <= r["sm_clock_mhz"] <= 2300.0
    per_s = r["n_sm"] * r["mufu_ex2_per_clk_per_sm"] * r["sm_clock_mhz"] * 1e6
    assert abs(r["mufu_ex2_per_s"] - per_s) <= 0.03 * per_s                       # CUDA events agree with clock64 x clock
    assert r["red_f64_l2_per_s"] > 1e11 and r["red_f64_hbm_per_s"] > 5e10
    assert r["red_f64_l2_per_s"] > r["red_f64_hbm_per_s"]                        # an L2-resident table takes the REDs faster
    small = nd.nd_microbench(workspace_bytes=80 << 20)                           # no room for the HBM-resident table
    assert small["red_f64_hbm_per_s"] == 0.0 and 15.0 <= small["mufu_ex2_per_clk_per_sm"] <= 16.5
