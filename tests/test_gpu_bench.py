"""bench.py contract on the GPU box: one JSON line with the keys the driver reads, produced by the CUDA path."""
import json
import os
import subprocess
import sys

import pytest

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_bench_line_contract():
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--steps", "12", "--warmup", "3", "--config", "cfg2",
                        "--no-large"], capture_output=True, text=True, timeout=900, cwd=ROOT)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1, "bench.py must print exactly one JSON line"
    d = json.loads(lines[0])
    assert d["metric"] == "fp64_gflops_davidson_iteration" and d["unit"] == "GFLOP/s" and d["dtype"] == "f64"
    assert d["n_gpus"] == 1 and d["steps"] == 12 and d["warmup"] == 3 and d["higher_is_better"] is True
    assert d["data"] == "synthetic" and d["scaling"] == "weak" and d["vs_baseline"] is None
    assert d["value"] > 0 and d["ms_per_step"] > 0
    assert "cfg2" in d["config"]["workload"] and "flushed" in d["config"]["l2"]
    # 12 steps of >= 6 launches each, counted by the library
    assert d["gpu_launches"] >= 6 * 12
    rf = d["roofline"]
    assert rf["bound"] == "tensor" and rf["unit"] == "TFLOP/s"
    # the denominator is the DMMA issue rate: 148 SMs x 128 FLOP/clk x the SM clock (37.2 TFLOP/s at 1965 MHz); it may sit
    # below the figure for the maximum clock when the box runs power-capped, never above it
    per_mhz = 148 * 128 * 1e6 / 1e12
    assert 0.80 * per_mhz * d["clocks"]["sm_mhz"] <= rf["peak"] <= 1.03 * per_mhz * d["clocks"]["sm_max_mhz"]
    assert rf["vendor_dgemm_tflops"] is None or 5.0 < rf["vendor_dgemm_tflops"] < 60.0
    assert rf["frac"] == pytest.approx(rf["achieved"] / rf["peak"]) and 0.0 < rf["frac"] < 1.0
    e = d["e2e"]
    assert 0 < e["value"] < d["value"] and e["h2d_bytes_per_step"] == 8 * 35465 and e["d2h_bytes_per_step"] == 8 * 35465 + 24
    cb = d["cpu_baseline"]
    assert cb["kind"] == "oracle" and cb["value"] > 0 and cb["cores"] >= 1 and "cfg2" in cb["sample"]
    assert d["value"] > cb["value"]
    c = d["clocks"]
    assert c["sm_max_mhz"] >= c["sm_mhz"] > 0 and isinstance(c["reasons"], list)
    assert set(d["hpsi_curve"]) >= {"cfg2", "cfg4", "cfg5a", "heis4096"}
    b = d["block_davidson"]
    assert "error" not in b and b["solve"]["single"]["rc"] == 0 and b["solve"]["block_nb2"]["rc"] == 0
    assert abs(b["solve"]["single"]["lambda"] - b["solve"]["block_nb2"]["theta"][0]) <= 1e-8
