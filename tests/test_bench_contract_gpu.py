"""bench.py prints ONE JSON line with the contract's keys (small n so that it runs in seconds)."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
pytestmark = pytest.mark.gpu


def test_bench_line_has_the_contract_keys():
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--n", "22", "--steps", "5", "--warmup", "3",
                        "--batched", "10:12", "--sweep", "24", "--sweep-fused", "22:2,22:6"], capture_output=True, text=True, timeout=900)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [ln for ln in r.stdout.splitlines() if ln.strip()]
    assert len(lines) == 1
    d = json.loads(lines[0])
    for key in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
                "vs_baseline", "dtype", "data", "config", "roofline", "e2e", "cpu_baseline", "gpu_launches", "clocks"):
        assert key in d, key
    assert d["metric"] == "dft_equiv_gflops" and d["unit"] == "GFLOP/s" and d["dtype"] == "f32"
    assert d["n_gpus"] == 1 and d["steps"] == 5 and d["warmup"] == 3 and d["higher_is_better"] is True
    assert d["vs_baseline"] is None and d["data"] == "synthetic" and "workload" in d["config"]
    assert d["value"] > 0 and abs(d["value"] - 5.0 * (1 << 22) * 22 / (d["ms_per_step"] * 1e-3) / 1e9) < 1e-6 * d["value"]
    rf = d["roofline"]
    assert rf["bound"] == "hbm" and rf["unit"] == "GB/s" and rf["peak"] > 0
    assert abs(rf["frac"] - rf["achieved"] / rf["peak"]) < 1e-9
    e2e = d["e2e"]
    assert e2e["h2d_bytes_per_step"] == 8 << 22 and e2e["d2h_bytes_per_step"] == 8 << 22 and e2e["value"] > 0
    assert e2e["value"] < d["value"]  # the copies are inside the timed region
    cb = d["cpu_baseline"]
    assert cb["kind"] == "oracle" and cb["cores"] >= 1 and cb["value"] > 0 and cb["sample"]
    assert d["gpu_launches"] == 5 * d["config"]["passes"]
    assert d["batched"][0]["n"] == 10 and d["batched"][0]["log2_batch"] == 12
    sw = d["sweep"][0]
    assert sw["n"] == 24 and sw["passes"] >= sw["ideal_passes"] and 0 < sw["roofline_frac"] < 1.2
    fs = d["max_fused_sweep"]  # BASELINE config 3's dimension (max_fused_size)
    assert [(f["n"], f["max_fused_qubits"]) for f in fs] == [(22, 2), (22, 6)] and fs[0]["passes"] > fs[1]["passes"] >= 3
    assert all(0 < f["slowest_pass_frac"] <= f["roofline_frac"] * 1.5 and f["median_ms"] > 0 for f in fs)
    assert "seconds_n22" in cb and "seconds_n26" in cb and len(cb["trials_n26"]) == 3  # whole circuits, timed
    assert rf["traffic"] is None or rf["traffic_source"]
