"""bench.py prints ONE JSON line with the keys the driver reads (run on the small cfg1 workload so it takes seconds)."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.mark.gpu
def test_bench_line_has_the_contract_keys():
    p = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--workload", "cfg1", "--steps", "3", "--warmup", "3"],
                       capture_output=True, text=True, timeout=600)
    assert p.returncode == 0, p.stderr[-2000:]
    lines = [ln for ln in p.stdout.splitlines() if ln.strip()]
    assert len(lines) == 1
    d = json.loads(lines[0])
    for k in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
              "vs_baseline", "dtype", "data", "config", "roofline", "cpu_baseline", "e2e", "gpu_launches", "clocks"):
        assert k in d, k
    assert d["n_gpus"] == 1 and d["steps"] == 3 and d["warmup"] == 3 and d["higher_is_better"] is True
    assert d["unit"] == "clusters/s" and d["dtype"] == "f32" and d["data"] == "synthetic" and d["vs_baseline"] is None
    assert d["value"] > 0 and abs(d["value"] - d["config"]["n_clusters_total"] / (d["ms_per_step"] * 1e-3)) < 1e-6 * d["value"]
    r = d["roofline"]
    for k in ("bound", "achieved", "peak", "unit", "frac", "traffic"):
        assert k in r, k
    assert r["bound"] == "hbm" and r["unit"] == "GB/s" and abs(r["frac"] - r["achieved"] / r["peak"]) < 1e-12
    c = d["cpu_baseline"]
    assert c["kind"] == "oracle" and c["cores"] >= 1 and c["value"] > 0 and c["unit"] == "clusters/s" and c["sample"]
    assert c["one_thread"]["cores"] == 1 and c["one_thread"]["value"] > 0            # (i) one thread, (ii) sector-parallel
    assert d["parity_before_timing"]["ok"] is True and d["parity_before_timing"]["sectors"]
    assert d["repeats"] >= 10 and d["ms_per_step_best"] <= d["ms_per_step_median"]
    e = d["e2e"]
    assert e["value"] > 0 and e["h2d_bytes_per_step"] == d["config"]["n_clusters_per_gpu"] * 10 and e["d2h_bytes_per_step"] > 0
    assert d["gpu_launches"] >= 20 * d["steps"]
    assert "reasons" in d["clocks"]
