"""bench.py prints ONE JSON line with the keys the driver reads (base contract + the roofline / cpu_baseline objects)."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.mark.gpu
def test_bench_prints_the_contract_line():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--steps", "2", "--warmup", "3", "--cpu-baseline-seconds", "1"],
                         capture_output=True, text=True, timeout=900, cwd=ROOT)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [l for l in out.stdout.splitlines() if l.strip()]
    assert len(lines) == 1, out.stdout[-2000:]
    d = json.loads(lines[0])
    for k in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling", "vs_baseline",
              "dtype", "data", "config", "clocks", "roofline", "e2e", "gpu_launches", "cpu_baseline"):
        assert k in d, k
    assert d["unit"] == "V-cycles/s" and d["n_gpus"] == 1 and d["steps"] == 2 and d["dtype"] == "f64" and d["data"] == "synthetic"
    assert d["higher_is_better"] is True and d["scaling"] == "weak" and d["vs_baseline"] is None and "workload" in d["config"]
    assert d["value"] > 500.0 and d["converged"] and d["gpu_launches"] > 100
    r = d["roofline"]
    for k in ("bound", "achieved", "peak", "unit", "frac", "traffic"):
        assert k in r, k
    assert r["bound"] == "hbm" and r["unit"] == "GB/s" and abs(r["frac"] - r["achieved"] / r["peak"]) < 1e-12 and 0.2 < r["frac"] < 1.0
    e = d["e2e"]
    assert e["unit"] == "V-cycles/s" and e["h2d_bytes_per_step"] == 257 * 257 * 8 and e["d2h_bytes_per_step"] == 5 * 257 ** 3 * 8
    assert 0.0 < e["blocking"]["value"] <= e["value"] * 1.05 and e["value"] <= d["value"] * 1.05
    c = d["cpu_baseline"]
    assert c["kind"] == "oracle" and c["unit"] == "V-cycles/s" and c["cores"] >= 1 and c["value"] > 0 and "sample" in c
    assert set(d["clocks"]) >= {"sm_mhz", "sm_max_mhz", "reasons"}
