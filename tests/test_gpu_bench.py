"""bench.py keeps its contract: one JSON line with the keys the driver reads, a value that is
the units of the K timed steps over their device time, a roofline object for the pair-force
kernel and an end-to-end leg with the bytes it copied."""
import json
import os
import subprocess
import sys

import pytest

pytestmark = pytest.mark.gpu

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_bench_line_schema():
    cmd = [sys.executable, os.path.join(ROOT, "bench.py"), "--workload", "C2", "--steps", "20",
           "--warmup", "3", "--no-cpu-baseline", "--no-variants", "--snapshots", "--other-workloads"]
    r = subprocess.run(cmd, capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [ln for ln in r.stdout.strip().splitlines() if ln.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    for k in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step",
              "higher_is_better", "scaling", "vs_baseline", "dtype", "data", "config", "clocks",
              "e2e", "gpu_launches", "roofline"):
        assert k in d, k
    assert d["n_gpus"] == 1 and d["steps"] == 20 and d["warmup"] == 3
    assert d["unit"] == "particle-steps/s" and d["higher_is_better"] is True
    assert d["vs_baseline"] is None and d["dtype"] == "f32" and d["data"] == "synthetic"
    n = d["config"]["n_particles"]
    assert d["value"] == pytest.approx(n * 20 / (d["ms_per_step"] * 20 * 1e-3), rel=1e-9)
    assert d["gpu_launches"] == 20 * d["launches_per_step"] > 0
    rf = d["roofline"]
    assert rf["bound"] == "alu" and rf["unit"] == "TFLOP/s"
    assert rf["frac"] == pytest.approx(rf["achieved"] / rf["peak"], rel=1e-9)
    assert 0.0 < rf["frac"] < 1.0 and 0.0 < rf["share_of_step"] <= 1.0
    e = d["e2e"]
    assert e["h2d_bytes_per_step"] == 28 * n and e["d2h_bytes_per_step"] >= 28 * n
    assert 0.0 < e["value"] < d["value"]          # copies inside the timed region
    assert "workload" in d["config"] and "model" not in d["config"]
    assert d["config"]["force_path"] == "list" and d["list"]["fallback_steps_in_timed_region"] == 0
