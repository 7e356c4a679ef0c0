"""bench.py's contract on a small problem (N = 16 384): the ONE JSON line carries every key the measurement
section of the task names, the timed steps ran this library's kernels, and the numbers are self-consistent."""
import json
import os
import subprocess
import sys

import pytest

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_bench_line_has_the_contract_keys():
    p = subprocess.run([sys.executable, "bench.py", "--particles", "16384", "--steps", "2", "--warmup", "3"],
                       cwd=ROOT, capture_output=True, text=True, timeout=900)
    assert p.returncode == 0, p.stderr[-2000:]
    lines = [l for l in p.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    for k in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
              "vs_baseline", "dtype", "data", "config", "roofline", "cpu_baseline", "e2e", "clocks", "gpu_launches"):
        assert k in d, k
    assert d["n_gpus"] == 1 and d["steps"] == 2 and d["warmup"] == 3 and d["dtype"] == "f64" and d["vs_baseline"] is None
    assert "workload" in d["config"] and d["scaling"] == "weak" and d["higher_is_better"] is True
    n = 16384.0
    assert abs(d["value"] - 2 * n * n / (2 * d["ms_per_step"] * 1e-3)) <= 1e-6 * d["value"]     # pairs / device time
    r = d["roofline"]
    assert r["bound"] == "alu" and r["unit"] == "TFLOP/s" and 0.3 < r["frac"] < 0.81 and abs(r["frac"] - r["achieved"] / r["peak"]) < 1e-12
    c = d["cpu_baseline"]
    assert c["kind"] == "oracle" and c["cores"] >= 1 and c["value"] > 0 and c["unit"] == d["unit"]
    e = d["e2e"]
    assert e["h2d_bytes_per_step"] == 16384 * 21 * 8 == e["d2h_bytes_per_step"] and 0 < e["value"] <= d["value"] * 1.001
    assert d["gpu_launches"] >= 2 * 5                         # at least next-block, predict, force, correct per step
    # the clocks sampler ticks every 200 ms: a timed region this short may end before its first sample
    assert "sm_mhz" in d["clocks"] and isinstance(d["clocks"]["reasons"], list)
    assert d["clocks"]["sm_mhz"] is None or d["clocks"]["sm_mhz"] > 0
    b = d["block_step_wall_time"]
    assert len(b) == 2 and all(x["block_steps"] > 100 and x["us_per_block_step"] > 0 and abs(x["dE_over_E"]) < 1e-8 for x in b)
