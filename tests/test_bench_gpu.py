"""bench.py on a real GPU: the JSON line keeps its contract and its numbers are sane."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
pytestmark = pytest.mark.gpu


def _run(*extra):
    r = subprocess.run([sys.executable, "bench.py", "--steps", "3", "--warmup", "3", *extra], cwd=ROOT,
                       capture_output=True, text=True, timeout=900)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    return json.loads(lines[0])


def test_default_bench_line_contract():
    d = _run()
    for k in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better",
              "scaling", "vs_baseline", "dtype", "data", "config", "gpu_launches", "clocks", "e2e",
              "roofline", "cpu_baseline"):
        assert k in d, k
    assert d["n_gpus"] == 1 and d["steps"] == 3 and d["warmup"] >= 3 and d["dtype"] == "f64"
    assert d["config"]["workload"].startswith("scene2:") and "route=ppe" in d["config"]["workload"]
    n = 89228
    assert abs(d["value"] - n * 3 / (d["ms_per_step"] * 3e-3)) <= 1e-6 * d["value"]
    assert 0.2 < d["ms_per_step"] < 50 and d["gpu_launches"] >= 3 * 12
    r = d["roofline"]
    assert r["kernel"] == "cg_spmv" and r["bound"] == "hbm" and r["unit"] == "GB/s"
    assert 0.0 < r["frac"] < 1.0 and abs(r["frac"] - r["achieved"] / r["peak"]) < 1e-12
    # the instrumented replay times steps 4-6 of the run, the main arm may have warmed up longer
    assert abs(r["uses"] - (d["cg_iters_per_step"] * 3 + 3)) <= 0.1 * r["uses"] and r["traffic"] > 0
    assert 0.0 < r["on_chip_ceilings"]["l1_gather_frac"] < 1.2
    e = d["e2e"]
    assert 0 < e["value"] < d["value"] and e["h2d_bytes_per_step"] == n * 56 and e["d2h_bytes_per_step"] == n * 56
    c = d["cpu_baseline"]
    assert c["kind"] == "oracle" and c["cores"] == 1 and 0 < c["value"] < d["value"]
    assert 40 < d["cg_iters_per_step"] < 70 and d["clocks"]["sm_mhz"]


def test_explicit_route_line():
    d = _run("--config", "1", "--no-cpu-baseline", "--no-e2e")
    assert "route=explicit" in d["config"]["workload"] and d["cg_iters_per_step"] == 0
    assert d["roofline"]["kernel"] in ("bin_list", "bin_sort") and 0.0 < d["roofline"]["frac"] < 1.0
