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
              "roofline", "cpu_baseline", "routes", "cg"):
        assert k in d, k
    assert d["n_gpus"] == 1 and d["steps"] == 3 and d["warmup"] >= 3 and d["dtype"] == "f64"
    # the size north_star names: the 2M point of BASELINE configs[4], PPE route
    assert d["config"]["workload"].startswith("scene5[3]:") and "route=ppe" in d["config"]["workload"]
    n = 1994776
    assert abs(d["value"] - n * 3 / (d["ms_per_step"] * 3e-3)) <= 1e-6 * d["value"]
    assert 5 < d["ms_per_step"] < 200 and d["gpu_launches"] >= 3 * 8 and 0 <= d["bins_per_step"] <= 2
    r = d["roofline"]
    assert r["kernel"] == "cg_spmv" and r["bound"] == "hbm" and r["unit"] == "GB/s"
    assert 0.0 < r["frac"] < 1.0 and abs(r["frac"] - r["achieved"] / r["peak"]) < 1e-12
    # frac reproduces from the printed bytes and microseconds
    assert abs(r["achieved"] - r["algorithmic_bytes_per_use"] / (r["us_per_use"] * 1e-6) / 1e9) <= 1e-6 * r["achieved"]
    assert r["uses"] == round(d["cg_iters_per_step"] * 3)
    assert r["traffic"] is None or 0.5 * r["algorithmic_bytes_per_use"] < r["traffic"] < 2.0 * r["algorithmic_bytes_per_use"]
    c = d["cg"]
    assert c["nnz"] > 100 * c["rows"] and 100 < c["ps_per_row_per_iteration"] < 1000
    e = d["e2e"]
    assert 0 < e["value"] < d["value"] and e["h2d_bytes_per_step"] == n * 56 and e["d2h_bytes_per_step"] == n * 56
    cb = d["cpu_baseline"]
    assert cb["kind"] == "oracle" and cb["cores"] == 1 and 0 < cb["value"] < d["value"] and "scene5[0]" in cb["sample"]
    assert 40 < d["cg_iters_per_step"] < 90 and d["clocks"]["sm_mhz"]
    # the explicit route of the same scene rides in the same line
    x = d["routes"]["explicit"]
    assert x["value"] > d["value"] and x["roofline"]["kernel"] in ("viscosity", "bin_list")
    assert 0.0 < x["roofline"]["frac"] < 1.0
    if x["roofline"]["kernel"] == "viscosity":
        assert x["roofline"]["bound"].startswith("l1-gather") and 0.3 < x["roofline"]["l1_gather"]["frac"] < 1.2


def test_scene2_line_says_l2_resident_when_traffic_is_known():
    d = _run("--config", "2", "--no-cpu-baseline", "--no-e2e", "--no-other-route")
    assert d["config"]["workload"].startswith("scene2:") and "route=ppe" in d["config"]["workload"]
    r = d["roofline"]
    assert r["kernel"] == "cg_spmv"
    if r["traffic"] is not None:        # profiles/r02_traffic.json has this workload: 47 MB of matrix live in L2
        assert r["bound"].startswith("L2-resident")


def test_explicit_route_line():
    d = _run("--config", "1", "--no-cpu-baseline", "--no-e2e", "--no-other-route")
    assert "route=explicit" in d["config"]["workload"] and "cg" not in d
    assert d["roofline"]["kernel"] in ("bin_list", "bin_sort", "viscosity") and 0.0 < d["roofline"]["frac"] < 1.0
