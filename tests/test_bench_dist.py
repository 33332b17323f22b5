"""Host logic of the N > 1 bench path (replicas only) on CPU:
two processes over gloo run bench.py's own setup / reduction helpers and the
per-rank scene recipe; the reference arm prints on rank 0 only."""
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import json, os, sys
sys.path.insert(0, {root!r})
import argparse
import torch
import bench
args = argparse.Namespace(config=1, sweep_index=0, route=None)
world, rank, local = bench.dist_setup(args)
assert world == 2 and rank == int(os.environ["RANK"])
dev = torch.device("cpu")
scene, route = bench.make_scene(args, rank)
# per-rank timing: max over ranks; particle count: sum over ranks
ms = bench.barrier_and_max(world, 10.0 + 5.0 * rank, dev)
n_all = bench.all_sum(world, scene.n, dev)
import numpy as np
out = dict(rank=rank, ms=ms, n_all=n_all, n=scene.n, route=route,
           x_sum=float(np.sum(scene.x)), name=bench.workload_name(argparse.Namespace(config=1, sweep_index=0), scene, route))
with open(os.path.join({out!r}, "rank%d.json" % rank), "w") as f:   # one file per rank: stdout lines can interleave
    json.dump(out, f)
torch.distributed.barrier()
torch.distributed.destroy_process_group()
"""


def _torchrun(script_args, port):
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
           "--master-addr", "127.0.0.1", "--master-port", str(port)] + script_args
    env = dict(os.environ, CUDA_VISIBLE_DEVICES="", OMP_NUM_THREADS="1")
    return subprocess.run(cmd, cwd=ROOT, env=env, capture_output=True, text=True, timeout=600)


def test_world2_gloo_replicas(tmp_path):
    w = tmp_path / "worker.py"
    w.write_text(WORKER.format(root=ROOT, out=str(tmp_path)))
    r = _torchrun([str(w)], 29731)
    assert r.returncode == 0, r.stderr[-2000:]
    res = [json.load(open(tmp_path / f"rank{k}.json")) for k in (0, 1)]
    assert sorted(x["rank"] for x in res) == [0, 1]
    a, b = sorted(res, key=lambda x: x["rank"])
    # max over ranks of the per-rank time, sum over ranks of the particle counts
    assert a["ms"] == b["ms"] == 15.0
    assert a["n_all"] == b["n_all"] == a["n"] + b["n"] == 2 * 19468
    # independent replicas: same geometry, different seeded jitter
    assert a["x_sum"] != b["x_sum"] and a["route"] == b["route"] == 0
    assert a["name"].startswith("scene1:config1_dam4k_explicit:N=19468")


def test_reference_arm_prints_on_rank0_only():
    r = _torchrun(["bench.py", "--impl", "reference", "--gpus", "2", "--config", "1",
                   "--steps", "1", "--warmup", "0"], 29733)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["gpu_launches"] == 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["cores"] == 1
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["value"] > 0
