"""Run W warm-up steps, then ONE step between cudaProfilerStart / cudaProfilerStop.

    ncu --profile-from-start off --set full ... python -m paper_2105_01677_b200.profile_step \
        --config 5 --sweep-index 3 --route ppe [--warmup 3] [--steps 1] [--ppe-operator 1] [--key-mode 0] [--row-skin S]

so that an Nsight Compute capture holds exactly the kernels of the profiled step(s).  --warmup 0 profiles the
first step, the one that bins (with the default skin the later steps of a scene at rest skip their bins).  Run
it with MPS_B200_COND=0: Nsight Compute cannot see kernels of a graph that holds conditional nodes.  Measurement
tooling: argument marshalling only, every kernel is the library's.
"""
from __future__ import annotations

import argparse
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--config", type=int, default=5)
    ap.add_argument("--sweep-index", type=int, default=3)
    ap.add_argument("--route", default="ppe", choices=["explicit", "ppe"])
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--steps", type=int, default=1)
    ap.add_argument("--ppe-operator", type=int, default=None)
    ap.add_argument("--key-mode", type=int, default=None)
    ap.add_argument("--row-skin", type=float, default=None)
    ap.add_argument("--param", action="append", default=[], help="KEY=VALUE: any other scene parameter (e.g. ppe_source=2)")
    a = ap.parse_args()
    import torch
    import __graft_entry__ as ge
    ge.build()
    from paper_2105_01677_b200 import binding as B, scenes
    s = scenes.make_scene(a.config, sweep_index=a.sweep_index)
    if a.ppe_operator is not None:
        s.params["ppe_operator"] = a.ppe_operator
    if a.key_mode is not None:
        s.params["key_mode"] = a.key_mode
    if a.row_skin is not None:
        s.params["row_skin"] = a.row_skin
    for kv in a.param:
        k, v = kv.split("=", 1)
        s.params[k] = type(s.params[k])(float(v)) if k in s.params and not isinstance(s.params[k], tuple) else float(v)
    route = 1 if a.route == "ppe" else 0
    g = B.Mps(s)
    g.step(a.warmup, route)
    torch.cuda.synchronize()
    torch.cuda.cudart().cudaProfilerStart()
    g.step(a.steps, route)
    torch.cuda.synchronize()
    torch.cuda.cudart().cudaProfilerStop()
    st = g.stats()
    print(f"profiled {a.steps} step(s) of scene {a.config}[{a.sweep_index}] N={s.n} route={a.route}: "
          f"cg iters last solve {st['cg_iters']}, rows {st['n_rows']}, nnz {st['cg_nnz']}")
    g.close()


if __name__ == "__main__":
    main()
