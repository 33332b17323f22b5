#!/usr/bin/env python
"""bench.py -- throughput of the MPS time step (arXiv 2105.01677) on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C] [--route R]
    python bench.py --impl reference ...        # the CPU oracle, as it stands

One "step" is one pass of the whole hot path (SURVEY.md 8(a) rows S1-S11:
bin, viscosity, predictor, bin, density, pressure, gradient, corrector) over
all particles of one seeded synthetic dam-break scene.  Default workload:
BASELINE.json configs[1] (scene 2: 89,228 particles, semi-implicit PPE route).

Prints ONE JSON line (rank 0).  Keys beyond the base contract:
  roofline      dominant kernel: algorithmic bytes per launch / CUDA-event time
                per launch (a second, instrumented replay of the same steps)
  kernels       per kernel category: ms per step, launches per step
  cpu_baseline  the oracle timed on this box's host cores on a bounded sample
  e2e           the same metric through mps_upload_host / mps_step /
                mps_download_host with pinned HOST buffers, copies timed
N > 1 (torchrun): one replica of the workload per GPU (different seeds), no
data-path collective ("replicas only"), weak scaling.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "particle_steps_per_sec"
UNIT = "particle-steps/s"
L2_FLUSH_BYTES = 256 << 20  # > the 126 MB L2 of B200
ROUTE_NAME = {0: "explicit", 1: "ppe"}


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--config", type=int, default=2, help="scene 1..5 (SURVEY.md 8(d)); default 2 = BASELINE configs[1]; 6 = paper-shaped 2D dam break")
    ap.add_argument("--sweep-index", type=int, default=0, help="size index 0..4 of scene 5")
    ap.add_argument("--route", default=None, choices=[None, "explicit", "ppe"])
    ap.add_argument("--rebin-every", type=int, default=1,
                    help="K > 1: the paper's neighbour-list reuse (PAPER.md:433), NOT the BASELINE workload")
    ap.add_argument("--ppe-operator", type=int, default=None, choices=[0, 1],
                    help="0 matrix-free, 1 assembled once per solve (library default)")
    ap.add_argument("--warm-start", action="store_true", help="cg_warm_start = 1")
    ap.add_argument("--key-mode", type=int, default=None, choices=[0, 1], help="0 linear cell key, 1 Morton")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-replay", action="store_true", help="skip the instrumented per-kernel replay")
    return ap.parse_args()


def peaks():
    """Measured roofline denominators (driver-written), else the guide's fallback."""
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md: 6.65 TB/s)"


def workload_name(args, scene, route):
    tag = f"scene{args.config}"
    if args.config >= 5:
        tag += f"[{args.sweep_index}]"
    return f"{tag}:{scene.name}:N={scene.n}:fluid={scene.n_fluid}:route={ROUTE_NAME[route]}"


def make_scene(args, rank=0):
    from paper_2105_01677_b200 import scenes
    seed = scenes.BASE_SEED + args.config + (args.sweep_index if args.config >= 5 else 0) + 1000 * rank
    s = scenes.make_scene(args.config, seed=seed, sweep_index=args.sweep_index)
    route = s.route if args.route is None else {"explicit": 0, "ppe": 1}[args.route]
    if getattr(args, "ppe_operator", None) is not None:
        s.params["ppe_operator"] = int(args.ppe_operator)
    if getattr(args, "warm_start", False):
        s.params["cg_warm_start"] = 1
    if getattr(args, "key_mode", None) is not None:
        s.params["key_mode"] = int(args.key_mode)
    if getattr(args, "rebin_every", 1) > 1:
        s.params["rebin_every"] = int(args.rebin_every)
        s.name += f"_reuse{args.rebin_every}"
    return s, route


class ClockSampler(threading.Thread):
    """Samples nvidia-smi clocks and throttle reasons while the timed region runs."""

    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_id: str):
        super().__init__(daemon=True)
        self.gpu_id = gpu_id
        self.rows = []
        self.proc = None

    def run(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", self.gpu_id, f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                 "-lms", "20"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            for line in self.proc.stdout:
                self.rows.append([c.strip() for c in line.split(",")])
        except Exception:
            pass

    def stop(self):
        if self.proc is not None:
            try:
                self.proc.terminate()
                self.proc.wait(timeout=5)
            except Exception:
                pass
        self.join(timeout=5)
        sm, mx, reasons = [], 0.0, set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[0]))
                mx = max(mx, float(r[1]))
                for k, nm in enumerate(names):
                    if r[3 + k].lower().startswith("active"):
                        reasons.add(nm)
            except Exception:
                continue
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": mx or None,
                "reasons": sorted(reasons), "samples": len(sm)}


# --------------------------------------------------------------------------------
# Algorithmic bytes per launch of each kernel category (the
# per-unit figures are SURVEY.md 8(d)'s).  N = stored particles, R = PPE rows
# (bc == 0), kn / kl = mean neighbour count within re_n / re_lap, klr = the same
# over PPE rows only.  "launches" = launches of the category per step.
def algorithmic_bytes(cat, N, R, kn, kl, klr):
    if cat == "cg_spmv":      # per application: list + own (x,y,z) + r_i + bc + y_i
        return R * (4.0 * klr + 24 + 8 + 1 + 8)
    if cat == "cg_update":    # p, s, x, r read+write; w read (rows only)
        return R * 72.0
    if cat == "bin_list":     # positions + type in, counts + rows out (per bin)
        return N * (24 + 1 + 8 + 4.0 * kl)
    if cat == "bin_sort":     # keys (28 B) + histogram/scatter/reorder (116 B) (per bin)
        return N * 144.0
    if cat == "density":      # re_n prefix of the rows + position + n out
        return N * (4.0 * kn + 24 + 8)
    if cat == "viscosity":    # nu_eff pass (+ re_n prefix if Cs > 0 not counted) + re_lap rows
        return N * (4.0 * kl + 24 + 24 + 1 + 24)
    if cat == "gradient":     # p-hat pass + gradient pass, each over the re_n prefix
        return N * (2 * 4.0 * kn + 24 + 8 + 8 + 8 + 24)
    if cat == "predict" or cat == "correct":
        return N * 96.0
    if cat == "pressure_explicit":
        return N * 17.0
    if cat == "ppe_setup":
        return N * (8 + 1 + 1 + 8 * 5)
    return None


def dist_setup(args):
    import torch
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world > 1:
        import torch.distributed as dist
        backend = "nccl" if torch.cuda.is_available() else "gloo"
        if backend == "nccl":
            torch.cuda.set_device(local)
        dist.init_process_group(backend=backend)
    return world, rank, local


def barrier_and_max(world, value_ms, device):
    """Barrier, then the max over ranks of a per-rank duration."""
    if world == 1:
        return value_ms
    import torch
    import torch.distributed as dist
    t = torch.tensor([value_ms], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def all_sum(world, value, device):
    if world == 1:
        return value
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())


def timed_steps(torch, world, g, route, K, flush, stream):
    """K steps, each bracketed by CUDA events on the ctx's stream; L2 flushed
    (untimed) before each.  Returns per-rank total ms."""
    ev0 = [torch.cuda.Event(enable_timing=True) for _ in range(K)]
    ev1 = [torch.cuda.Event(enable_timing=True) for _ in range(K)]
    torch.cuda.synchronize()
    if world > 1:
        torch.distributed.barrier()
    torch.cuda.synchronize()
    for k in range(K):
        flush.zero_()
        ev0[k].record(stream)
        g.step(1, route)
        ev1[k].record(stream)
    torch.cuda.synchronize()
    if world > 1:
        torch.distributed.barrier()
    torch.cuda.synchronize()
    return sum(a.elapsed_time(b) for a, b in zip(ev0, ev1))


def cpu_baseline(scene, route, budget_s=12.0, max_steps=5):
    """The oracle as it stands (single thread) on whole steps of the same scene,
    until about budget_s of CPU time has been spent."""
    from oracle import mps_oracle as O
    o = O.Oracle(scene)
    t0 = time.perf_counter()
    steps = 0
    while steps < max_steps:
        o.step(1, route)
        steps += 1
        if time.perf_counter() - t0 >= budget_s:
            break
    dt = time.perf_counter() - t0
    return {"value": scene.n * steps / dt, "unit": UNIT, "cores": 1, "kind": "oracle",
            "sample": f"{steps} whole step(s) of the same scene and route from t=0 "
                      f"({dt:.1f} s, single thread, cg iters last step {o.stats()['cg_iters']})",
            "host_cores_present": os.cpu_count()}


def run_b200(args):
    import numpy as np
    import torch
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the B200 path has no CPU fallback")
    world, rank, local = dist_setup(args)
    dev = torch.device("cuda", local if world > 1 else 0)
    torch.cuda.set_device(dev)
    import __graft_entry__ as ge
    if rank == 0:
        ge.build()
    if world > 1:
        torch.distributed.barrier()
    from paper_2105_01677_b200 import binding as B

    scene, route = make_scene(args, rank)
    K, W = args.steps, max(args.warmup, 3)
    stream = torch.cuda.current_stream(dev)
    flush = torch.empty(L2_FLUSH_BYTES, dtype=torch.uint8, device=dev)
    try:
        gpu_id = "GPU-" + str(torch.cuda.get_device_properties(dev).uuid)
    except Exception:
        gpu_id = str(dev.index)

    # ---- device-resident arm: the headline value -------------------------------------
    g = B.Mps(scene, device=str(dev))
    # the sampler runs over warm-up and timed steps: the timed region alone (tens of ms) is
    # shorter than nvidia-smi's start-up, and both are the same load
    sampler = ClockSampler(gpu_id)
    sampler.start()
    g.step(max(W, 3), route)
    t_end = time.perf_counter() + 0.5
    while time.perf_counter() < t_end and len(sampler.rows) < 3:
        g.step(1, route)               # untimed: keep the GPU under load until the sampler reports
    l0 = g.launch_count()
    st0 = g.stats()
    cg_before, loop_before = st0["cg_iters_total"], st0["cg_loop_ms_total"]
    ms_rank = timed_steps(torch, world, g, route, K, flush, stream)
    launches = g.launch_count() - l0
    clocks = sampler.stop()
    ms_total = barrier_and_max(world, ms_rank, dev)
    stats = g.stats()
    cg_timed_main = stats["cg_iters_total"] - cg_before
    cg_loop_ms = stats["cg_loop_ms_total"] - loop_before   # device-timed (%globaltimer) CG loops of the timed steps
    n_all = all_sum(world, scene.n, dev)
    value = n_all * K / (ms_total * 1e-3)

    # neighbour statistics of the last state, for the algorithmic-byte model
    bc = g.get("bc") if route == 1 else None
    g.bin()
    cl = g.neighbour_counts(B.RADIUS_LAP).astype(np.float64)
    cn = g.neighbour_counts(B.RADIUS_N).astype(np.float64)
    kl, kn = float(cl.mean()), float(cn.mean())
    rows = int((bc == 0).sum()) if bc is not None else 0
    klr = float(cl[bc == 0].mean()) if rows else 0.0
    # candidates the row builder must test (27 cells around every particle), for its ALU roofline
    nx_, ny_, nz_, ncell = g.grid()
    cs = g.cell_start().astype(np.int64)
    cnt = np.diff(cs[:ncell + 1]).reshape(nz_, ny_, nx_)
    R_ = int(np.ceil(scene.params["re_lap"] / (max(scene.params["re_n"], scene.params["re_lap"]) / scene.params["cell_div"]) - 1e-12))
    pad = np.pad(cnt, R_)
    cand = np.zeros_like(cnt)
    for dz in range(2 * R_ + 1):
        for dy in range(2 * R_ + 1):
            for dx in range(2 * R_ + 1):
                cand += pad[dz:dz + nz_, dy:dy + ny_, dx:dx + nx_]
    key_now = g.get("key"); typ_now = g.get("type")
    live = key_now < ncell
    fl_cnt = np.bincount(key_now[live & (typ_now == 0)], minlength=ncell).reshape(nz_, ny_, nx_)
    tests_all = float((cnt * cand).sum())       # a bin that builds every row
    tests_fluid = float((fl_cnt * cand).sum())  # the first bin of a step (fluid rows only)
    g.close()

    # ---- instrumented replay of the same steps: per-kernel CUDA-event times ------------
    kernels, roof = {}, None
    if not args.no_replay:
        g = B.Mps(scene, device=str(dev))
        g.step(W, route)
        cg_before_replay = g.stats()["cg_iters_total"]
        g.timers_enable((1 << len(B.TIMERS)) - 1)
        ms_replay = timed_steps(torch, 1, g, route, K, flush, stream)
        tm = g.timers_read()
        g.timers_enable(0)
        st_r = g.stats()
        g.close()
        # full operator applications / vector updates actually performed (launches issued after
        # convergence return at once; their time stays in the category's total)
        cg_iters_timed = st_r["cg_iters_total"] - cg_before_replay
        cg_uses = {"cg_spmv": cg_iters_timed + K, "cg_update": cg_iters_timed}
        peak, peak_src = peaks()
        n_bins = tm["bin_list"][1]          # one row-builder launch per bin (2 per step; fewer with list reuse)
        for cat, (ms, ln) in tm.items():
            if ln == 0:
                continue
            ab = algorithmic_bytes(cat, scene.n, rows, kn, kl, klr)
            # categories with several kernels per use: bytes are per use, not per launch
            uses = {"bin_sort": n_bins, "bin_list": n_bins, "viscosity": K, "gradient": K,
                    "ppe_setup": K, **cg_uses}.get(cat, ln)
            kernels[cat] = {"ms_per_step": ms / K, "launches_per_step": ln / K,
                            "us_per_launch": 1e3 * ms / ln,
                            "algorithmic_gbs": (ab * uses / (ms * 1e-3) / 1e9) if (ab and ms > 0) else None}
        top = max(kernels, key=lambda c: kernels[c]["ms_per_step"])
        ab = algorithmic_bytes(top, scene.n, rows, kn, kl, klr)
        ms, ln = tm[top]
        uses = {"bin_sort": n_bins, "bin_list": n_bins, "viscosity": K, "gradient": K, "ppe_setup": K,
                **cg_uses}.get(top, ln)
        achieved = ab * uses / (ms * 1e-3) / 1e9
        roof = {"kernel": top, "bound": "hbm", "per": "use (cg_spmv: one operator application; one k_ppe_cg launch runs a whole solve)",
                "achieved": achieved, "peak": peak, "unit": "GB/s",
                "frac": achieved / peak, "traffic": NCU_TRAFFIC.get((args.config, ROUTE_NAME[route], top)),
                "peak_source": peak_src, "algorithmic_bytes_per_use": ab, "uses": uses,
                "us_per_use": 1e3 * ms / max(uses, 1), "launches": ln,
                "share_of_step": (ms / K) / (ms_replay / K),
                "units": {"N": scene.n, "ppe_rows": rows, "mean_k_re_n": kn, "mean_k_re_lap": kl,
                          "mean_k_re_lap_rows": klr},
                "ms_per_step_instrumented": ms_replay / K}
        if top == "bin_list":
            # the row builder is bound by the fp64 pipe / instruction issue, not by HBM: report it
            # against the fp64 pipe (148 SMs x 64 lanes x 1.965 GHz; 10 fp64-pipe
            # instructions per candidate: 3 sub, 3 mul, 2 add, 2 compares)
            reuse = int(scene.params.get("rebin_every", 1))
            tests = n_bins * tests_all if reuse > 1 else K * (tests_all + tests_fluid)
            a_alu = tests * 10.0 / (ms * 1e-3) / 1e12
            roof.update({"bound": "alu", "hbm_achieved_gbs": roof["achieved"], "hbm_frac": roof["frac"],
                         "achieved": a_alu, "peak": 18.61, "unit": "T fp64-pipe instructions/s",
                         "frac": a_alu / 18.61, "peak_source": "148 SMs x 64 fp64 lanes x 1.965 GHz (measured 18.5 DADD/DMUL)",
                         "candidate_tests_per_step": tests / K})
        if top == "cg_spmv" and rows:
            # the two on-chip ceilings of a list-driven sweep (profiles/r01_ceilings_microbench.md):
            # 15 fp64 instructions per pair at 1.86e13/s, and the record gather at 30.8 SM-cycles
            # per 32 pairs (texture + LSU split) on 148 SMs at 1.965 GHz
            pairs = rows * klr
            t_use = 1e-3 * ms / max(uses, 1)
            roof["on_chip_ceilings"] = {
                "fp64_pipe_frac": pairs * 15.0 / 1.86e13 / t_use,
                "l1_gather_frac": pairs / 32.0 * 30.8 / (148 * 1.965e9) / t_use,
                "note": "fractions of the time of one operator application that the fp64 pipe and the "
                        "L1 record gather would need at their measured peaks; the gather binds"}

    # ---- end to end: pinned host buffers in, one step, host buffers out, every step ----
    e2e = None
    if not args.no_e2e:
        names = ("x", "y", "z", "u", "v", "w")
        host = {k: torch.from_numpy(np.ascontiguousarray(getattr(scene, k), np.float64)).pin_memory() for k in names}
        host["type"] = torch.from_numpy(np.ascontiguousarray(scene.type, np.int32)).pin_memory()
        host["phase"] = torch.from_numpy(np.ascontiguousarray(scene.phase, np.int32)).pin_memory()
        host["p"] = torch.zeros(scene.n, dtype=torch.float64).pin_memory()
        up = [host[k].data_ptr() for k in names + ("type", "phase")]
        down = [host[k].data_ptr() for k in names + ("p",)]
        g = B.Mps(scene, device=str(dev))

        def one():
            g.upload_host(up)
            g.step(1, route)
            g.download_host(down)

        for _ in range(W):
            one()
        e0 = [torch.cuda.Event(enable_timing=True) for _ in range(K)]
        e1 = [torch.cuda.Event(enable_timing=True) for _ in range(K)]
        torch.cuda.synchronize()
        if world > 1:
            torch.distributed.barrier()
        for k in range(K):
            flush.zero_()
            e0[k].record(stream)
            one()
            e1[k].record(stream)
        torch.cuda.synchronize()
        ms_e = barrier_and_max(world, sum(a.elapsed_time(b) for a, b in zip(e0, e1)), dev)
        g.close()
        e2e = {"value": n_all * K / (ms_e * 1e-3), "unit": UNIT,
               "h2d_bytes_per_step": int(scene.n * (6 * 8 + 2 * 4) * world),
               "d2h_bytes_per_step": int(scene.n * 7 * 8 * world),
               "ms_per_step": ms_e / K,
               "api": "mps_upload_host + mps_step(1) + mps_download_host on pinned host arrays"}

    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        cpu = cpu_baseline(scene, route)

    if rank == 0:
        out = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
            "ms_per_step": ms_total / K, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": workload_name(args, scene, route),
                       "baseline_config": (f"BASELINE.json configs[{args.config - 1}]" if args.config <= 5 else
                                           "none: the paper's own 2D dam-break shape (PAPER.md:397), context only"),
                       "parallelism": "single GPU" if world == 1 else f"{world} independent replicas (no collective)",
                       "l2": "flushed before every timed step (256 MiB write, untimed)",
                       "timing": "CUDA events on the ctx stream around each mps_step(1), summed; max over ranks"},
            "gpu_launches": int(launches), "clocks": clocks,
            "cg_iters_per_step": cg_timed_main / K,
            "fluid_particle_steps_per_sec": value * scene.n_fluid / scene.n,
            "roofline": roof, "kernels": kernels, "e2e": e2e, "cpu_baseline": cpu,
        }
        if route == 1:
            out["cg_iters_per_sec"] = cg_timed_main / (ms_total * 1e-3)
            out["cg"] = {"operator": {0: "matrix-free", 1: "assembled once per solve"}[int(scene.params.get("ppe_operator", 1))],
                         "rows": int(stats["n_rows"]), "loop_ms_per_step": cg_loop_ms / K,
                         "setup_ms_last_solve": stats["cg_setup_ms"],
                         "us_per_iteration": 1e3 * cg_loop_ms / max(cg_timed_main, 1),
                         "ps_per_row_per_iteration": 1e9 * cg_loop_ms / max(cg_timed_main, 1) / max(int(stats["n_rows"]), 1),
                         "timing": "%globaltimer of block 0 inside k_ppe_cg around the iteration loop"}
        print(json.dumps(out))
    if world > 1:
        torch.distributed.destroy_process_group()


# dram__bytes_read.sum + dram__bytes_write.sum per launch of the dominant kernel, copied by
# hand from the ncu --set full capture summarised under profiles/ (key: scene, route, category).
NCU_TRAFFIC = {
    # profiles/r01d_scene2_scene3_ppe.md: per operator application (whole-solve DRAM bytes / applications)
    (2, "ppe", "cg_spmv"): (20.16e6 + 0.38e6) / 53,
    (3, "ppe", "cg_spmv"): (9.293e9 + 1.011e9) / 62,
}


def run_reference(args):
    """The reference arm of this tier: the CPU oracle, as it stands, on host cores.

    Each timed "step" is one whole oracle step of a BOUNDED SAMPLE of the workload:
    the same tank, parameters and route at twice the particle spacing (1/8 of the
    fluid particles; for scene 2 this is scene 1's particle set), so that
    --steps 20 --warmup 3 ends within a few minutes (a full scene-2 PPE step takes
    the oracle about 15 s).  particle-steps/s is normalised by the particle count."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from oracle import build as orc_build
    orc_build.build()
    from oracle import mps_oracle as O
    from paper_2105_01677_b200 import scenes
    full, route = make_scene(args, 0)
    if args.config in (1,):
        sample, what = full, "the whole scene"
    else:
        l0 = 2.0 * full.params["l0"]
        geo = {2: ((40, 20, 30), (20, 20, 10)), 3: ((100, 25, 50), (50, 25, 25))}.get(args.config)
        if geo is None:
            geo = ((40, 20, 30), (20, 20, 10))
        sample = scenes.dam_break(l0, geo[0], geo[1], scenes.BASE_SEED + args.config, "reference_sample")
        for k in ("grad_variant", "n_phases", "rho", "nu", "cs", "rho_pair_mean", "nu_pair_mean"):
            sample.params[k] = full.params[k]
        what = (f"same tank and parameters at 2x spacing: N={sample.n} "
                f"(fluid {sample.n_fluid}) instead of N={full.n}")
    K, W = args.steps, args.warmup
    o = O.Oracle(sample)
    o.step(W, route)
    t0 = time.perf_counter()
    o.step(K, route)
    dt = time.perf_counter() - t0
    value = sample.n * K / dt
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": K, "warmup": W, "ms_per_step": 1e3 * dt / K, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": workload_name(args, full, route), "sample": what},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": what,
                         "host_cores_present": os.cpu_count()},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }))


def main():
    args = parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_b200(args)


if __name__ == "__main__":
    main()
