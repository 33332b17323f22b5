#!/usr/bin/env python
"""bench.py -- throughput of the MPS time step (arXiv 2105.01677) on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C] [--route R]
    python bench.py --impl reference ...        # the CPU oracle, as it stands

One "step" is one pass of the whole hot path (SURVEY.md 8(a) rows S1-S11:
bin, viscosity, predictor, bin, density, pressure, gradient, corrector) over
all particles of one seeded synthetic dam-break scene.  Default workload:
BASELINE.json configs[4] at its 2M point (scene 5[3]: 1,994,776 particles), semi-implicit
PPE route; the explicit route of the same scene is measured too and reported under
"routes".  --config 2 gives BASELINE configs[1] (89,228 particles).

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
    ap.add_argument("--steps", type=int, default=50, help="timed steps (BASELINE.json configs[4]: 50 steps each)")
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--config", type=int, default=5, help="scene 1..5 (SURVEY.md 8(d)); default 5 = BASELINE configs[4], the throughput sweep; 6 = paper-shaped 2D dam break")
    ap.add_argument("--sweep-index", type=int, default=3, help="size index 0..4 of scene 5 (default 3: N = 1,994,776)")
    ap.add_argument("--route", default=None, choices=[None, "explicit", "ppe"], help="default: ppe for scene 5, else the scene's own")
    ap.add_argument("--no-other-route", action="store_true", help="do not measure the other pressure route of the scene")
    ap.add_argument("--rebin-every", type=int, default=1,
                    help="K > 1: the paper's neighbour-list reuse (PAPER.md:433), NOT the BASELINE workload")
    ap.add_argument("--ppe-operator", type=int, default=None, choices=[0, 1],
                    help="0 matrix-free, 1 assembled once per solve (library default)")
    ap.add_argument("--warm-start", action="store_true", help="cg_warm_start = 1")
    ap.add_argument("--key-mode", type=int, default=None, choices=[0, 1], help="0 linear cell key, 1 Morton")
    ap.add_argument("--row-skin", type=float, default=None,
                    help="Verlet skin of mps_step's rows in units of l0 (library default 0.1; < 0: two bins per step)")
    ap.add_argument("--pre-steps", type=int, default=0,
                    help="untimed steps before the warm-up (0: the timed window starts W steps from rest, as BASELINE.json's "
                         "workloads do; e.g. 400 puts it in the developed dam-break flow)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-developed", action="store_true", help="skip the developed-flow leg (400 untimed steps, then K timed)")
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
    route = (1 if args.config == 5 else s.route) if args.route is None else {"explicit": 0, "ppe": 1}[args.route]
    if getattr(args, "ppe_operator", None) is not None:
        s.params["ppe_operator"] = int(args.ppe_operator)
    if getattr(args, "warm_start", False):
        s.params["cg_warm_start"] = 1
    if getattr(args, "key_mode", None) is not None:
        s.params["key_mode"] = int(args.key_mode)
    if getattr(args, "rebin_every", 1) > 1:
        s.params["rebin_every"] = int(args.rebin_every)
        s.name += f"_reuse{args.rebin_every}"
    if getattr(args, "row_skin", None) is not None:
        s.params["row_skin"] = float(args.row_skin)
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
    stream = g.stream                      # the ctx's own stream: flush, events and kernels in one queue
    for k in range(K):
        with torch.cuda.stream(stream):
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


def neighbour_statistics(np, B, g, scene, route):
    """Mean neighbour counts, PPE rows and the candidate tests of one row build (for the byte / ALU models)."""
    bc = g.get("bc") if route == 1 else None
    typ = g.get("type")
    g.bin()
    cl = g.neighbour_counts(B.RADIUS_LAP).astype(np.float64)
    cn = g.neighbour_counts(B.RADIUS_N).astype(np.float64)
    rows = int((bc == 0).sum()) if bc is not None else 0
    # candidates the row builder tests: the particles of the (2R+1)^3 cells around each particle's cell
    p = scene.params
    h = max(p["re_n"], p["re_lap"]) / p["cell_div"]
    nx_, ny_, nz_, _ = g.grid()
    R_ = int(np.ceil(p["re_lap"] / h - 1e-9))
    live = typ != 3
    cx = np.floor((g.get("x")[live] - p["domain_min"][0]) / h).astype(np.int64).clip(0, nx_ - 1)
    cy = np.floor((g.get("y")[live] - p["domain_min"][1]) / h).astype(np.int64).clip(0, ny_ - 1)
    cz = np.floor((g.get("z")[live] - p["domain_min"][2]) / h).astype(np.int64).clip(0, nz_ - 1)
    lin = cx + nx_ * (cy + ny_ * cz)
    cnt = np.bincount(lin, minlength=nx_ * ny_ * nz_).reshape(nz_, ny_, nx_)
    fl_cnt = np.bincount(lin[typ[live] == 0], minlength=nx_ * ny_ * nz_).reshape(nz_, ny_, nx_)
    pad = np.pad(cnt, R_)
    cand = np.zeros_like(cnt)
    for dz in range(2 * R_ + 1):
        for dy in range(2 * R_ + 1):
            for dx in range(2 * R_ + 1):
                cand += pad[dz:dz + nz_, dy:dy + ny_, dx:dx + nx_]
    fl, fw = typ == 0, (typ == 0) | (typ == 1)
    return {"kl": float(cl.mean()), "kn": float(cn.mean()), "rows": rows,
            "n_fluid": int(fl.sum()), "kl_fluid": float(cl[fl].mean()) if fl.any() else 0.0,
            "kn_fluid": float(cn[fl].mean()) if fl.any() else 0.0,
            "n_fw": int(fw.sum()), "kn_fw": float(cn[fw].mean()) if fw.any() else 0.0,
            "klr": float(cl[bc == 0].mean()) if rows else 0.0,
            "tests_all": float((cnt * cand).sum()), "tests_fluid": float((fl_cnt * cand).sum())}


def load_traffic():
    """dram bytes per use of the dominant kernels, written from the committed ncu captures by
    `python -m paper_2105_01677_b200.ncu_summary` (profiles/r02_traffic.json)."""
    try:
        with open(os.path.join(ROOT, "profiles", "r02_traffic.json")) as f:
            return json.load(f)
    except Exception:
        return {}


def pre_steps(g, route, n):
    """n untimed steps in calls of 16: the library looks at its row skin between mps_step calls."""
    while n > 0:
        g.step(min(n, 16), route)
        n -= 16


def measure_route(torch, np, B, args, scene, route, world, dev, stream, flush, K, W, sample_clocks):
    """One route of one scene: the device-resident timed steps, then an instrumented replay of the
    same steps with per-kernel CUDA events, and the roofline of the dominant kernel."""
    clocks = None
    if sample_clocks:
        try:
            gpu_id = "GPU-" + str(torch.cuda.get_device_properties(dev).uuid)
        except Exception:
            gpu_id = str(dev.index)
        # the sampler runs over warm-up and timed steps: the timed region alone can be shorter than
        # nvidia-smi's start-up, and both are the same load.  Until it reports, a scratch copy of the scene
        # keeps the GPU under the same load, so that the measured ctx always times steps W .. W+K from rest
        # (how often the skin rows are rebuilt depends on how far the flow has developed)
        sampler = ClockSampler(gpu_id)
        sampler.start()
        g0 = B.Mps(scene, device=str(dev))
        t_end = time.perf_counter() + 1.0
        while time.perf_counter() < t_end and len(sampler.rows) < 3:
            g0.step(1, route)
        g0.close()
    g = B.Mps(scene, device=str(dev))
    pre_steps(g, route, int(getattr(args, "pre_steps", 0)))
    g.step(max(W, 3), route)
    l0 = g.launch_count()
    st0 = g.stats()
    ms_rank = timed_steps(torch, world, g, route, K, flush, stream)
    launches = g.launch_count() - l0
    if sample_clocks:
        clocks = sampler.stop()
    ms_total = barrier_and_max(world, ms_rank, dev)
    stats = g.stats()
    cg_iters = stats["cg_iters_total"] - st0["cg_iters_total"]
    cg_loop_ms = stats["cg_loop_ms_total"] - st0["cg_loop_ms_total"]  # device-timed (%globaltimer) CG loops
    n_all = all_sum(world, scene.n, dev)
    value = n_all * K / (ms_total * 1e-3)
    ns = neighbour_statistics(np, B, g, scene, route)
    g.close()
    N, rows, kn, kl, klr = scene.n, ns["rows"], ns["kn"], ns["kl"], ns["klr"]
    asm = int(scene.params.get("ppe_operator", 1)) == 1
    out = {"value": value, "ms_per_step": ms_total / K, "gpu_launches": int(launches), "clocks": clocks,
           "bins_per_step": (stats["bins_total"] - st0["bins_total"]) / K,
           "fluid_particle_steps_per_sec": value * scene.n_fluid / scene.n,
           "units": {"N": N, "ppe_rows": rows, "mean_k_re_n": kn, "mean_k_re_lap": kl, "mean_k_re_lap_rows": klr}}
    cg = None
    if route == 1:
        nnz = int(stats["cg_nnz"]) if asm else None
        # bytes one CG iteration must move: the operator application plus the vector updates (the
        # device-timed loop covers both).  Assembled: one 8-byte word per stored pair (24-bit column +
        # 40-bit coefficient) + per row count, diagonal term, scale, r_g and w_g; matrix-free: 4 B per
        # listed pair + position, r_i, bc, w_i
        per_iter = (8.0 * nnz + rows * (4 + 8 + 8 + 8 + 8) if asm else rows * (4.0 * klr + 24 + 8 + 1 + 8)) + rows * 72.0
        cg = {"operator": "assembled once per solve (ppe_operator 1)" if asm else "matrix-free (ppe_operator 0)",
              "rows": rows, "nnz": nnz, "iters_per_step": cg_iters / K, "iters_per_sec": cg_iters / (ms_total * 1e-3),
              "loop_ms_per_step": cg_loop_ms / K, "setup_ms_last_solve": stats["cg_setup_ms"],
              "us_per_iteration": 1e3 * cg_loop_ms / max(cg_iters, 1),
              "ps_per_row_per_iteration": 1e9 * cg_loop_ms / max(cg_iters, 1) / max(rows, 1),
              "algorithmic_bytes_per_iteration": per_iter,
              "algorithmic_gbs": per_iter * cg_iters / (cg_loop_ms * 1e-3) / 1e9 if cg_loop_ms > 0 else None,
              "timing": "%globaltimer of block 0 inside k_ppe_cg around the iteration loop"}
        out["cg"] = cg
    if args.no_replay:
        out.update({"kernels": {}, "roofline": None})
        return out

    # ---- instrumented replay of the same steps: per-kernel CUDA-event times ------------------
    g = B.Mps(scene, device=str(dev))
    pre_steps(g, route, int(getattr(args, "pre_steps", 0)))
    g.step(W, route)
    bins0 = g.stats()["bins_total"]
    g.timers_enable((1 << len(B.TIMERS)) - 1)
    ms_replay = timed_steps(torch, 1, g, route, K, flush, stream)
    tm = g.timers_read()
    g.timers_enable(0)
    # bins that ran (with a skin the bin kernels are launched twice per step and return at once unless the
    # device flag is up: the launch count is not the bin count)
    n_bins = max(int(g.stats()["bins_total"] - bins0), 1)
    g.close()
    peak, peak_src = peaks()
    kernels = {}
    for cat, (ms, ln) in tm.items():
        if ln == 0:
            continue
        ab = algorithmic_bytes(cat, N, rows, kn, kl, klr)
        # categories with several kernels per use: bytes are per use, not per launch
        uses = {"bin_sort": n_bins, "bin_list": n_bins, "viscosity": K, "gradient": K, "ppe_setup": K}.get(cat, ln)
        kernels[cat] = {"ms_per_step": ms / K, "launches_per_step": ln / K, "us_per_launch": 1e3 * ms / ln,
                        "algorithmic_gbs": (ab * uses / (ms * 1e-3) / 1e9) if (ab and ms > 0 and cat != "cg_spmv") else None}
    top = max(kernels, key=lambda c: kernels[c]["ms_per_step"])
    ms_top, ln_top = tm[top]
    tag = f"scene{args.config}" + (f"[{args.sweep_index}]" if args.config >= 5 else "")
    traffic = load_traffic().get(f"{tag}:{ROUTE_NAME[route]}:{top}" + (":asm" if (top == "cg_spmv" and asm) else ""))
    roof = {"kernel": top, "share_of_step": (ms_top / K) / (ms_replay / K), "ms_per_step_instrumented": ms_replay / K,
            "peak_source": peak_src}
    if top == "cg_spmv" and cg:
        # one launch of k_ppe_cg is a whole solve; the unit of the roofline is one CG iteration
        # (operator application + vector updates), timed on the device inside the kernel
        ach = cg["algorithmic_gbs"]
        tr = traffic["dram_bytes_per_use"] if traffic else None
        l2_resident = tr is not None and tr < 0.5 * cg["algorithmic_bytes_per_iteration"]
        roof.update({"per": "CG iteration (operator application + vector updates) inside k_ppe_cg",
                     "achieved": ach, "peak": peak, "unit": "GB/s", "frac": ach / peak,
                     "traffic": tr, "traffic_source": traffic.get("source") if traffic else None,
                     "algorithmic_bytes_per_use": cg["algorithmic_bytes_per_iteration"], "uses": cg_iters,
                     "us_per_use": cg["us_per_iteration"], "launches": ln_top,
                     "bound": ("L2-resident: the iteration's data stay in the 126 MB L2, the HBM fraction is not a "
                               "roofline here; grid barriers and L2 latency bind") if l2_resident else
                              ("hbm" if asm else "l1-gather (one 32-byte record gather per pair; no unit saturated "
                                                 "in ncu, HBM fraction reported against the measured copy peak)")})
    elif top == "bin_list":
        # the row builder is bound by the fp64 pipe / instruction issue, not by HBM: report it against
        # the fp64 pipe (148 SMs x 64 lanes x 1.965 GHz; 10 fp64-pipe instructions
        # per candidate: 3 sub, 3 mul, 2 add, 2 compares)
        ab = algorithmic_bytes(top, N, rows, kn, kl, klr)
        reuse = int(scene.params.get("rebin_every", 1))
        # one full scan per step when mps_step carries its rows across the corrector, else a fluid-only
        # scan at r^k and a full one at r*
        tests = n_bins * ns["tests_all"] if (reuse > 1 or n_bins <= K) else K * (ns["tests_all"] + ns["tests_fluid"])
        a_alu = tests * 10.0 / (ms_top * 1e-3) / 1e12
        hbm = ab * n_bins / (ms_top * 1e-3) / 1e9
        roof.update({"per": "row build (one per bin)", "bound": "alu", "achieved": a_alu, "peak": 18.61,
                     "unit": "T fp64-pipe instructions/s", "frac": a_alu / 18.61,
                     "peak_source": "148 SMs x 64 fp64 lanes x 1.965 GHz (measured 18.5 T DADD/DMUL per s)",
                     "hbm_achieved_gbs": hbm, "hbm_frac": hbm / peak, "candidate_tests_per_step": tests / K,
                     "traffic": traffic["dram_bytes_per_use"] if traffic else None, "uses": n_bins,
                     "us_per_use": 1e3 * ms_top / max(n_bins, 1), "launches": ln_top})
    else:
        ab = algorithmic_bytes(top, N, rows, kn, kl, klr)
        uses = {"viscosity": K, "gradient": K, "ppe_setup": K}.get(top, ln_top)
        ach = ab * uses / (ms_top * 1e-3) / 1e9
        roof.update({"per": "use", "bound": "hbm", "achieved": ach, "peak": peak, "unit": "GB/s", "frac": ach / peak,
                     "traffic": traffic["dram_bytes_per_use"] if traffic else None, "uses": uses,
                     "us_per_use": 1e3 * ms_top / max(uses, 1), "launches": ln_top})
        # the list-driven sweeps gather one 32-byte record (sector) per pair and array from the L1: by measurement
        # (profiles/r01_ceilings_microbench.md: 31 SM-cycles per 32 records with the texture + LSU split) that, not
        # HBM, binds them.  Sectors counted from the exact sets (the skin's extra pairs are not credited).
        sectors = {"viscosity": ns["n_fluid"] * ns["kl_fluid"] * 2.0,                      # position + velocity record
                   "density": N * kn,
                   "gradient": ns["n_fw"] * ns["kn_fw"] + ns["n_fluid"] * ns["kn_fluid"]}.get(top)  # p-hat pass + sum
        if sectors:
            sm, ghz = 148, 1.965
            per_clk = sectors * uses / (ms_top * 1e-3) / (sm * ghz * 1e9)
            roof.update({"bound": "l1-gather (one 32-byte record per pair and array through the L1; the HBM fraction is "
                                  "reported against the measured copy peak but is not what binds)",
                         "l1_gather": {"achieved_sectors_per_sm_clk": per_clk, "ceiling": 32.0 / 31.0,
                                       "frac": per_clk / (32.0 / 31.0),
                                       "ceiling_source": "stand-alone gather of the same shape, texture + LSU split: 31 SM-cycles per 32 records"}})
    out.update({"kernels": kernels, "roofline": roof})
    return out


def sample_scene(args, full):
    """A bounded sample of the workload for the CPU oracle (it needs minutes per step at 1M+ particles):
    the same shape, parameters and route at a size one oracle step finishes in seconds."""
    from paper_2105_01677_b200 import scenes
    if full.n <= 120000:
        return full, "the whole scene"
    if args.config == 5:
        s = scenes.make_scene(5, seed=scenes.BASE_SEED + 5, sweep_index=0)
        what = f"scene5[0]: the same dam-break shape, parameters and route at N={s.n} (fluid {s.n_fluid}) instead of N={full.n}"
    else:
        l0 = 2.0 * full.params["l0"]
        geo = {3: ((100, 25, 50), (50, 25, 25))}.get(args.config, ((40, 20, 30), (20, 20, 10)))
        s = scenes.dam_break(l0, geo[0], geo[1], scenes.BASE_SEED + args.config, "reference_sample")
        what = f"same tank and parameters at 2x spacing: N={s.n} (fluid {s.n_fluid}) instead of N={full.n}"
    for k in ("grad_variant", "n_phases", "rho", "nu", "cs", "rho_pair_mean", "nu_pair_mean"):
        s.params[k] = full.params[k]
    return s, what


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

    main = measure_route(torch, np, B, args, scene, route, world, dev, stream, flush, K, W, sample_clocks=True)
    n_all = all_sum(world, scene.n, dev)

    # the other pressure route of the same scene, in the same line (single GPU only)
    other = None
    if world == 1 and not args.no_other_route and args.rebin_every == 1:
        r2 = 1 - route
        o = measure_route(torch, np, B, args, scene, r2, 1, dev, stream, flush, K, W, sample_clocks=False)
        other = {ROUTE_NAME[r2]: {k: o[k] for k in ("value", "ms_per_step", "bins_per_step", "gpu_launches", "roofline", "kernels")
                                  if k in o} | ({"cg": o["cg"]} if "cg" in o else {})}

    # the same scene once the flow has developed (the timed window of BASELINE.json's workloads starts from rest,
    # where particles move little and the skin rows last for many steps): 400 untimed steps first, no replay
    developed = None
    if world == 1 and not args.no_developed and args.pre_steps == 0 and args.rebin_every == 1:
        import copy
        a2 = copy.copy(args)
        a2.pre_steps, a2.no_replay = 400, True
        developed = {"pre_steps": 400}
        for r_ in ((route, 1 - route) if not args.no_other_route else (route,)):
            o = measure_route(torch, np, B, a2, scene, r_, 1, dev, stream, flush, K, W, sample_clocks=False)
            developed[ROUTE_NAME[r_]] = {k: o[k] for k in ("value", "ms_per_step", "bins_per_step", "gpu_launches")} | (
                {"cg_iters_per_step": o["cg"]["iters_per_step"], "ps_per_row_per_iteration": o["cg"]["ps_per_row_per_iteration"]}
                if "cg" in o else {})

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
            with torch.cuda.stream(g.stream):
                flush.zero_()
            e0[k].record(g.stream)
            one()
            e1[k].record(g.stream)
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
        smp, what = sample_scene(args, scene)
        cpu = cpu_baseline(smp, route)
        cpu["sample"] = what + "; " + cpu["sample"]

    if rank == 0:
        out = {
            "metric": METRIC, "value": main["value"], "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
            "ms_per_step": main["ms_per_step"], "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": workload_name(args, scene, route),
                       "baseline_config": (f"BASELINE.json configs[{args.config - 1}]" + (f", size index {args.sweep_index} of its sweep" if args.config == 5 else "")
                                           if args.config <= 5 else
                                           "none: the paper's own 2D dam-break shape (PAPER.md:397), context only"),
                       "parallelism": "single GPU" if world == 1 else f"{world} independent replicas (no collective)",
                       "options": {k: scene.params.get(k) for k in ("ppe_operator", "cg_warm_start", "key_mode", "cell_div", "rebin_every", "row_skin")},
                       "pre_steps": int(getattr(args, "pre_steps", 0)),
                       "l2": "flushed before every timed step (256 MiB write, untimed)",
                       "timing": "CUDA events on the ctx stream around each mps_step(1), summed; max over ranks"},
            "gpu_launches": main["gpu_launches"], "clocks": main["clocks"], "bins_per_step": main["bins_per_step"],
            "fluid_particle_steps_per_sec": main["fluid_particle_steps_per_sec"],
            "roofline": main["roofline"], "kernels": main["kernels"], "units": main["units"],
            "e2e": e2e, "cpu_baseline": cpu,
        }
        if "cg" in main:
            out["cg"] = main["cg"]
            out["cg_iters_per_step"] = main["cg"]["iters_per_step"]
            out["cg_iters_per_sec"] = main["cg"]["iters_per_sec"]
        if other:
            out["routes"] = other
        if developed:
            out["developed_flow"] = developed
        print(json.dumps(out))
    if world > 1:
        torch.distributed.destroy_process_group()


def run_reference(args):
    """The reference arm of this tier: the CPU oracle, as it stands, on host cores.

    Each timed "step" is one whole oracle step of a BOUNDED SAMPLE of the workload (sample_scene):
    the same shape, parameters and route at a size where --steps 20 --warmup 5 ends within a few
    minutes (one oracle PPE step of the 2M-particle default takes minutes).  particle-steps/s is
    normalised by the sample's particle count."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from oracle import build as orc_build
    orc_build.build()
    from oracle import mps_oracle as O
    full, route = make_scene(args, 0)
    sample, what = sample_scene(args, full)
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
