"""Turn an Nsight Compute report into the text summaries kept under profiles/.

    python -m paper_2105_01677_b200.ncu_summary REPORT.ncu-rep --title "..." --command "..." \
        --out profiles/r02_kernels_scene5_3.md [--traffic KEY=KERNEL_REGEX:DIVISOR ...]

Reads the report with `ncu -i REPORT --page raw --csv` (no GPU needed), writes one table row per
kernel name (launches captured, mean duration, DRAM bytes and % of peak, L2 / L1 hit rates, L1 and
L2 throughput, fp64 pipe, issue slots, achieved occupancy, registers) and, for every --traffic
argument, stores dram__bytes_read.sum + dram__bytes_write.sum of the first matching launch divided by
DIVISOR (the uses inside that launch, e.g. the CG iterations of one k_ppe_cg launch) in
profiles/r02_traffic.json under KEY -- the file bench.py reads its `roofline.traffic` from.
This is measurement tooling: it does no arithmetic of the method.
"""
from __future__ import annotations

import argparse
import csv
import io
import json
import os
import re
import subprocess

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
TRAFFIC = os.path.join(ROOT, "profiles", "r02_traffic.json")

COLS = [
    ("time us", "gpu__time_duration.sum", None),
    ("dram read MB", "dram__bytes_read.sum", None),
    ("dram write MB", "dram__bytes_write.sum", None),
    ("dram %", "gpu__dram_throughput.avg.pct_of_peak_sustained_elapsed", 1),
    ("L2 hit %", "lts__t_sector_hit_rate.pct", 1),
    ("L1 hit %", "l1tex__t_sector_hit_rate.pct", 1),
    ("l1tex %", "l1tex__throughput.avg.pct_of_peak_sustained_elapsed", 1),
    ("lts %", "lts__throughput.avg.pct_of_peak_sustained_elapsed", 1),
    ("fp64 pipe %", "sm__inst_executed_pipe_fp64.avg.pct_of_peak_sustained_active", 1),
    ("issue %", "sm__inst_issued.avg.pct_of_peak_sustained_active", 1),
    ("warps active %", "sm__warps_active.avg.pct_of_peak_sustained_active", 1),
    ("regs", "launch__registers_per_thread", 0),
]
UNIT_SCALE = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9, "Tbyte": 1e12,
              "ns": 1e-3, "us": 1.0, "ms": 1e3, "s": 1e6, "usecond": 1.0, "msecond": 1e3, "nsecond": 1e-3, "second": 1e6}


def read_report(path):
    txt = subprocess.run(["ncu", "-i", path, "--page", "raw", "--csv"], capture_output=True, text=True,
                         check=True).stdout
    rows = list(csv.reader(io.StringIO(txt)))
    hdr, units, body = rows[0], rows[1], rows[2:]
    col = {h: k for k, h in enumerate(hdr)}

    def val(r, name):
        if name not in col:
            return None
        v, u = r[col[name]], units[col[name]]
        try:
            x = float(v.replace(",", ""))
        except ValueError:
            return None
        return x * UNIT_SCALE.get(u, 1.0)   # bytes, or microseconds, or the plain number

    out = []
    for r in body:
        if len(r) < len(hdr):
            continue
        name = r[col["Kernel Name"]]
        short = re.sub(r"\(.*", "", name).replace("<unnamed>::", "")
        out.append({"name": short, "full": name, "grid": r[col.get("Grid Size", 0)], "block": r[col.get("Block Size", 0)],
                    **{c[1]: val(r, c[1]) for c in COLS}})
    return out


def hot_lines(path, launches, rx, top=14):
    """SASS lines by warp-stall samples (`ncu --page source --csv`) of the longest launch whose name matches rx."""
    idx = [k for k, l in enumerate(launches) if re.search(rx, l["full"])]
    if not idx:
        return [f"`{rx}`: no launch in the report"]
    best = max(idx, key=lambda k: launches[k]["gpu__time_duration.sum"] or 0.0)
    skip = idx.index(best)
    txt = subprocess.run(["ncu", "-i", path, "--page", "source", "--csv", "--kernel-name", "regex:" + rx],
                         capture_output=True, text=True).stdout
    # one block of rows per matching launch, each opened by a "Kernel Name" row: keep the block of the launch wanted
    blocks = []
    for r in csv.reader(io.StringIO(txt)):
        if r and r[0] == "Kernel Name":
            blocks.append([])
        elif blocks:
            blocks[-1].append(r)
    body = [r for r in (blocks[skip] if skip < len(blocks) else []) if len(r) > 5 and r[2].isdigit() and r[5].isdigit()]
    if not body:
        return [f"`{rx}`: no source page in the report"]
    tot, toti = sum(int(r[2]) for r in body), sum(int(r[5]) for r in body)
    out = [f"Hottest SASS lines of `{launches[best]['name']}` ({launches[best]['gpu__time_duration.sum']:.1f} us; {toti} warp "
           f"instructions, {tot} stall samples; `ncu --page source --csv`, sorted by samples):", "", "```"]
    for r in sorted(body, key=lambda r: -int(r[2]))[:top]:
        out.append(f"{100 * int(r[2]) / max(tot, 1):5.1f}% samples {100 * int(r[5]) / max(toti, 1):5.2f}% instr        {r[1].strip()}")
    return out + ["```"]


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("report")
    ap.add_argument("--title", default="")
    ap.add_argument("--command", default="", help="the full command that made the report (recorded in the summary)")
    ap.add_argument("--out", required=True)
    ap.add_argument("--traffic", action="append", default=[], help="KEY=KERNEL_REGEX:DIVISOR")
    ap.add_argument("--note", action="append", default=[])
    ap.add_argument("--hot", action="append", default=[],
                    help="KERNEL_REGEX: append the SASS lines with the most warp-stall samples of the longest launch that matches")
    ap.add_argument("--traffic-file", default=TRAFFIC, help="where the traffic table lives (default profiles/r02_traffic.json)")
    ap.add_argument("--source-name", default=None, help="path recorded as the entry's source (default: --out)")
    a = ap.parse_args()
    launches = read_report(a.report)
    groups = {}
    for l in launches:
        groups.setdefault(l["name"], []).append(l)
    # mps_step launches the kernels of its two skin bins in every step and those of a bin that is not needed
    # return at once: keep them apart from the launches that ran
    split = {}
    for name, ls in groups.items():
        tmax = max((l["gpu__time_duration.sum"] or 0.0) for l in ls)
        ran = [l for l in ls if (l["gpu__time_duration.sum"] or 0.0) >= 0.05 * tmax]
        idle = [l for l in ls if l not in ran]
        split[name] = ran
        if idle:
            split[name + " (bin not needed: returned at once)"] = idle
    groups = split
    lines = [f"# {a.title}", "", "Command (one B200 under `gpurun`, after the same command exited 0 without ncu):", "",
             "    " + a.command, "",
             f"Summary written by `python -m paper_2105_01677_b200.ncu_summary {os.path.basename(a.report)} ...` "
             "from `ncu --page raw --csv`; per-launch means over the captured launches of each kernel.", ""]
    lines += ["| kernel | launches | grid x block | " + " | ".join(c[0] for c in COLS) + " |",
              "|---|---|---|" + "---|" * len(COLS)]
    for name, ls in groups.items():
        cells = []
        for label, key, digits in COLS:
            vs = [l[key] for l in ls if l[key] is not None]
            if not vs:
                cells.append("-")
                continue
            m = sum(vs) / len(vs)
            if "MB" in label:
                cells.append(f"{m / 1e6:.2f}")
            elif label == "time us":
                cells.append(f"{m:.1f}")
            else:
                cells.append(f"{m:.{digits}f}")
        lines.append(f"| {name} | {len(ls)} | {ls[0]['grid']} x {ls[0]['block']} | " + " | ".join(cells) + " |")
    for n in a.note:
        lines += ["", n]
    for rx in a.hot:
        lines += ["", *hot_lines(a.report, launches, rx)]
    if a.traffic:
        try:
            with open(a.traffic_file) as f:
                table = json.load(f)
        except Exception:
            table = {}
        lines += ["", "Traffic entries written to `profiles/r02_traffic.json` (dram read + write of the first matching launch / uses):", ""]
        for t in a.traffic:
            key, rest = t.split("=", 1)
            rx, div = rest.rsplit(":", 1)
            hit = next((l for l in launches if re.search(rx, l["full"])), None)
            if hit is None:
                raise SystemExit(f"no launch matches {rx}")
            tot = (hit["dram__bytes_read.sum"] or 0.0) + (hit["dram__bytes_write.sum"] or 0.0)
            table[key] = {"dram_bytes_per_use": tot / float(div), "uses_in_launch": float(div),
                          "dram_bytes_launch": tot, "kernel": hit["name"], "launch_us": hit["gpu__time_duration.sum"],
                          "source": a.source_name or os.path.relpath(a.out, ROOT)}
            lines.append(f"* `{key}`: {tot / 1e6:.1f} MB / {div} = {tot / float(div) / 1e6:.2f} MB per use ({hit['name']})")
        with open(a.traffic_file, "w") as f:
            json.dump(table, f, indent=1, sort_keys=True)
            f.write("\n")
    with open(a.out, "w") as f:
        f.write("\n".join(lines) + "\n")
    print("\n".join(lines))


if __name__ == "__main__":
    main()
