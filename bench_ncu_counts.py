"""bench_ncu_counts.py — turn one ncu capture of k_substep_fused into the numbers bench.py quotes beside its timings.

    ncu -i <rep> --page source --csv > src.csv ; ncu -i <rep> --page raw --csv > raw.csv
    python bench_ncu_counts.py --workload C4 --source src.csv --raw raw.csv --command "<the ncu command line>"

Reads the two text exports of a `ncu --set full --import-source on` capture (the capture itself is taken on the GPU box as
profiles/*.md describe; this script only parses text and can run anywhere), and merges into profiles/fp64_counts.txt,
per workload and averaged over the captured launches of k_substep_fused (C4 alternates its HLL and GLF instantiations):

  fp64_thread_inst_per_cell   executed, predicated-on thread instructions of the fp64 pipe (DFMA, DMUL, DADD, DSETP)
                              per interior cell of the grid
  pipe_fp64_active_pct        sm__inst_executed_pipe_fp64.avg.pct_of_peak_sustained_active
  dram_bytes_per_launch       dram__bytes_read.sum + dram__bytes_write.sum
  warp_inst_per_launch, time_ms_under_ncu, issue_active_pct
  issue_cycles_per_warp_of_cells   sum over the executed warp instructions of the cycles each holds the issue slot of its
                              SM sub-partition, per 32 cells: max(pipe, distinct even source registers, distinct odd
                              source registers) with pipe = 2 for the fp64 instructions and 1 for the rest (the register
                              file delivers one even and one odd register per cycle; a 64-bit operand is one of each).
                              rt_measure_fp64's 204/304/214/314 modes measure exactly these charges (DESIGN.md Sect. 5).
                              The operand reuse cache and the MUFU / shared-memory rates are left out.

together with the sha256 of the CUDA sources in the tree: bench.py refuses the numbers when the sources have changed
since (a kernel edit must be followed by a new capture)."""
import argparse
import csv
import json
import os
import re
import sys

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)
FP64_OPS = ("DFMA", "DMUL", "DADD", "DSETP")
UNIT = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9, "Tbyte": 1e12, "ns": 1e-6, "us": 1e-3, "ms": 1.0, "s": 1e3}


def issue_cycles(sass):
    """cycles one warp instruction holds the issue slot (see the module docstring)"""
    t = sass.strip().split(None, 1)
    if t and t[0].startswith("@"):
        t = t[1].split(None, 1) if len(t) > 1 else []
    if not t:
        return 1
    opc = t[0].split(".")[0]
    parts = [p.strip() for p in (t[1] if len(t) > 1 else "").rstrip(" ;").split(",")]
    if opc == "DSETP":
        srcs = parts[2:]
    elif opc in ("STS", "STG", "ST", "STL", "RED", "ATOMS", "ATOMG", "BRA", "BAR", "SYNCS", "UTMALDG", "CCTL"):
        srcs = parts
    else:
        srcs = parts[1:]
    wide = opc in FP64_OPS
    even, odd = set(), set()
    for p in srcs:
        for r in re.findall(r"(?<![A-Za-z])R(\d+)", p):
            n = int(r)
            (even if n % 2 == 0 else odd).add(n)
            if wide:
                (odd if n % 2 == 0 else even).add(n + 1)
    return max(2 if wide else 1, len(even), len(odd))


def parse_source(path, kernel="k_substep_fused"):
    """[(kernel name, fp64 thread instructions, warp instructions, issue cycles)] per captured launch (duplicate
    sections dropped)"""
    out, seen = [], set()
    name, hdr, fp64, warp, cyc = None, None, 0, 0, 0

    def flush():
        if name and kernel in name and (name, fp64, warp) not in seen:
            seen.add((name, fp64, warp))
            out.append((name, fp64, warp, cyc))

    with open(path, newline="") as fh:
        for r in csv.reader(fh):
            if not r:
                continue
            if r[0] == "Kernel Name":
                flush()
                name, hdr, fp64, warp, cyc = r[1], None, 0, 0, 0
                continue
            if r[0] == "Address":
                hdr = {h: i for i, h in enumerate(r)}
                continue
            if hdr is None:
                continue
            op = r[hdr["Source"]].split()
            if op and op[0].startswith("@"):
                op = op[1:]
            opc = op[0].split(".")[0] if op else ""
            warp += int(r[hdr["Instructions Executed"]])
            cyc += int(r[hdr["Instructions Executed"]]) * issue_cycles(r[hdr["Source"]])
            if opc in FP64_OPS:
                fp64 += int(r[hdr["Predicated-On Thread Instructions Executed"]])
    flush()
    return out


def parse_raw(path, kernel="k_substep_fused"):
    with open(path, newline="") as fh:
        rows = list(csv.reader(fh))
    hdr, units = rows[0], rows[1]
    col = {h: i for i, h in enumerate(hdr)}

    def val(r, key):
        i = col[key]
        return float(r[i]) * UNIT.get(units[i], 1.0)

    out = []
    for r in rows[2:]:
        if kernel not in r[col["Kernel Name"]]:
            continue
        out.append({"name": r[col["Kernel Name"]],
                    "time_ms": val(r, "gpu__time_duration.sum"),
                    "dram_bytes": val(r, "dram__bytes_read.sum") + val(r, "dram__bytes_write.sum"),
                    "pipe_fp64": val(r, "sm__inst_executed_pipe_fp64.avg.pct_of_peak_sustained_active"),
                    "issue": val(r, "sm__issue_active.avg.pct_of_peak_sustained_elapsed")})
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--workload", required=True)
    ap.add_argument("--source", required=True)
    ap.add_argument("--raw", required=True)
    ap.add_argument("--command", default="")
    a = ap.parse_args()
    import bench
    w = bench.make_workload(a.workload)
    src, raw = parse_source(a.source), parse_raw(a.raw)
    if not src or not raw:
        raise SystemExit("no k_substep_fused launch in the exports")
    mean = lambda xs: sum(xs) / len(xs)
    short = lambda n: (n[:n.index(">(") + 1] if ">(" in n else n).replace("void rtm1::", "").replace("(bool)", "")
    entry = {"launches": [short(s[0]) for s in src],
             "fp64_thread_inst_per_cell": round(mean([s[1] for s in src]) / w.ncells, 1),
             "fp64_thread_inst_per_cell_each": [round(s[1] / w.ncells, 1) for s in src],
             "warp_inst_per_launch": mean([s[2] for s in src]),
             "issue_cycles_per_warp_of_cells": round(mean([s[3] for s in src]) / (w.ncells / 32.0), 1),
             "issue_cycles_per_warp_of_cells_each": [round(s[3] / (w.ncells / 32.0), 1) for s in src],
             "pipe_fp64_active_pct": round(mean([r["pipe_fp64"] for r in raw]), 2),
             "issue_active_pct": round(mean([r["issue"] for r in raw]), 2),
             "dram_bytes_per_launch": mean([r["dram_bytes"] for r in raw]),
             "time_ms_under_ncu": [round(r["time_ms"], 4) for r in raw],
             "command": a.command}
    path = os.path.join(ROOT, "profiles", "fp64_counts.txt")
    try:
        with open(path) as fh:
            d = json.load(fh)
    except Exception:
        d = {}
    h = bench.csrc_hash()
    if d.get("csrc_hash") != h:
        d = {"csrc_hash": h, "workloads": {}}
    d["workloads"][a.workload] = entry
    with open(path, "w") as fh:
        json.dump(d, fh, indent=1)
    print(json.dumps(entry, indent=1))


if __name__ == "__main__":
    main()
