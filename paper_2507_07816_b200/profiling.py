"""Turn Nsight Compute captures of the library's kernels into the text summaries under profiles/.

    python -m paper_2507_07816_b200.profiling full    X.ncu-rep            -> markdown: metric table + hottest SASS
    python -m paper_2507_07816_b200.profiling list    launches.csv         -> markdown: per-kernel launch table
    python -m paper_2507_07816_b200.profiling summary KEY=X.ncu-rep[@profiles/file.md] ... [--commit HASH]
                                                                           -> profiles/ncu_summary.json

`summary` writes, per workload key ("cfg4:f32", "cfg3:u8", ...), what ONE launch of the
gather-accumulate kernel did under `ncu --set full`: DRAM bytes, warp instructions, issue-active,
FP64 pipe, duration, the kernel's name, the profile file holding the full command, and the commit
of the build that was captured.  bench.py reads that file for `roofline.traffic` and for the
instruction count of `roofline_binding`; it never runs this module.  Needs `ncu` on PATH (to read
the report; no GPU).
"""
from __future__ import annotations

import csv
import io
import json
import os
import subprocess
import sys
from collections import defaultdict

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WANT = [
    "gpu__time_duration.sum", "dram__bytes_read.sum", "dram__bytes_write.sum", "dram__bytes_read.sum.per_second",
    "dram__throughput.avg.pct_of_peak_sustained_elapsed",
    "lts__t_sector_hit_rate.pct", "lts__t_sectors.sum", "lts__t_bytes.sum", "lts__throughput.avg.pct_of_peak_sustained_elapsed",
    "l1tex__data_pipe_lsu_wavefronts_mem_shared.sum", "l1tex__data_bank_conflicts_pipe_lsu_mem_shared.sum",
    "l1tex__throughput.avg.pct_of_peak_sustained_elapsed", "smsp__inst_executed.sum",
    "smsp__inst_executed_pipe_fp64.sum",
    "sm__inst_executed_pipe_fp64.sum.pct_of_peak_sustained_active", "sm__pipe_fp64_cycles_active.avg.pct_of_peak_sustained_elapsed",
    "smsp__issue_active.avg.pct_of_peak_sustained_active", "sm__warps_active.avg.pct_of_peak_sustained_active",
    "sm__throughput.avg.pct_of_peak_sustained_elapsed", "sm__cycles_elapsed.avg", "launch__registers_per_thread",
    "launch__occupancy_limit_shared_mem", "launch__occupancy_limit_registers", "launch__occupancy_limit_warps",
    "launch__grid_size", "launch__block_size", "launch__shared_mem_per_block_dynamic",
]
STALL = "smsp__average_warps_issue_stalled_"
UNIT_SCALE = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9, "Tbyte": 1e12,
              "ns": 1e-6, "us": 1e-3, "ms": 1.0, "s": 1e3}


def _raw(rep):
    out = subprocess.run(["ncu", "-i", rep, "--page", "raw", "--csv"], capture_output=True, text=True, check=True).stdout
    rows = list(csv.reader(io.StringIO(out)))
    return rows[0], rows[1], rows[2:]


def _num(x: str) -> float:
    try:
        return float(x.replace(",", ""))
    except ValueError:
        return 0.0


def full(rep):
    hdr, units, data = _raw(rep)
    idx = {h: i for i, h in enumerate(hdr)}
    kn = idx.get("Kernel Name")
    print("Kernel(s): " + "; ".join(sorted({d[kn] for d in data})))
    print()
    print("| metric | unit | " + " | ".join(f"launch {i}" for i in range(len(data))) + " |")
    print("|---|---|" + "---|" * len(data))
    names = [n for n in WANT if n in idx] + sorted(h for h in hdr if h.startswith(STALL) and h.endswith("per_issue_active.ratio"))
    for n in names:
        vals = [d[idx[n]] for d in data]
        if n.startswith(STALL) and all(_num(v) < 0.08 for v in vals):
            continue
        print(f"| `{n}` | {units[idx[n]]} | " + " | ".join(vals) + " |")
    out = subprocess.run(["ncu", "-i", rep, "--page", "source", "--csv"], capture_output=True, text=True).stdout
    h, recs = None, []
    for r in csv.reader(io.StringIO(out)):
        if "Source" in r and any("Sampl" in c for c in r):
            h = {c: i for i, c in enumerate(r)}
            continue
        if h and len(r) >= len(h):
            recs.append(r)
    if not h:
        return
    scol = next(c for c in h if c.startswith("# Samples") or "Sampling (All" in c)
    ecol = next((c for c in h if c.startswith("Instructions Executed")), None) or next(c for c in h if "Instructions Executed" in c)
    tot = sum(int(_num(r[h[scol]])) for r in recs)
    top = sorted(range(len(recs)), key=lambda i: -_num(recs[i][h[scol]]))[:28]
    print()
    print(f"Hottest SASS instructions ({tot} warp-stall samples, first profiled launch):")
    print()
    print("| # | SASS | samples | share | inst executed |")
    print("|---|---|---|---|---|")
    for i in sorted(top):
        r = recs[i]
        print(f"| {i} | `{r[h['Source']].strip()}` | {int(_num(r[h[scol]]))} | {_num(r[h[scol]]) / max(tot, 1):.3f} | {int(_num(r[h[ecol]]))} |")


def launches(path):
    with open(path) as f:
        lines = [ln for ln in f if not ln.startswith("==")]
    agg = defaultdict(lambda: [0, 0.0])
    for r in csv.DictReader(io.StringIO("".join(lines))):
        if r.get("Metric Name") != "gpu__time_duration.sum":
            continue
        us = _num(r["Metric Value"]) * {"ns": 1e-3, "us": 1.0, "ms": 1e3, "s": 1e6}.get(r["Metric Unit"], 1e-3)
        a = agg[r["Kernel Name"]]
        a[0] += 1
        a[1] += us
    tot = sum(a[1] for a in agg.values())
    print("| kernel | launches | total ms | avg us | share |")
    print("|---|---|---|---|---|")
    for k, a in sorted(agg.items(), key=lambda kv: -kv[1][1]):
        print(f"| `{k[:110]}` | {a[0]} | {a[1] / 1e3:.3f} | {a[1] / a[0]:.1f} | {a[1] / tot:.4f} |")


def summary(argv):
    commit = None
    if "--commit" in argv:
        i = argv.index("--commit")
        commit = argv[i + 1]
        argv = argv[:i] + argv[i + 2:]
    if commit is None:
        commit = subprocess.run(["git", "-C", ROOT, "rev-parse", "--short", "HEAD"], capture_output=True, text=True).stdout.strip()
    path = os.path.join(ROOT, "profiles", "ncu_summary.json")
    doc = {"captures": {}}
    if os.path.exists(path):
        with open(path) as f:
            doc = json.load(f)
    doc["commit"] = commit
    doc["how"] = ("one launch of the gather-accumulate kernel per workload under `ncu --set full --clock-control none`; "
                  "the full command is in each entry's profile file; written by paper_2507_07816_b200/profiling.py summary")
    for item in argv:
        key, rest = item.split("=", 1)
        rep, _, prof = rest.partition("@")
        hdr, units, data = _raw(rep)
        idx = {h: i for i, h in enumerate(hdr)}
        d = data[0]

        def get(name, scale=True):
            if name not in idx:
                return None
            v = _num(d[idx[name]])
            return v * UNIT_SCALE.get(units[idx[name]], 1.0) if scale else v
        doc["captures"][key] = {
            "kernel": d[idx["Kernel Name"]], "profile": prof or None, "commit": commit,
            "duration_ms": get("gpu__time_duration.sum"),
            "dram_bytes_read": get("dram__bytes_read.sum"), "dram_bytes_write": get("dram__bytes_write.sum"),
            "inst_executed": get("smsp__inst_executed.sum", False),
            "issue_active_pct": get("smsp__issue_active.avg.pct_of_peak_sustained_active", False),
            "fp64_pipe_pct": get("sm__pipe_fp64_cycles_active.avg.pct_of_peak_sustained_elapsed", False),
            "lds_wavefronts": get("l1tex__data_pipe_lsu_wavefronts_mem_shared.sum", False),
            "l2_hit_pct": get("lts__t_sector_hit_rate.pct", False),
            "l2_sectors": get("lts__t_sectors.sum", False),
            "registers_per_thread": get("launch__registers_per_thread", False),
            "grid_size": get("launch__grid_size", False),
        }
    with open(path, "w") as f:
        json.dump(doc, f, indent=1, sort_keys=True)
        f.write("\n")
    print(path)


if __name__ == "__main__":
    if len(sys.argv) < 3 or sys.argv[1] not in ("full", "list", "summary"):
        raise SystemExit(__doc__)
    if sys.argv[1] == "summary":
        summary(sys.argv[2:])
    else:
        {"full": full, "list": launches}[sys.argv[1]](sys.argv[2])
