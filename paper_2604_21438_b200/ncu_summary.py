"""Turns `ncu --page raw --csv` output into the text summaries kept under profiles/.

    ncu -i rep.ncu-rep --page raw --csv | python -m paper_2604_21438_b200.ncu_summary [--kernel REGEX] > summary.md
    ncu -i rep.ncu-rep --page raw --csv | python -m paper_2604_21438_b200.ncu_summary --figures --cells N \
        --source "<the ncu command that wrote the report>" > profiles/<name>_figures.json

Default: a markdown table, one column per profiled launch, of the metrics that explain a kernel of this library
(duration, DRAM bytes, pipe and issue utilisation, shared-memory wavefronts, stall reasons).  --figures: the
numbers bench.py reads back (per-launch DRAM traffic of the corrector, fp64 instructions per cell-update of the two
stage kernels; N = cells one launch updates).  Reads only its standard input; runs nothing.
"""
import argparse
import csv
import json
import re
import sys

METRICS = [
    "gpu__time_duration.sum",
    "dram__bytes_read.sum",
    "dram__bytes_write.sum",
    "gpu__dram_throughput.avg.pct_of_peak_sustained_elapsed",
    "sm__pipe_fp64_cycles_active.avg.pct_of_peak_sustained_active",
    "sm__inst_executed_pipe_fp64.sum",
    "smsp__issue_active.avg.pct_of_peak_sustained_active",
    "smsp__inst_executed.sum",
    "l1tex__data_pipe_lsu_wavefronts_mem_shared.sum",
    "l1tex__data_pipe_lsu_wavefronts_mem_shared.sum.pct_of_peak_sustained_elapsed",
    "l1tex__data_bank_conflicts_pipe_lsu_mem_shared.sum",
    "lts__t_sector_hit_rate.pct",
    "sm__warps_active.avg.pct_of_peak_sustained_active",
    "launch__registers_per_thread",
    "launch__grid_size",
    "launch__block_size",
    "sm__cycles_elapsed.avg",
    "sm__cycles_elapsed.avg.per_second",
]
STALL = re.compile(r"smsp__average_warps_issue_stalled_(\w+)_per_issue_active\.ratio$")
SCALE = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9, "Tbyte": 1e12,
         "ns": 1e-9, "us": 1e-6, "ms": 1e-3, "s": 1.0, "usecond": 1e-6, "nsecond": 1e-9, "msecond": 1e-3, "second": 1.0}


def read_raw(stream):
    rows = [r for r in csv.reader(stream) if r]
    start = next(i for i, r in enumerate(rows) if "Kernel Name" in r)
    names, units = rows[start], rows[start + 1]
    launches = [dict(zip(names, r)) for r in rows[start + 2:] if len(r) == len(names)]
    return names, dict(zip(names, units)), launches


def number(text):
    try:
        return float(text.replace(",", ""))
    except ValueError:
        return None


def si(launch, units, name):
    """Value of a metric in base units (bytes, seconds) where the unit column gives a scale."""
    v = number(launch.get(name, ""))
    if v is None:
        return None
    return v * SCALE.get(units.get(name, ""), 1.0)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--kernel", default=".", help="regex on the kernel name")
    ap.add_argument("--figures", action="store_true")
    ap.add_argument("--cells", type=float, default=0.0, help="--figures: cells one stage launch updates")
    ap.add_argument("--source", default="", help="--figures: the ncu command that wrote the report")
    a = ap.parse_args()
    names, units, launches = read_raw(sys.stdin)
    launches = [l for l in launches if re.search(a.kernel, l["Kernel Name"])]
    if a.figures:
        out = {"source": a.source, "cells_per_launch": a.cells}
        f64 = 0.0
        for stage, key in ((0, "predictor"), (1, "corrector")):
            sel = [l for l in launches if re.search(r"stage_kernel<(\(int\))?%d\b" % stage, l["Kernel Name"])]
            if not sel:
                continue
            n = len(sel)
            traffic = sum(si(l, units, "dram__bytes_read.sum") + si(l, units, "dram__bytes_write.sum") for l in sel) / n
            inst = sum(number(l.get("sm__inst_executed_pipe_fp64.sum", "")) or 0.0 for l in sel) / n
            out[key + "_dram_bytes_per_launch"] = traffic
            out[key + "_fp64_warp_inst_per_launch"] = inst
            out[key + "_time_us_under_ncu"] = sum(si(l, units, "gpu__time_duration.sum") for l in sel) / n * 1e6
            out[key + "_launches_averaged"] = n
            f64 += inst * 32.0
        if a.cells > 0 and f64 > 0:
            out["fp64_thread_inst_per_cell_update"] = f64 / a.cells
        json.dump(out, sys.stdout, indent=1)
        print()
        return
    stall = sorted(n for n in names if STALL.search(n))
    cols = ["%s #%d" % (re.sub(r"^void |sfh::|\(.*$", "", l["Kernel Name"]), i) for i, l in enumerate(launches)]
    print("| metric | unit | " + " | ".join(cols) + " |")
    print("|---|---|" + "---|" * len(cols))
    for n in METRICS + stall:
        if n not in units:
            continue
        label = STALL.search(n).group(1) + " (stall, warps per issue)" if STALL.search(n) else n
        print("| %s | %s | %s |" % (label, units[n], " | ".join(l.get(n, "") for l in launches)))


if __name__ == "__main__":
    main()
