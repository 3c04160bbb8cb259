"""Turns `ncu --page raw --csv` output into the text summaries kept under profiles/.

    ncu -i rep.ncu-rep --page raw --csv | python ncu_summary.py [--kernel REGEX] > summary.md
    ncu -i rep.ncu-rep --page raw --csv | python ncu_summary.py --figures --cells N \
        --source "<the ncu command that wrote the report>" > profiles/<name>_figures.json

    ncu -i rep.ncu-rep --page source --csv | python ncu_summary.py --source-page --cells N

Default: a markdown table, one column per profiled launch, of the metrics that explain a kernel of this library
(duration, DRAM bytes, pipe and issue utilisation, shared-memory wavefronts, stall reasons).  --figures: the
numbers bench.py reads back (per-launch DRAM traffic of the corrector; N = cells one launch updates); with
--source-csv FILE (the `--page source --csv` export of the same report) also the fp64 instructions the two stage
kernels execute per cell-update (DFMA + DMUL + DADD + DSETP thread instructions, predicated on).  --source-page:
per kernel the SASS opcode mix (share of warp instructions, thread instructions per cell-update, shared-memory
wavefronts) and the warp-stall samples by reason.  Reads only its inputs; runs nothing.
"""
import collections
import argparse
import csv
import json
import re
import sys

# The kernel sources the stage-kernel figures depend on: their hash goes into the figures file, bench.py compares it
# with the sources it runs and flags a stale file.
STAGE_SOURCES = ("sfh_stage.cuh", "sfh_device.cuh", "sfh_kernels.cuh")


def stage_source_hash():
    import hashlib
    import os
    h = hashlib.sha256()
    csrc = os.path.join(os.path.dirname(os.path.abspath(__file__)), "paper_2604_21438_b200", "csrc")
    for name in STAGE_SOURCES:
        with open(os.path.join(csrc, name), "rb") as f:
            h.update(f.read())
    return h.hexdigest()


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


FP64_OPS = ("DFMA", "DMUL", "DADD", "DSETP")
STALL_COLS = ("stall_barrier", "stall_branch_resolving", "stall_dispatch", "stall_long_sb", "stall_math", "stall_mio",
              "stall_no_inst", "stall_not_selected", "stall_selected", "stall_short_sb", "stall_wait", "stall_lg")


def read_source(stream):
    """{kernel name: [row dict per SASS instruction]} from `ncu --page source --csv`."""
    out, kern, hdr = collections.OrderedDict(), None, None
    for r in csv.reader(stream):
        if not r:
            continue
        if r[0] == "Kernel Name":
            kern = r[1]
            out[kern] = []
        elif r[0] == "Address":
            hdr = r
        elif kern is not None and hdr is not None and len(r) == len(hdr):
            out[kern].append(dict(zip(hdr, r)))
    return out


def opcode_of(row):
    src = re.sub(r"^@!?U?P\w+\s+", "", row["Source"].strip())
    return src.split()[0].split(".")[0] if src else "?"


def count(row, name):
    try:
        return int(row.get(name) or 0)
    except ValueError:
        return 0


def fp64_per_cell(kernels, cells):
    """fp64 thread instructions (predicated on) per cell of the predictor + corrector launches in a source export."""
    tot = 0.0
    for name, rows in kernels.items():
        if re.search(r"stage_kernel|predictor_kernel|corrector_kernel", name):
            tot += sum(count(r, "Predicated-On Thread Instructions Executed") for r in rows if opcode_of(r) in FP64_OPS)
    return tot / cells if cells > 0 else None


def source_page(kernels, cells, kernel_re):
    for name, rows in kernels.items():
        if not re.search(kernel_re, name):
            continue
        warp, thr, wf, stalls = collections.Counter(), collections.Counter(), collections.Counter(), collections.Counter()
        for r in rows:
            op = opcode_of(r)
            warp[op] += count(r, "Instructions Executed")
            thr[op] += count(r, "Predicated-On Thread Instructions Executed")
            wf[op] += count(r, "L1 Wavefronts Shared")
            for c in STALL_COLS:
                stalls[c] += count(r, c)
        tot = sum(warp.values()) or 1
        print("### %s" % re.sub(r"^void |sfh::|\(int\)|\(bool\)|\(sfh::.*$", "", name))
        print()
        print("warp instructions %d; fp64 thread instructions per cell %.1f" %
              (tot, sum(thr[o] for o in FP64_OPS) / cells if cells > 0 else float("nan")))
        print()
        print("| opcode | share of warp instructions % | thread instructions per cell | shared-memory wavefronts |")
        print("|---|---|---|---|")
        for op, n in warp.most_common(24):
            print("| %s | %.2f | %.2f | %d |" % (op, 100.0 * n / tot, thr[op] / cells if cells > 0 else 0.0, wf[op]))
        ts = sum(stalls.values()) or 1
        print()
        print("warp-stall samples: " + ", ".join("%s %.1f %%" % (c[6:], 100.0 * v / ts) for c, v in stalls.most_common()))
        print()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--kernel", default=".", help="regex on the kernel name")
    ap.add_argument("--figures", action="store_true")
    ap.add_argument("--cells", type=float, default=0.0, help="--figures: cells one stage launch updates")
    ap.add_argument("--source", default="", help="--figures: the ncu command that wrote the report")
    ap.add_argument("--source-csv", default="", help="--figures: `--page source --csv` export of the same report")
    ap.add_argument("--source-page", action="store_true", help="standard input is a `--page source --csv` export")
    a = ap.parse_args()
    if a.source_page:
        source_page(read_source(sys.stdin), a.cells, a.kernel)
        return
    names, units, launches = read_raw(sys.stdin)
    launches = [l for l in launches if re.search(a.kernel, l["Kernel Name"])]
    if a.figures:
        out = {"source": a.source, "cells_per_launch": a.cells, "stage_source_sha256": stage_source_hash()}
        for stage, key in ((0, "predictor"), (1, "corrector")):
            sel = [l for l in launches if re.search(r"stage_kernel<(\(int\))?%d\b" % stage, l["Kernel Name"])]
            if not sel:
                continue
            n = len(sel)
            traffic = sum(si(l, units, "dram__bytes_read.sum") + si(l, units, "dram__bytes_write.sum") for l in sel) / n
            out[key + "_dram_bytes_per_launch"] = traffic
            out[key + "_time_us_under_ncu"] = sum(si(l, units, "gpu__time_duration.sum") for l in sel) / n * 1e6
            out[key + "_launches_averaged"] = n
        if a.source_csv and a.cells > 0:
            with open(a.source_csv) as f:
                out["fp64_thread_inst_per_cell_update"] = fp64_per_cell(read_source(f), a.cells)
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
