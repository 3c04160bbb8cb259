#!/usr/bin/env python
"""bench.py — hydro cell-updates/s of the B200 AMR hydro step (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C2] [--impl ours|reference]

A "step" is one coarse step of the whole hot path (CFL reduction, ghost fill incl. prolongation,
predictor, corrector, flux registers, restriction, reflux; all sub-steps of the finer levels in
adaptive mode) over one synthetic problem; one cell-update = one predictor+corrector update of one
cell of one block of any level (the paper's unit).  Default workload: C2 =
BASELINE.json configs[1], uniform periodic 256^3 in 8^3 blocks (the paper's Table 5 shape).
Prints ONE JSON line (rank 0).  N > 1 runs N independent replicas, one per GPU (DESIGN.md:
"replicas only"; the path has no multi-GPU exchange in scope).
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "hydro cell-updates/sec (fp64, 1xB200)"
UNIT = "cell-updates/s"
CORRECTOR_BYTES_PER_CELL = 120.0   # read U^n, U^{n+1/2}, write U^{n+1}, 5 fp64 each
PREDICTOR_BYTES_PER_CELL = 80.0    # read U^n, write U^{n+1/2}
# dram__bytes_read.sum + dram__bytes_write.sum of one corrector launch on C2, from the ncu --set full
# capture summarised in profiles/ (None until captured)
CORRECTOR_TRAFFIC_BYTES_C2 = 1.490592e9 + 0.649133e9   # profiles/r1_c2_ncu_final.md
# fp64 instructions (DFMA + DMUL + DADD + DSETP) per cell-update of the two stage kernels, counted on the ncu
# source page (profiles/r1_c2_ncu_final.md), and the measured DFMA issue rate of this B200 (profiles/r1_fp64_peak.txt)
FP64_INST_PER_CELL_UPDATE = 236.0 + 380.0
FP64_PEAK_INST_PER_S = 17.069e12


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", default="C2", choices=["C1", "C2", "C3", "C4", "C5"])
    ap.add_argument("--scale", type=int, default=1, help="shrink the base grid (debugging only; invalid as a bench value)")
    ap.add_argument("--riemann", default="hllc", choices=["hllc", "roe"],
                    help="Riemann solver (PAPER.md:126); the paper's benchmarks and BASELINE.json use HLLC")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--extras", action="store_true",
                    help="also time the regrid pieces (refinement indicators, state transfer) on this config")
    return ap.parse_args()


def peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json, copy bandwidth)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md)"


class ClockSampler:
    """SM clock and throttle reasons during the timed region.  NVML is polled from a thread every
    few ms (the timed region of the default run lasts tens of ms, shorter than one `nvidia-smi -lms`
    period); `nvidia-smi` is the fallback when the NVML binding is missing."""
    REASONS = (("hw_slowdown", 0x8), ("hw_thermal_slowdown", 0x40), ("sw_thermal_slowdown", 0x20),
               ("sw_power_cap", 0x4))

    def __init__(self, index):
        self.rows = []          # (time, sm_mhz, reasons bitmask, power W)
        self.max_mhz = None
        self.stop_flag = False
        self.th = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = float(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
            self._sample()
            self.th = threading.Thread(target=self._poll, daemon=True)
            self.th.start()
        except Exception:
            self.nv = None
            self._smi(index)

    def _sample(self):
        nv = self.nv
        mhz = float(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
        try:
            why = int(nv.nvmlDeviceGetCurrentClocksEventReasons(self.h))
        except Exception:
            why = int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h))
        try:
            watts = nv.nvmlDeviceGetPowerUsage(self.h) / 1e3
        except Exception:
            watts = 0.0
        self.rows.append((time.time(), mhz, why, watts))

    def _poll(self):
        while not self.stop_flag:
            try:
                self._sample()
            except Exception:
                break
            time.sleep(0.002)

    def _smi(self, index):
        q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
             "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
             "clocks_event_reasons.sw_power_cap")
        try:
            res = subprocess.run(["nvidia-smi", "-i", str(index), "--query-gpu=" + q, "--format=csv,noheader,nounits"],
                                 capture_output=True, text=True, timeout=20)
            r = res.stdout.strip().split(", ")
            self.max_mhz = float(r[1])
            why = sum(bit for (_, bit), x in zip(self.REASONS, r[3:7]) if x.strip().lower() == "active")
            self.rows.append((time.time(), float(r[0]), why, float(r[2])))
        except Exception:
            pass

    def stop(self, t0, t1):
        self.stop_flag = True
        if self.th is not None:
            self.th.join(timeout=2)
        rows = [r for r in self.rows if t0 <= r[0] <= t1]
        where = "timed region"
        if not rows:
            rows, where = self.rows, "around the timed region"
        if not rows:
            return None
        sm = sorted(r[1] for r in rows)
        mask = 0
        for r in rows:
            mask |= r[2]
        return {"sm_mhz": sm[len(sm) // 2], "sm_max_mhz": self.max_mhz, "sm_mhz_min": sm[0],
                "reasons": [n for n, bit in self.REASONS if mask & bit], "samples": len(rows), "window": where,
                "power_w_max": max(r[3] for r in rows), "source": "nvml" if self.nv else "nvidia-smi"}


def cell_updates(census, nupd):
    return float(sum(512 * c * int(n) for c, n in zip(census, nupd)))


def max_over_ranks(ms, world, device="cpu"):
    """The job's time is the slowest rank's (device time, max over ranks)."""
    if world <= 1:
        return float(ms)
    import torch
    import torch.distributed as dist
    t = torch.tensor([ms], device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_value(cu_per_rank, ms, world):
    """N independent replicas of the same workload: the units all ranks processed / the time."""
    return world * cu_per_rank / (ms * 1e-3)


def oracle_sample(config, scale_hint, riemann="hllc"):
    """The oracle on a bounded sample of the same workload: the same recipe on a smaller base grid."""
    from oracle import oracle_for
    from sfh_inputs import make_config
    sample_scale = {"C1": 1, "C2": 1, "C3": 2, "C4": 2, "C5": 4}[config] * max(1, scale_hint)
    p = make_config(config, sample_scale)
    o = oracle_for(p)
    o.set_riemann(riemann)
    o.restrict_all(0)
    n = p.nb0[0] * 8
    what = "%s recipe at base %d^3 (1/%d of the base cells), blocks/level %s" % (config, n, sample_scale ** 3, p.census())
    return p, o, what


def run_reference(args):
    """--impl reference: the CPU oracle as it stands, on the host cores (rank 0 only)."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    p, o, what = oracle_sample(args.config, args.scale, args.riemann)
    cores = len(os.sched_getaffinity(0))
    for _ in range(args.warmup):
        o.advance(1, p.mode)
    o.nupd[:] = 0
    t0 = time.perf_counter()
    o.advance(args.steps, p.mode)
    dt = time.perf_counter() - t0
    cu = cell_updates(p.census(), o.nupd)
    val = cu / dt
    sample = what + ", %d coarse step(s) per run" % args.steps
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": p.notes.get("workload", p.name), "config": args.config, "sample": sample,
                   "riemann": args.riemann},
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}))


def main():
    args = parse()
    if args.impl == "reference":
        return run_reference(args)

    import numpy as np
    import torch
    import torch.distributed as dist
    import paper_2604_21438_b200 as sfh
    from sfh_inputs import make_config

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (libsfh has no CPU fallback)")
    torch.cuda.set_device(local)
    dev = "cuda:%d" % local
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device(dev))

    p = make_config(args.config, args.scale)
    census = p.census()
    g = sfh.Mesh.from_problem(p, device=dev)
    g.set_riemann(args.riemann)
    U0 = torch.from_numpy(p.U).pin_memory()
    Ud = U0.to(dev)

    def reset():
        g.set_state(Ud)
        g.restrict_all(0)
        g.nupd[:] = 0
        torch.cuda.synchronize()

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- warm-up
    reset()
    for _ in range(max(args.warmup, 0)):
        g.advance(1, p.mode)
    bad_warm = g.status()

    # ---- timed region: K coarse steps, state resident in HBM (no per-launch events: they cost 1.5 % on C2
    # and 5 % on C4, measured; the kernel spans are taken in a second pass of the same K steps below)
    reset()
    l0 = g.launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    sampler = ClockSampler(local) if rank == 0 else None
    t0 = time.time()
    e0.record()
    g.advance(args.steps, p.mode)
    e1.record()
    barrier()
    t1 = time.time()
    clocks = sampler.stop(t0, t1) if sampler else None
    ms = e0.elapsed_time(e1)
    launches = g.launch_count() - l0
    nupd = g.nupd.copy()
    cu = cell_updates(census, nupd)
    bad = g.status()
    ms = max_over_ranks(ms, world, dev)
    value = whole_job_value(cu, ms, world)

    # ---- the same K steps again with CUDA events around every launch (sfh_profile): per-kernel spans
    reset()
    g.profile(True)
    g.kernel_times()
    g.advance(args.steps, p.mode)
    torch.cuda.synchronize()
    kt = g.kernel_times()
    g.profile(False)

    # ---- end to end through sfh_advance_host: pinned host buffers, H2D and D2H every step
    reset()
    hin = g.get_state().cpu().pin_memory()    # restriction-consistent initial hierarchy, caller layout
    hout = torch.empty_like(hin).pin_memory()
    g.advance_host(hin, hout, 1, p.mode)      # warm
    g.nupd[:] = 0
    barrier()
    e0.record()
    for _ in range(args.steps):
        g.advance_host(hin, hout, 1, p.mode)
        hin, hout = hout, hin
    e1.record()
    barrier()
    ms_e2e = e0.elapsed_time(e1)
    cu_e2e = cell_updates(census, g.nupd)
    ms_e2e = max_over_ranks(ms_e2e, world, dev)
    state_bytes = int(U0.numel() * 8)

    # ---- roofline of the dominant kernel (the corrector stage), CUDA events around each launch
    peak, peak_src = peaks()
    c_ms, c_n = kt["corrector"]
    corr_bytes = CORRECTOR_BYTES_PER_CELL * cu            # every cell-update passes the corrector once
    achieved = corr_bytes / (c_ms * 1e-3) / 1e9 if c_ms > 0 else 0.0
    roofline = {"bound": "hbm", "kernel": "stage_kernel<1> (corrector)", "achieved": achieved, "peak": peak,
                "unit": "GB/s", "frac": achieved / peak, "peak_source": peak_src,
                "traffic": CORRECTOR_TRAFFIC_BYTES_C2 if (args.config == "C2" and args.scale == 1 and
                                                          args.riemann == "hllc") else None,
                "algorithmic_bytes_per_launch": corr_bytes / max(c_n, 1), "launches": c_n,
                "avg_launch_ms": c_ms / max(c_n, 1),
                "kernel_ms": {k: round(v[0], 4) for k, v in kt.items()},
                "kernel_launches": {k: v[1] for k, v in kt.items()},
                "step_hbm_GBps_at_200B_per_update": 200.0 * cu / (ms * 1e-3) / 1e9}
    # the second ceiling: the stage kernels are bound by fp64 instruction issue, not by HBM
    stage_ms = kt["predictor"][0] + kt["corrector"][0]
    f64 = FP64_INST_PER_CELL_UPDATE * cu / (stage_ms * 1e-3) if stage_ms > 0 else 0.0
    roofline_fp64 = {"bound": "alu", "kernel": "stage_kernel<0> + stage_kernel<1>", "achieved": f64,
                     "peak": FP64_PEAK_INST_PER_S, "unit": "fp64 inst/s", "frac": f64 / FP64_PEAK_INST_PER_S,
                     "inst_per_cell_update": FP64_INST_PER_CELL_UPDATE,
                     "peak_source": "measured DFMA issue rate (profiles/r1_fp64_peak.txt)"}
    if args.riemann != "hllc":
        roofline_fp64 = None          # the instruction count was taken with the HLLC kernels

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    extras = None
    if args.extras and world == 1:
        # the indicator kernel reads the state once (40 B/cell + halos through L2); the
        # transfer onto an identical mesh copies it (80 B/cell)
        reset()
        g.fill_ghosts(-1, 0, 0, 0.0)
        ncell = 512.0 * sum(census)
        ev = [torch.cuda.Event(enable_timing=True) for _ in range(2)]

        def timed(fn, reps=5):
            fn()
            torch.cuda.synchronize()
            ev[0].record()
            for _ in range(reps):
                fn()
            ev[1].record()
            torch.cuda.synchronize()
            return ev[0].elapsed_time(ev[1]) / reps

        ms_c = timed(lambda: g.refine_indicator(0))
        ms_j = timed(lambda: g.refine_indicator(1))
        g2 = sfh.Mesh.from_problem(p, device=dev)
        ms_t = timed(lambda: g2.transfer_from(g), reps=3)
        extras = {"refine_indicator_curvature": {"ms": ms_c, "GBps_at_40B_per_cell": 40.0 * ncell / ms_c / 1e6},
                  "refine_indicator_jeans": {"ms": ms_j, "GBps_at_40B_per_cell": 40.0 * ncell / ms_j / 1e6},
                  "transfer_state_identity": {"ms": ms_t, "GBps_at_80B_per_cell": 80.0 * ncell / ms_t / 1e6,
                                              "note": "includes building and uploading the block map on the host"}}
        del g2

    cpu = None
    if world == 1 and not args.no_cpu_baseline:
        # the oracle as it stands on this box's host cores, on a bounded sample: whole coarse steps of
        # the same recipe (at a smaller base grid for the large configs) until ~12 s have passed
        ps, o, what = oracle_sample(args.config, args.scale, args.riemann)
        tt, nst = time.perf_counter(), 0
        while nst < max(args.steps, 1) and (nst == 0 or time.perf_counter() - tt < 12.0):
            o.advance(1, ps.mode)
            nst += 1
        tt = time.perf_counter() - tt
        cpu = {"value": cell_updates(ps.census(), o.nupd) / tt, "unit": UNIT, "cores": len(os.sched_getaffinity(0)),
               "kind": "oracle", "sample": what + ", %d coarse step(s), %.1f s" % (nst, tt)}

    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": p.notes.get("workload", p.name), "config": args.config, "scale": args.scale,
                   "riemann": args.riemann,
                   "blocks_per_level": census, "updates_per_level": [int(x) for x in nupd],
                   "mode": "adaptive" if p.mode else "synchronous",
                   "l2": "inputs larger than L2 (one state copy %.0f MB vs 126 MB L2)" % (state_bytes / 1e6),
                   "kernel_spans": "second pass of the same K steps with CUDA events around every launch",
                   "parallelism": "replicas x%d" % world, "bad_cells": int(bad), "bad_cells_after_warmup": int(bad_warm)},
        "clocks": clocks,
        "e2e": {"value": whole_job_value(cu_e2e, ms_e2e, world), "unit": UNIT, "h2d_bytes_per_step": state_bytes,
                "d2h_bytes_per_step": state_bytes, "ms_per_step": ms_e2e / args.steps},
        "gpu_launches": int(launches),
        "roofline": roofline,
        "roofline_fp64": roofline_fp64,
        "extras": extras,
        "cpu_baseline": cpu,
    }
    print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
