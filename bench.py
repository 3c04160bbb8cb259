#!/usr/bin/env python
"""bench.py — hydro cell-updates/s of the B200 AMR hydro step (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C2] [--impl ours|reference]
                    [--per-config C3,C4,C5 | --no-per-config] [--peaks]

A "step" is one coarse step of the whole hot path (CFL reduction, ghost fill incl. prolongation,
predictor, corrector, flux registers, restriction, reflux; all sub-steps of the finer levels in
adaptive mode) over one synthetic problem; one cell-update = one predictor+corrector update of one
cell of one block of any level (the paper's unit).  Headline workload: C2 =
BASELINE.json configs[1], uniform periodic 256^3 in 8^3 blocks (the paper's Table 5 shape); the same
JSON line carries a `config.per_config` record for the other full-size configs (C3, C4, C5), each timed
the same way.  K steps are timed as ceil(K / nsteps) runs of the configured length (BASELINE.json: 10 steps
for C2-C4, 5 for C5) from the initial state, with an untimed re-initialisation between runs, so that no
number is taken on a state older than the config describes (`bad_cells` counts non-positive rho / P).
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
CORRECTOR_BYTES_PER_CELL = 120.0   # read U^n, W^{n+1/2}, write U^{n+1}, 5 fp64 each
STEP_BYTES_PER_CELL_UPDATE = 200.0  # predictor 80 + corrector 120
# Figures that come from an ncu capture, not from this run: per-launch DRAM traffic of the corrector and the
# fp64 instructions the two stage kernels execute per cell-update.  Written by
#   ncu -i <report> --page raw --csv | python ncu_summary.py --json
# (the full command is in the file) and tracked under profiles/.
NCU_FIGURES = os.path.join(ROOT, "profiles", "r3_c2_stage_figures.json")


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
    ap.add_argument("--threads", type=int, default=0, help="--impl reference: OpenMP threads of the oracle (0 = all cores)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--per-config", default="C3,C4,C5", help="other full-size configs reported in config.per_config")
    ap.add_argument("--no-per-config", action="store_true")
    ap.add_argument("--peaks", action="store_true", help="print the measured fp64 issue rates of this device and exit")
    ap.add_argument("--nscalar", type=int, default=0,
                    help="passive scalars advected with the gas (eq. 12-13, PAPER.md:80-88; SURVEY.md 8(f) row 4): smooth "
                         "seeded concentrations, 40 B more per scalar and cell-update")
    ap.add_argument("--ncell", type=int, default=8, choices=[8, 16],
                    help="hand the workload over in blocks of 16^3 cells (sfh.h; PAPER.md:536, 579): the same cells and the "
                         "same kernels on the 8^3 octants, only the caller's layout differs")
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


def ncu_figures():
    """The figures file, plus "stale": True when the stage-kernel sources differ from the ones it was captured on
    (or the file does not say which those were)."""
    try:
        with open(NCU_FIGURES) as f:
            fig = json.load(f)
    except Exception:
        return {}
    try:
        import ncu_summary
        fig["stale"] = fig.get("stage_source_sha256") != ncu_summary.stage_source_hash()
    except Exception:
        fig["stale"] = True
    return fig


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

    def stop(self, windows):
        """windows: [(t0, t1)] wall-clock spans of the timed runs."""
        self.stop_flag = True
        if self.th is not None:
            self.th.join(timeout=2)
        rows = [r for r in self.rows if any(a <= r[0] <= b for a, b in windows)]
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


def cell_updates(census, nupd, ncell=8):
    return float(sum(ncell ** 3 * c * int(n) for c, n in zip(census, nupd)))


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


def run_lengths(steps, nsteps):
    """K steps as runs of at most the configured length: [nsteps, nsteps, ..., remainder]."""
    nsteps = max(1, int(nsteps))
    out = [nsteps] * (steps // nsteps)
    if steps % nsteps:
        out.append(steps % nsteps)
    return out or [0]


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
    if args.threads > 0:
        os.environ["OMP_NUM_THREADS"] = str(args.threads)      # before the oracle's library is loaded
    p, o, what = oracle_sample(args.config, args.scale, args.riemann)
    cores = args.threads if args.threads > 0 else len(os.sched_getaffinity(0))
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


def measure(sfh, torch, name, args, dev, world, barrier, steps, warmup, sampler_index=None, e2e=False):
    """One full-size config on this rank: value pass (device-resident, CUDA events around each run of the configured
    length), kernel-span pass (same runs with events around every launch), optionally the end-to-end pass."""
    from sfh_inputs import make_config
    p = make_config(name, args.scale)
    if args.nscalar > 0:
        import numpy as np
        from sfh_inputs import add_scalars
        tp = 2.0 * np.pi
        p = add_scalars(p, [(lambda X, Y, Z, q=q: 0.5 + 0.4 * np.sin(tp * (X + 0.13 * q)) * np.cos(tp * (Y - 0.07 * q)) *
                             np.cos(tp * Z)) for q in range(args.nscalar)])
    if args.ncell == 16:
        from sfh_inputs import to16
        p = to16(p)[0]
    census = p.census()
    g = sfh.Mesh.from_problem(p, device=dev)
    g.set_riemann(args.riemann)
    U0 = torch.from_numpy(p.U).pin_memory()
    Ud = U0.to(dev)
    state_bytes = int(U0.numel() * 8)
    runs = run_lengths(steps, p.nsteps) if steps > 0 else [p.nsteps]     # steps 0: one run of the configured length

    def reset():
        g.set_state(Ud)
        g.restrict_all(0)
        g.nupd[:] = 0
        torch.cuda.synchronize()

    # ---- warm-up
    reset()
    for _ in range(max(warmup, 0)):
        g.advance(1, p.mode)
    bad_warm = g.status()

    # ---- timed region: the runs, state resident in HBM (no per-launch events here: they cost 1.5 % on C2 and 5 %
    # on C4, measured; the kernel spans are taken in a second pass of the same runs below)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    sampler = ClockSampler(sampler_index) if sampler_index is not None else None
    ms, launches, cu, bad, windows = 0.0, 0, 0.0, 0, []
    nupd_tot = None
    for n in runs:
        reset()
        l0 = g.launch_count()
        barrier()
        t0 = time.time()
        e0.record()
        g.advance(n, p.mode)
        e1.record()
        barrier()
        windows.append((t0, time.time()))
        ms += e0.elapsed_time(e1)
        launches += g.launch_count() - l0
        cu += cell_updates(census, g.nupd, args.ncell)
        nupd_tot = g.nupd.copy() if nupd_tot is None else nupd_tot + g.nupd
        bad = max(bad, g.status())
    clocks = sampler.stop(windows) if sampler else None
    ms = max_over_ranks(ms, world, dev)
    value = whole_job_value(cu, ms, world)

    # ---- the same runs again with CUDA events around every launch (sfh_profile): per-kernel spans
    g.profile(True)
    g.kernel_times()
    kt = None
    for n in runs:
        reset()
        g.kernel_times()              # drop the spans of the reset (none are timed) before the run
        g.advance(n, p.mode)
        torch.cuda.synchronize()
        k = g.kernel_times()
        kt = k if kt is None else {c: (kt[c][0] + k[c][0], kt[c][1] + k[c][1]) for c in k}
    g.profile(False)

    peak, peak_src = peaks()
    c_ms, c_n = kt["corrector"]
    corr_bytes = CORRECTOR_BYTES_PER_CELL * cu            # every cell-update passes the corrector once
    achieved = corr_bytes / (c_ms * 1e-3) / 1e9 if c_ms > 0 else 0.0
    figs = ncu_figures()
    is_ref_case = name == "C2" and args.scale == 1 and args.riemann == "hllc"
    roofline = {"bound": "hbm", "kernel": "stage_kernel<1> (corrector)", "achieved": achieved, "peak": peak,
                "unit": "GB/s", "frac": achieved / peak, "peak_source": peak_src,
                "traffic": figs.get("corrector_dram_bytes_per_launch") if is_ref_case else None,
                "traffic_source": figs.get("source") if is_ref_case else None,
                "traffic_stale": bool(figs.get("stale", True)) if is_ref_case else None,
                "algorithmic_bytes_per_launch": corr_bytes / max(c_n, 1), "launches": c_n,
                "avg_launch_ms": c_ms / max(c_n, 1),
                "kernel_ms": {k: round(v[0], 4) for k, v in kt.items()},
                "kernel_launches": {k: v[1] for k, v in kt.items()},
                "step_hbm_GBps_at_200B_per_update": STEP_BYTES_PER_CELL_UPDATE * cu / (ms * 1e-3) / 1e9,
                "step_frac_at_200B_per_update": STEP_BYTES_PER_CELL_UPDATE * cu / (ms * 1e-3) / 1e9 / peak}
    out = {"p": p, "g": g, "census": census, "workload": p.notes.get("workload", p.name),
           "mode": "adaptive" if p.mode else "synchronous", "value": value, "ms": ms, "steps": sum(runs), "runs": runs,
           "launches": launches, "nupd": nupd_tot, "bad": bad, "bad_warm": bad_warm, "clocks": clocks, "kt": kt,
           "roofline": roofline, "cu": cu, "state_bytes": state_bytes, "reset": reset}

    if e2e:
        # ---- end to end through sfh_advance_host: pinned host buffers, H2D and D2H of the state every step
        reset()
        hin = g.get_state().cpu().pin_memory()    # restriction-consistent initial hierarchy, caller layout
        hout = torch.empty_like(hin).pin_memory()
        h0 = hin.clone().pin_memory()
        g.advance_host(hin, hout, 1, p.mode)      # warm
        ms_e2e, cu_e2e = 0.0, 0.0
        for n in runs:
            hin.copy_(h0)
            g.nupd[:] = 0
            a, b = hin, hout
            barrier()
            e0.record()
            for _ in range(n):
                g.advance_host(a, b, 1, p.mode)
                a, b = b, a
            e1.record()
            barrier()
            ms_e2e += e0.elapsed_time(e1)
            cu_e2e += cell_updates(census, g.nupd, args.ncell)
        ms_e2e = max_over_ranks(ms_e2e, world, dev)
        out["e2e"] = {"value": whole_job_value(cu_e2e, ms_e2e, world), "unit": UNIT, "h2d_bytes_per_step": state_bytes,
                      "d2h_bytes_per_step": state_bytes, "ms_per_step": ms_e2e / sum(runs)}
        del hin, hout, h0
    return out


def main():
    args = parse()
    if args.impl == "reference":
        return run_reference(args)

    import torch
    import torch.distributed as dist
    import paper_2604_21438_b200 as sfh

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (libsfh has no CPU fallback)")
    torch.cuda.set_device(local)
    dev = "cuda:%d" % local
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device(dev))

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- the second ceiling's denominator, measured live: fp64 issue rate of this device
    fp64_peak = sfh.measure_fp64_rate(8)
    fp64_dep = sfh.measure_fp64_rate(1)
    if args.peaks:
        if rank == 0:
            print(json.dumps({"fp64_dfma_per_s": fp64_peak, "fp64_tflops": 2e-12 * fp64_peak,
                              "fp64_dfma_per_s_one_chain_per_thread": fp64_dep,
                              "how": "sfh_measure_fp64_rate: 2 CTAs x 1024 threads per SM, 8 (1) independent DFMA chains per "
                                     "thread, best of 3 launches, CUDA events", "hbm_gbs": peaks()[0], "hbm_source": peaks()[1]}))
        return

    m = measure(sfh, torch, args.config, args, dev, world, barrier, args.steps, args.warmup,
                sampler_index=local if rank == 0 else None, e2e=True)
    p, g = m["p"], m["g"]
    figs = ncu_figures()
    roofline_fp64 = None
    ipc = figs.get("fp64_thread_inst_per_cell_update")
    if ipc and args.riemann == "hllc":        # the instruction count was taken with the HLLC kernels
        stage_ms = m["kt"]["predictor"][0] + m["kt"]["corrector"][0]
        f64 = ipc * m["cu"] / (stage_ms * 1e-3) if stage_ms > 0 else 0.0
        roofline_fp64 = {"bound": "alu", "kernel": "stage_kernel<0> + stage_kernel<1>", "achieved": f64,
                         "peak": fp64_peak, "unit": "fp64 inst/s", "frac": f64 / fp64_peak, "inst_per_cell_update": ipc,
                         "inst_source": figs.get("source"), "inst_stale": bool(figs.get("stale", True)),
                         "peak_source": "measured in this run (sfh_measure_fp64_rate, 8 chains per thread)"}

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    extras = None
    if args.extras and world == 1:
        # the indicator kernel reads the state once (40 B/cell + halos through L2); the
        # transfer onto an identical mesh copies it (80 B/cell)
        m["reset"]()
        ncell = 512.0 * sum(m["census"])
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

    per_config = {}
    if world == 1 and not args.no_per_config and args.scale == 1:
        del m["g"], m["p"], m["reset"], g, p
        torch.cuda.empty_cache()
        for name in [c for c in args.per_config.split(",") if c and c != args.config]:
            t0 = time.time()
            q = measure(sfh, torch, name, args, dev, world, barrier, 0, args.warmup)
            per_config[name] = {
                "workload": q["workload"], "value": q["value"], "ms_per_step": q["ms"] / q["steps"],
                "steps": q["steps"], "mode": q["mode"],
                "blocks_per_level": q["census"], "updates_per_level": [int(x) for x in q["nupd"]],
                "bad_cells": int(q["bad"]), "bad_cells_after_warmup": int(q["bad_warm"]), "gpu_launches": int(q["launches"]),
                "roofline_frac": q["roofline"]["frac"],
                "step_hbm_GBps_at_200B_per_update": q["roofline"]["step_hbm_GBps_at_200B_per_update"],
                "step_frac_at_200B_per_update": q["roofline"]["step_frac_at_200B_per_update"],
                "kernel_ms": q["roofline"]["kernel_ms"], "kernel_launches": q["roofline"]["kernel_launches"],
                "wall_s_incl_input_generation": round(time.time() - t0, 1)}
            del q
            torch.cuda.empty_cache()

    # the driver's parsed record keeps the scalar entries of `config` only: the headline figures of the other configs
    # once more as scalars (value in cell-updates/s, fraction of the 200 B per cell-update HBM roofline)
    per_config_flat = {}
    for name, q in per_config.items():
        per_config_flat["%s_value" % name] = q["value"]
        per_config_flat["%s_step_frac_at_200B_per_update" % name] = q["step_frac_at_200B_per_update"]

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
        "metric": METRIC, "value": m["value"], "unit": UNIT, "n_gpus": world, "steps": m["steps"], "warmup": args.warmup,
        "ms_per_step": m["ms"] / m["steps"], "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": m["workload"], "config": args.config, "scale": args.scale, "riemann": args.riemann,
                   "blocks_per_level": m["census"], "updates_per_level": [int(x) for x in m["nupd"]],
                   "mode": m["mode"], "cells_per_block_edge": args.ncell, "passive_scalars": args.nscalar,
                   "algorithmic_bytes_per_cell_update": STEP_BYTES_PER_CELL_UPDATE + 40.0 * args.nscalar,
                   "timed_runs": m["runs"],
                   "l2": "inputs larger than L2 (one state copy %.0f MB vs 126 MB L2)" % (m["state_bytes"] / 1e6),
                   "kernel_spans": "second pass of the same runs with CUDA events around every launch",
                   "parallelism": "replicas x%d" % world, "bad_cells": int(m["bad"]),
                   "bad_cells_after_warmup": int(m["bad_warm"]), "per_config": per_config, **per_config_flat},
        "clocks": m["clocks"],
        "e2e": m["e2e"],
        "gpu_launches": int(m["launches"]),
        "roofline": m["roofline"],
        "roofline_fp64": roofline_fp64,
        "fp64_rates": {"dfma_per_s_8_chains": fp64_peak, "dfma_per_s_1_chain": fp64_dep},
        "extras": extras,
        "cpu_baseline": cpu,
    }
    print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
