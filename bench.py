#!/usr/bin/env python
"""bench.py -- spin-updates/s of the ASD hot path on B200 (BASELINE.json metric), one JSON line on stdout.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 4] [--heun-per-step 50]

A "step" is one pass of the whole hot path over one batch: `heun_per_step` stochastic Heun steps (one fused kernel
each on HBM-streaming films, a predictor and a corrector kernel otherwise) of the synthetic HAMR window, the head-field scale of the drive schedule, and asd_shift_window whenever the
Heun-step counter crosses the shift cadence (every 5000 Heun steps, Q8).  Default workload: BASELINE
configs[4], the 881x220x27 L1_0 window (5.23 M sites) -- the configuration the metric's roofline target is quoted on.

N > 1 (torchrun): independent replica windows, one per GPU, no data-path collective ("replicas only", DESIGN.md
sec. 9); value = all ranks' site updates / max-over-ranks device time.
--impl reference: the fp64 CPU oracle as it stands, timed on the host cores on a bounded sample of the same workload.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import asd_inputs as ai  # noqa: E402

METRIC = "atomistic spin-updates/sec (Heun steps x spins)"
UNIT = "spin-updates/s"
# Algorithmic HBM bytes per lattice site per stage kernel: predictor reads S 12 + sigma 4 + B 12,
# writes S~ 12 + A 12; corrector reads S~ 12 + A 12 + sigma 4 + B 12, writes S 12.  Column/grain tables are cached.
BYTES_PER_SITE_PER_STAGE = 52.0


def _peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md)"


class ClockSampler:
    """Samples nvidia-smi SM clocks and throttle reasons during the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.rows, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append(line.strip())

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            f = [x.strip() for x in r.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1]))
                try:
                    pw.append(float(f[2]))
                except ValueError:
                    pass
            except ValueError:
                continue
            for n, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm), "power_w": float(np.median(pw)) if pw else None}


def _workload(cfg: int, seed_offset: int = 0) -> ai.Workload:
    w = ai.make_config(cfg)
    w.seed += seed_offset
    return w


def reduce_over_ranks(ms_local: float, updates_local: float, dist=None, device="cpu"):
    """Whole-job figures from per-rank ones: time = MAX over ranks, work = SUM over ranks (replicas, DESIGN.md
    sec. 9).  `dist` is torch.distributed (any backend) or None for a single process."""
    if dist is None:
        return ms_local, updates_local
    import torch
    t = torch.tensor([ms_local], device=device, dtype=torch.float64)
    u = torch.tensor([updates_local], device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(t.item()), float(u.item())


def _gpu_desc(asd, w: ai.Workload, ell=None):
    """Workload -> asd.LatticeDesc (argument marshalling; the product path never imports oracle/ or tests/)."""
    extra = {} if ell is None else {"ell_idx": ell[0], "ell_J": ell[1]}
    return asd.desc_from_workload(w, **extra)


def _drive(w: ai.Workload, heun_per_step: int, start_heun: int = 0):
    """Per bench step: (field scale, planes to shift after the step or 0).  DESIGN.md Q8 schedule.  start_heun: where
    on the schedule's step-index clock the run begins (bench.py starts shortly before a shift so that the window shift
    falls inside the timed region whatever --steps is)."""
    bits = ai.nrz_bits(64, w.bit_seed)
    state = {"heun": start_heun, "q": (start_heun // w.shift_every) if w.shift_every else 0}

    def next_step():
        s = ai.field_scale_at(state["heun"], bits, w.bit_steps) if w.bit_steps else 1.0
        state["heun"] += heun_per_step
        p = 0
        if w.shift_every and state["heun"] // w.shift_every > state["q"]:
            state["q"] += 1
            p = ai.planes_for_shift(state["q"], w.spacing_nm[0])
        return s, p
    return next_step


def _start_heun(w: ai.Workload, hps: int, warmup: int, steps: int) -> int:
    """Schedule position at which the first warm-up step starts so that a shift closes the middle timed step."""
    if not w.shift_every:
        return 0
    per = max(1, w.shift_every // hps)                      # bench steps per shift period
    return (per - (warmup + max(1, (steps + 1) // 2)) % per) % per * hps


# Algorithmic HBM bytes.  Survey floors: two-kernel step, k1 recomputed / structured.
SURVEY_FLOOR_BYTES = {ai.SC: 92.0, ai.L10: 96.0}
FUSED_BYTES_PER_SITE_STEP = 40.0
# Plain-ALU roof: one warp instruction per scheduler per clock.
SM_COUNT, SCHEDULERS_PER_SM, LANES = 148, 4, 32
# Arithmetic a fused Heun step needs per site, thread instructions (DESIGN.md sec. 6 derivation) by lattice
ALG_INST_PER_SITE_STEP = {ai.SC: 196.0, ai.L10: 222.0}


def _sm_max_hz():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        return float(json.load(open(p)).get("sm_max_mhz", 1965.0)) * 1e6
    return 1965e6


def _captured(workload: str, kernel_prefix: str):
    """(dram bytes per launch, executed warp instructions per launch) of a kernel from the committed ncu capture
    (profiles/traffic.csv), or (None, None)."""
    p = os.path.join(ROOT, "profiles", "traffic.csv")
    if not os.path.exists(p):
        return None, None
    tr, wi = [], []
    for line in open(p):
        f = [x.strip() for x in line.split(",")]
        if len(f) >= 3 and f[0] == workload and f[1].startswith(kernel_prefix):
            try:
                tr.append(float(f[2]))
                if len(f) >= 4 and f[3]:
                    wi.append(float(f[3]))
            except ValueError:
                pass
    return (float(np.mean(tr)) if tr else None), (float(np.mean(wi)) if wi else None)


class Run:
    """One context on one workload: warm-up, device-timed bench steps (Heun batches + the schedule's shifts)."""

    def __init__(self, asd, torch, w, device, hps, kernel="auto", ell=False, demag=False, demag_every=0, multiscale=None,
                 track_stray=False, track_exchange=False):
        self.asd, self.torch, self.w, self.hps = asd, torch, w, hps
        self.N = w.n_sites
        self.demag, self.demag_every, self.multiscale = demag, demag_every, (multiscale is not None)
        table = None
        if ell:
            # the same exchange bonds handed over as a general ELL table (per-pair J); such a table cannot follow the
            # window, so this variant runs without shifts
            table = ai.shell_ell_table(w)
            w.shift_every = 0
        self.ell_w = 0 if table is None else int(table[0].shape[1])
        self.ctx = asd.Context(_gpu_desc(asd, w, table), device=device)
        if demag:
            self.ctx.enable_demag([a * 1e-9 for a in w.spacing_nm])
            self.ctx.set_demag_every(demag_every)
            if track_stray:                              # + the frozen track's stray field, recomputed at every shift
                self.ctx.enable_track_stray(True, 0)
        if track_exchange:                           # window ends exchange coupled to the frozen track (reading E1)
            self.ctx.enable_track_exchange(True)
        if multiscale is not None:                   # micromagnetic meshes either side
            ai.apply_multiscale(self.ctx, multiscale)
        if kernel != "auto":
            self.ctx.set_kernel({"general": asd.KERNEL_GENERAL, "fast": asd.KERNEL_FAST, "tma": asd.KERNEL_TMA,
                                 "fused": asd.KERNEL_FUSED, "persistent": asd.KERNEL_PERSISTENT}[kernel])
        pin = lambda a: torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).pin_memory()
        self.hT, self.hBx, self.hBy, self.hBz = pin(w.T), pin(w.Bx), pin(w.By), pin(w.Bz)
        self.ctx.set_spins_host(pin(w.sx), pin(w.sy), pin(w.sz))
        self.ctx.set_fields_host(self.hT, self.hBx, self.hBy, self.hBz)
        torch.cuda.synchronize()
        self.nxt = None

    def start(self, warmup, steps):
        self.nxt = _drive(self.w, self.hps, _start_heun(self.w, self.hps, warmup, steps))
        for _ in range(warmup):
            self.one_step()

    def one_step(self, timed=None):
        torch, ctx = self.torch, self.ctx
        s, p = self.nxt()
        ctx.set_field_scale(s)
        if timed is not None:
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            lc = ctx.launch_count()
            e0.record(); ctx.step_heun(self.hps); e1.record()
            timed.append((e0, e1, ctx.launch_count() - lc))
        else:
            ctx.step_heun(self.hps)
        if p:
            ctx.shift_window(p)
        return p

    def timed(self, steps, barrier=None):
        """-> dict(ms, shifts, launches, heun_ms, heun_launches): CUDA events around the whole region and each batch."""
        torch = self.torch
        sync = barrier or torch.cuda.synchronize
        ev, shifts = [], 0
        l0 = self.ctx.launch_count()
        t0, t1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        sync()
        t0.record()
        for _ in range(steps):
            shifts += 1 if self.one_step(ev) else 0
        t1.record()
        sync()
        return {"ms": t0.elapsed_time(t1), "shifts": shifts, "launches": self.ctx.launch_count() - l0,
                "heun_ms": sum(a.elapsed_time(b) for a, b, _ in ev), "heun_launches": sum(n for _, _, n in ev),
                "steps": steps}

    def roofline(self, t, peak, peak_src):
        """The dominant kernel's roofline record from a timed() result."""
        hps, N, w = self.hps, self.N, self.w
        heun_steps = hps * t["steps"]
        per_step = t["heun_launches"] / max(1, heun_steps)            # kernels per Heun step: 1 fused, 2 stage kernels
        persistent = per_step < 0.5                                     # all Heun steps of a batch in one cluster launch
        fused = per_step < 1.5 and self.ell_w == 0 and not persistent
        avg_launch_s = t["heun_ms"] * 1e-3 / max(1, t["heun_launches"])
        if persistent:
            name = "heun_persistent (%d Heun steps per launch, lattice resident in distributed shared memory)" % hps
            alg, cap = 40.0 * N, "heun_persistent"                      # HBM bytes per LAUNCH: in and out once
        elif fused:
            name, alg = "heun_fused (one kernel per Heun step, 40 B/site)", FUSED_BYTES_PER_SITE_STEP * N
            cap = "heun_fused"
        elif self.ell_w:
            name = "heun_stage_ell (predictor + corrector, %d B/site each)" % (52 + 8 * self.ell_w)
            alg, cap = (BYTES_PER_SITE_PER_STAGE + 8.0 * self.ell_w) * N, "heun_stage_ell"
        else:
            name, alg = "stage kernels (predictor + corrector, 52 B/site each)", BYTES_PER_SITE_PER_STAGE * N
            cap = "heun_stage_fast"
        achieved = alg / avg_launch_s / 1e9
        step_s = t["heun_ms"] * 1e-3 / max(1, heun_steps)
        traffic, warp_inst = _captured(w.name, cap)
        r = {"bound": "hbm", "kernel": name, "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
             "peak_source": peak_src, "avg_launch_us": avg_launch_s * 1e6, "algorithmic_bytes_per_launch": alg,
             "traffic": traffic,
             # the same Heun steps accounted at SURVEY 8(d)'s two-kernel floor (92 B SC / 96 B L1_0 per site-step):
             # comparable across kernel designs and rounds
             "frac_survey_floor": SURVEY_FLOOR_BYTES[w.lattice] * N / step_s / 1e9 / peak if not self.ell_w else None,
             # DRAM bytes the committed ncu capture counted for this kernel / this run's launch time
             "frac_dram": (traffic / avg_launch_s / 1e9 / peak) if traffic else None}
        if self.demag or self.multiscale:
            # the launches of a Heun step include the field pipeline's (mesh kernels'): the events around a batch cannot
            # time the Heun kernel alone, so the record is the WHOLE step at the Heun kernels' algorithmic bytes -- a lower
            # bound on their own fraction; per-kernel times: profiles/r2_demag.md, r2_multiscale.md
            refreshes = (2.0 if self.demag_every < 1 else 1.0 / self.demag_every) if self.demag else 0.0   # 3 launches each
            one_kernel = (per_step - 3.0 * refreshes) < (1.9 if self.multiscale else 1.5)
            alg = (FUSED_BYTES_PER_SITE_STEP if one_kernel else 2 * BYTES_PER_SITE_PER_STAGE) * N
            extra = "demagnetising-field pipeline" if self.demag else "mesh kernels"
            r.update(kernel=("heun_fused, one kernel per Heun step (40 B/site)" if one_kernel else
                             "stage kernels (predictor + corrector, 52 B/site each)") + " + " + extra +
                            " (%.2f launches per Heun step)" % per_step,
                     achieved=alg / step_s / 1e9, frac=alg / step_s / 1e9 / peak, avg_launch_us=None,
                     algorithmic_bytes_per_launch=alg, traffic=None, frac_dram=None,
                     note="whole Heun step incl. the %s, at the Heun kernels' algorithmic bytes per step" % extra)
            return r
        if fused:
            issue_peak = SM_COUNT * SCHEDULERS_PER_SM * LANES * _sm_max_hz()
            alg_inst = ALG_INST_PER_SITE_STEP[w.lattice] * N
            r["alu"] = {"bound": "alu", "unit": "thread-instructions/s", "peak": issue_peak,
                        "peak_source": "148 SMs x 4 schedulers x 32 lanes x sm_max clock (one warp instruction per scheduler per clock)",
                        "achieved": alg_inst / avg_launch_s, "frac": alg_inst / avg_launch_s / issue_peak,
                        "algorithmic_thread_inst_per_site_step": ALG_INST_PER_SITE_STEP[w.lattice],
                        "frac_executed": (warp_inst * LANES / avg_launch_s / issue_peak) if warp_inst else None}
            r["note"] = ("the fused step moves 2.6x fewer bytes than the two-kernel step and is no longer HBM-bound: it is held "
                         "by instruction issue / latency at 16 warps per SM (shared memory and registers are both full); "
                         "frac = its own 40 B/site-step against the HBM peak, frac_survey_floor = the same steps at the "
                         "two-kernel floor, alu.frac = arithmetic needed / issue peak")
        return r


def run_ours(args):
    import torch
    import paper_2502_02236_b200 as asd

    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; libasd has no CPU fallback")
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    device = f"cuda:{local}"
    msw = None
    if args.multiscale:
        # [48-cell LLG mesh | atomistic mesh | 48-cell mesh] on the film of config 3 (SC) or 4 (L1_0); no shifts (a
        # multiscale window moves by whole 2 nm cells, not by the 1 nm of the configs' schedule)
        msw = ai.multiscale_film(ai.L10 if args.config == 4 else ai.SC, every=args.mm_every, seed=1 + rank)
        w = msw.w
    else:
        w = _workload(args.config, seed_offset=rank)
    N = w.n_sites
    hps = args.heun_per_step
    run = Run(asd, torch, w, device, hps, kernel=args.kernel, ell=args.ell, demag=args.demag, demag_every=args.demag_every,
              multiscale=msw, track_stray=args.track_stray, track_exchange=args.track_exchange)
    ctx, dev = run.ctx, run.ctx.device
    run.start(args.warmup, args.steps)
    barrier()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    t = run.timed(args.steps, barrier)
    clocks = sampler.stop() if rank == 0 else None
    ms, updates = reduce_over_ranks(t["ms"], float(args.steps) * hps * N, dist, dev)
    value = updates / (ms * 1e-3)

    # ---- e2e: the same steps through the C ABI with HOST buffers: H2D of the step's inputs, D2H of its result ----
    e2e_steps = max(1, min(args.steps, args.e2e_steps))
    nxt = run.nxt
    barrier()
    w0 = time.perf_counter()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    msum = 0.0
    # double-buffered upload (asd_stage_fields_host / asd_commit_fields): the H2D copy of step n+1's fields runs on the
    # library's copy stream while step n's kernels run; every step still uploads its own 16 B/site and reads its result
    ctx.stage_fields_host(run.hT, run.hBx, run.hBy, run.hBz)
    for it in range(e2e_steps):
        s, p = nxt()
        ctx.commit_fields()                              # wait for the staged copy, repack: fields of this step
        ctx.set_field_scale(s)
        ctx.step_heun(hps)
        if p:
            ctx.shift_window(p)
        if it + 1 < e2e_steps:
            ctx.stage_fields_host(run.hT, run.hBx, run.hBy, run.hBz)     # pinned host -> device, 16 B/site, for the next step
        m, _n = ctx.magnetisation()                      # device -> host, synchronises
        msum += float(m[2])
    e1.record()
    barrier()
    e2e_ms = e0.elapsed_time(e1)
    wall_ms = (time.perf_counter() - w0) * 1e3
    e2e_ms, e2e_updates = reduce_over_ranks(e2e_ms, float(e2e_steps) * hps * N, dist, dev)
    e2e_value = e2e_updates / (e2e_ms * 1e-3)

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return
    peak, peak_src = _peaks()
    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32", "data": "synthetic",
        "config": {"workload": w.name, "sites": N, "heun_steps_per_step": hps, "shifts_in_timed_region": t["shifts"],
                   "shift_every_heun_steps": w.shift_every, "dt": w.dt, "parallelism": f"replicas x{world}",
                   "ell_width": run.ell_w, "demag": bool(args.demag), "demag_every": args.demag_every if args.demag else None,
                   "track_stray": bool(args.demag and args.track_stray), "track_exchange": bool(args.track_exchange),
                   "kernel": args.kernel, "multiscale": ({"mesh_cells": list(msw.mcx), "every": msw.every} if msw else None),
                   "l2": "working set (13 fp32 arrays/site = %.0f MB) exceeds the 126 MB L2" % (13 * 4 * N / 1e6)},
        "clocks": clocks, "gpu_launches": int(t["launches"]),
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": 16 * N, "d2h_bytes_per_step": 32,
                "steps": e2e_steps, "ms_per_step": e2e_ms / e2e_steps, "wall_ms_per_step": wall_ms / e2e_steps,
                "note": "per step: 16 B/site of fields up (pinned host, double-buffered), the window magnetisation (32 B) "
                        "down; the spin state stays resident on the device and is not copied back"},
        "roofline": run.roofline(t, peak, peak_src),
    }
    if world == 1 and not args.no_sustained:
        out["sustained"] = sustained(run, args.sustained_seconds, ms / args.steps, local, peak, peak_src)
    if world == 1 and not args.no_secondary:
        del run, ctx
        torch.cuda.empty_cache()
        out["secondary"] = secondary(asd, torch, device, args, peak, peak_src)
    if world == 1 and not args.no_cpu_baseline:
        out["cpu_baseline"] = cpu_baseline(args.config, budget_s=args.cpu_budget)
    print(json.dumps(out), flush=True)
    if dist is not None:
        dist.destroy_process_group()


def sustained(run, seconds, ms_per_step, gpu_index, peak, peak_src):
    """>= `seconds` of back-to-back bench steps (the regime BASELINE cfg4's 1e5 steps live in: the board reaches its power
    cap), with its own clock record."""
    steps = int(max(10, np.ceil(seconds * 1e3 / max(ms_per_step, 1e-3))))
    sampler = ClockSampler(gpu_index)
    sampler.start()
    t = run.timed(steps)
    clocks = sampler.stop()
    r = run.roofline(t, peak, peak_src)
    value = float(steps) * run.hps * run.N / (t["ms"] * 1e-3)
    # energy per site update from the median board power over the run (20 samples in 2 s): under a power cap this, not
    # bytes or instructions, is what binds
    nj = (clocks["power_w"] / value * 1e9) if clocks.get("power_w") else None
    return {"value": value, "unit": UNIT, "steps": steps,
            "seconds": t["ms"] * 1e-3, "ms_per_step": t["ms"] / steps, "shifts_in_timed_region": t["shifts"],
            "clocks": clocks, "nj_per_spin_update": nj, "avg_launch_us": r["avg_launch_us"], "frac": r["frac"],
            "frac_survey_floor": r["frac_survey_floor"]}


def secondary(asd, torch, device, args, peak, peak_src):
    """Short runs of the other kernels / configs, each with its own roofline fraction (same timing rules, 6 timed steps of
    20 Heun steps after 3 warm-up steps; working sets > L2 except where noted)."""
    out = []
    w4 = None

    def one(label, cfg, **kw):
        nonlocal w4
        hps, steps, warm = kw.pop("hps", 20), kw.pop("steps", 6), 3
        try:
            if cfg == 4:
                w4 = w4 or _workload(4)
                import copy
                w = copy.copy(w4)
            elif cfg == "two_track":
                # the 80 nm wide two-track window: SC 400 x 268 x 27, spot on the bottom track
                w = ai.two_track_film(ai.SC, n_bits=4).w
            elif cfg == "multiscale":
                # [48-cell mesh | 336 x 200 x 27 SC atoms | 48-cell mesh]: the paper's three equal parts on cfg3's film
                kw["multiscale"] = ai.multiscale_film(ai.SC, every=kw.pop("every", 20))
                w = kw["multiscale"].w
            else:
                w = _workload(cfg)
            run = Run(asd, torch, w, device, hps, **kw)
            run.start(warm, steps)
            t = run.timed(steps)
            r = run.roofline(t, peak, peak_src)
            heun_steps = hps * steps
            rec = {"label": label, "workload": w.name, "sites": w.n_sites, "value": heun_steps * w.n_sites / (t["ms"] * 1e-3),
                   "unit": UNIT, "us_per_heun_step": t["heun_ms"] * 1e3 / heun_steps, "kernel": r["kernel"],
                   "avg_launch_us": r["avg_launch_us"], "frac": r["frac"], "frac_survey_floor": r["frac_survey_floor"],
                   "shifts_in_timed_region": t["shifts"]}
            if kw.get("multiscale") is not None or kw.get("demag"):
                rec.update(frac=None)      # the step includes other kernels: no single-kernel fraction to quote
            elif w.n_sites < (1 << 18):
                rec.update(frac=None, frac_survey_floor=None, note="launch-bound: no roofline fraction")
            elif 13 * 4 * w.n_sites < 126e6:
                rec["note"] = "working set fits the 126 MB L2: frac is not an HBM fraction"
            out.append(rec)
            del run
            torch.cuda.empty_cache()
        except Exception as e:                      # a secondary line must never cost the main one
            out.append({"label": label, "error": str(e)[:200]})

    one("cfg4, two-kernel film kernel (asd_set_kernel FAST)", 4, kernel="fast")
    one("cfg4 as a general ELL table, W = 10, per-pair J (no shifts)", 4, ell=True)
    one("cfg4 with the demagnetising field recomputed in every stage", 4, demag=True, demag_every=0)
    one("cfg4 with the demagnetising field recomputed once per Heun step and held for both stages (fused step)", 4,
        demag=True, demag_every=1)
    one("cfg4 with everything P:33 puts on the window: ends exchange coupled to the frozen track, demagnetising field "
        "once per Heun step, the track's stray field at every shift (fused step)", 4, demag=True, demag_every=1,
        track_stray=True, track_exchange=True)
    one("cfg3 SC 400x200x27", 3)
    one("cfg0 SC 16^3 periodic on the persistent cluster (us per Heun step is the figure)", 0, hps=1000, steps=3)
    one("cfg0 through CUDA-graph replay of the stage kernels (round 1's path)", 0, hps=1000, steps=3, kernel="general")
    one("multiscale window: 48-cell LLG mesh | SC 336x200x27 atoms | 48-cell mesh, mesh RK4 step every 20 Heun steps",
        "multiscale", every=20)
    one("multiscale window, meshes in lock-step (every Heun step)", "multiscale", every=1)
    one("two-track window SC 400x268x27 (pass 0 of the two-track write; profiles/r2_two_track.md has both passes)", "two_track")
    return out


# ------------------------------------------------------------------------------------------------------------
def _oracle_for(w: ai.Workload):
    from oracle import asd_oracle as orc
    return orc.from_workload(w)


def _crop(w: ai.Workload, nx: int) -> ai.Workload:
    """First nx planes of the window (same grains, fields, spins): a bounded sample of the same workload."""
    import copy
    c = copy.copy(w)
    plane = w.ny * w.nz
    c.nx = nx
    for name in ("T", "Bx", "By", "Bz", "sx", "sy", "sz"):
        setattr(c, name, getattr(w, name)[:nx * plane].copy())
    return c


def cpu_baseline(cfg: int, budget_s: float = 15.0):
    """The oracle as it stands, on this host's cores, on a bounded sample: the full lattice, as many Heun steps as fit
    in the budget with all threads; then the same lattice on ONE thread for a third of the budget."""
    from oracle import asd_oracle as orc
    w = _workload(cfg)
    o = _oracle_for(w)
    t = time.perf_counter(); o.step_heun(1); t1 = time.perf_counter() - t
    n = int(max(1, min(200, budget_s / max(t1, 1e-3))))
    t = time.perf_counter(); o.step_heun(n); dt = time.perf_counter() - t
    out = {"value": n * w.n_sites / dt, "unit": UNIT, "cores": orc.max_threads(), "kind": "oracle",
           "sample": f"{n} Heun steps of the full {w.name} lattice ({w.n_sites} sites), fp64, OpenMP"}
    # one thread: a crop of the first planes sized to ~budget/3 at the all-thread per-site rate x cores
    per_site_1 = dt / (n * w.n_sites) * orc.max_threads()
    nx1 = int(max(4, min(w.nx, (budget_s / 3.0) / (per_site_1 * w.ny * w.nz))))
    w1 = _crop(w, nx1)
    o1 = _oracle_for(w1)
    o1.set_threads(1)
    t = time.perf_counter(); o1.step_heun(1); d1 = time.perf_counter() - t
    out["single_thread"] = {"value": w1.n_sites / d1, "unit": UNIT, "cores": 1,
                            "sample": f"1 Heun step of the first {nx1} of {w.nx} planes ({w1.n_sites} sites), one thread"}
    return out


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from oracle import asd_oracle as orc
    w = _workload(args.config)
    # size the per-step sample so that (K + W) steps end within ~2 minutes: one Heun step of the first nx_s planes
    probe = _crop(w, min(w.nx, 32))
    o = _oracle_for(probe)
    o.step_heun(1)
    t = time.perf_counter(); o.step_heun(2); per_site = (time.perf_counter() - t) / (2 * probe.n_sites)
    budget = 120.0 / (args.steps + args.warmup)
    nx_s = int(max(4, min(w.nx, budget / (per_site * w.ny * w.nz))))
    ws = _crop(w, nx_s)
    o = _oracle_for(ws)
    for _ in range(args.warmup):
        o.step_heun(1)
    t = time.perf_counter()
    for _ in range(args.steps):
        o.step_heun(1)
    dt = time.perf_counter() - t
    value = args.steps * ws.n_sites / dt
    sample = (f"1 Heun step per bench step on the first {nx_s} of {w.nx} planes of {w.name} "
              f"({ws.n_sites} sites), fp64 oracle, OpenMP")
    out = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT,
           "n_gpus": int(os.environ.get("WORLD_SIZE", "1")), "steps": args.steps, "warmup": args.warmup,
           "ms_per_step": dt * 1e3 / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
           "dtype": "f64", "data": "synthetic", "config": {"workload": w.name, "sites": ws.n_sites},
           "cpu_baseline": {"value": value, "unit": UNIT, "cores": orc.max_threads(), "kind": "oracle", "sample": sample},
           "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
           "gpu_launches": 0}
    print(json.dumps(out), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=4)
    ap.add_argument("--heun-per-step", type=int, default=50)
    ap.add_argument("--e2e-steps", type=int, default=20)
    ap.add_argument("--cpu-budget", type=float, default=15.0)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-sustained", action="store_true", help="skip the >= 2 s back-to-back sub-record")
    ap.add_argument("--sustained-seconds", type=float, default=2.0)
    ap.add_argument("--no-secondary", action="store_true", help="skip the short runs of the other kernels / configs")
    ap.add_argument("--ell", action="store_true",
                    help="hand the exchange bonds over as a general ELL neighbour table with per-pair J (no window shifts)")
    ap.add_argument("--demag", action="store_true",
                    help="switch the demagnetising field on (Eq. (6)-(7): coarse-graining + FFT convolution per stage)")
    ap.add_argument("--demag-every", type=int, default=0,
                    help="0: demag field recomputed in every Heun stage; P >= 1: every P-th step, held in between")
    ap.add_argument("--track-stray", action="store_true",
                    help="with --demag: also the stray field of the frozen track (DESIGN.md sec. 12, reading D4)")
    ap.add_argument("--track-exchange", action="store_true",
                    help="window ends exchange coupled to the frozen track (DESIGN.md sec. 10, reading E1)")
    ap.add_argument("--multiscale", action="store_true",
                    help="the multiscale window: a micromagnetic LLG mesh either side of the atomistic mesh (DESIGN.md sec. 14)")
    ap.add_argument("--mm-every", type=int, default=20, help="Heun steps per RK4 step of the meshes")
    ap.add_argument("--kernel", default="auto", choices=["auto", "general", "fast", "tma", "fused", "persistent"],
                    help="stage-kernel variant (asd_set_kernel); auto = the library's choice")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
