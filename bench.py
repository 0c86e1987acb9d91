#!/usr/bin/env python
"""bench.py -- spin-updates/s of the ASD hot path on B200 (BASELINE.json metric), one JSON line on stdout.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 4] [--heun-per-step 50]

A "step" is one pass of the whole hot path over one batch: `heun_per_step` stochastic Heun steps (2 fused kernels
each) of the synthetic HAMR window, the head-field scale of the drive schedule, and asd_shift_window whenever the
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


def _traffic(workload: str):
    """dram bytes per launch of the stage kernel from the committed ncu capture (profiles/traffic.csv), or None."""
    p = os.path.join(ROOT, "profiles", "traffic.csv")
    if not os.path.exists(p):
        return None
    vals = []
    for line in open(p):
        f = [x.strip() for x in line.split(",")]
        if len(f) >= 3 and f[0] == workload and f[1].startswith("heun_stage"):
            try:
                vals.append(float(f[2]))
            except ValueError:
                pass
    return float(np.mean(vals)) if vals else None


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


def _drive(w: ai.Workload, heun_per_step: int):
    """Per bench step: (field scale, planes to shift after the step or 0).  DESIGN.md Q8 schedule."""
    bits = ai.nrz_bits(64, w.bit_seed)
    state = {"heun": 0, "q": 0}

    def next_step():
        s = ai.field_scale_at(state["heun"], bits, w.bit_steps) if w.bit_steps else 1.0
        state["heun"] += heun_per_step
        p = 0
        if w.shift_every and state["heun"] // w.shift_every > state["q"]:
            state["q"] += 1
            p = ai.planes_for_shift(state["q"], w.spacing_nm[0])
        return s, p
    return next_step


# ------------------------------------------------------------------------------------------------------------
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

    w = _workload(args.config, seed_offset=rank)
    N = w.n_sites
    ell = None
    if args.ell:
        # the same exchange bonds handed over as a general ELL table (per-pair J); such a table cannot follow the
        # window, so this variant runs without shifts
        ell = ai.shell_ell_table(w)
        w.shift_every = 0
    ell_w = 0 if ell is None else int(ell[0].shape[1])
    ctx = asd.Context(_gpu_desc(asd, w, ell), device=f"cuda:{local}")
    dev = ctx.device
    if args.demag:
        ctx.enable_demag([a * 1e-9 for a in w.spacing_nm])
        ctx.set_demag_every(args.demag_every)
    if args.kernel != "auto":
        ctx.set_kernel({"general": asd.KERNEL_GENERAL, "fast": asd.KERNEL_FAST, "tma": asd.KERNEL_TMA,
                        "fused": asd.KERNEL_FUSED}[args.kernel])
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).pin_memory()
    hT, hBx, hBy, hBz = pin(w.T), pin(w.Bx), pin(w.By), pin(w.Bz)
    ctx.set_spins_host(pin(w.sx), pin(w.sy), pin(w.sz))
    ctx.set_fields_host(hT, hBx, hBy, hBz)
    torch.cuda.synchronize()
    hps = args.heun_per_step
    nxt = _drive(w, hps)

    def one_step(timed_heun=None):
        s, p = nxt()
        ctx.set_field_scale(s)
        if timed_heun is not None:
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            lc = ctx.launch_count()
            e0.record(); ctx.step_heun(hps); e1.record()
            timed_heun.append((e0, e1, ctx.launch_count() - lc))
        else:
            ctx.step_heun(hps)
        if p:
            ctx.shift_window(p)
        return p

    for _ in range(args.warmup):
        one_step()
    barrier()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    l0 = ctx.launch_count()
    heun_events, shifts = [], 0
    t0, t1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    t0.record()
    for _ in range(args.steps):
        shifts += 1 if one_step(heun_events) else 0
    t1.record()
    barrier()
    ms = t0.elapsed_time(t1)
    clocks = sampler.stop() if rank == 0 else None
    launches = ctx.launch_count() - l0
    heun_ms = sum(a.elapsed_time(b) for a, b, _ in heun_events)
    ms, updates = reduce_over_ranks(ms, float(args.steps) * hps * N, dist, dev)
    value = updates / (ms * 1e-3)

    # ---- e2e: the same steps through the C ABI with HOST buffers: H2D of the step's inputs, D2H of its result ----
    e2e_steps = max(1, min(args.steps, args.e2e_steps))
    barrier()
    w0 = time.perf_counter()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    msum = 0.0
    # double-buffered upload (asd_stage_fields_host / asd_commit_fields): the H2D copy of step n+1's fields runs on the
    # library's copy stream while step n's kernels run; every step still uploads its own 16 B/site and reads its result
    ctx.stage_fields_host(hT, hBx, hBy, hBz)
    for it in range(e2e_steps):
        s, p = nxt()
        ctx.commit_fields()                              # wait for the staged copy, repack: fields of this step
        ctx.set_field_scale(s)
        ctx.step_heun(hps)
        if p:
            ctx.shift_window(p)
        if it + 1 < e2e_steps:
            ctx.stage_fields_host(hT, hBx, hBy, hBz)     # pinned host -> device, 16 B/site, for the next step
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
    n_stage_launches = sum(n for _, _, n in heun_events)
    fused = n_stage_launches == hps * len(heun_events)       # one kernel per Heun step
    avg_launch_s = heun_ms * 1e-3 / n_stage_launches
    # a general ELL table adds its own compulsory bytes: int32 index + fp32 J per slot per site per stage
    alg_bytes = (40.0 if fused else BYTES_PER_SITE_PER_STAGE + 8.0 * ell_w) * N
    achieved = alg_bytes / avg_launch_s / 1e9
    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32", "data": "synthetic",
        "config": {"workload": w.name, "sites": N, "heun_steps_per_step": hps, "shifts_in_timed_region": shifts,
                   "shift_every_heun_steps": w.shift_every, "dt": w.dt, "parallelism": f"replicas x{world}", "ell_width": ell_w, "demag": bool(args.demag), "demag_every": args.demag_every if args.demag else None,
                   "l2": "working set (13 fp32 arrays/site = %.0f MB) exceeds the 126 MB L2" % (13 * 4 * N / 1e6)},
        "clocks": clocks, "gpu_launches": int(launches),
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": 16 * N, "d2h_bytes_per_step": 32,
                "steps": e2e_steps, "ms_per_step": e2e_ms / e2e_steps, "wall_ms_per_step": wall_ms / e2e_steps},
        "roofline": {"bound": "hbm", "kernel": ("heun_stage_general<ELL> (predictor+corrector, %d B/site each)" % (52 + 8 * ell_w)) if ell_w else
                     ("heun_fused (one kernel per Heun step, 40 B/site)" if fused else
                      "heun_stage_fast (predictor+corrector, 52 B/site each)"),
                     "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                     "peak_source": peak_src, "avg_launch_us": avg_launch_s * 1e6,
                     "algorithmic_bytes_per_launch": alg_bytes, "traffic": _traffic(w.name)},
    }
    if world == 1 and not args.no_cpu_baseline:
        out["cpu_baseline"] = cpu_baseline(args.config, budget_s=args.cpu_budget)
    print(json.dumps(out), flush=True)
    if dist is not None:
        dist.destroy_process_group()


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
    """The oracle as it stands, on this host's cores, on a bounded sample: full lattice, as many Heun steps as fit."""
    from oracle import asd_oracle as orc
    w = _workload(cfg)
    o = _oracle_for(w)
    t = time.perf_counter(); o.step_heun(1); t1 = time.perf_counter() - t
    n = int(max(1, min(200, budget_s / max(t1, 1e-3))))
    t = time.perf_counter(); o.step_heun(n); dt = time.perf_counter() - t
    return {"value": n * w.n_sites / dt, "unit": UNIT, "cores": orc.max_threads(), "kind": "oracle",
            "sample": f"{n} Heun steps of the full {w.name} lattice ({w.n_sites} sites), fp64, OpenMP"}


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
    ap.add_argument("--ell", action="store_true",
                    help="hand the exchange bonds over as a general ELL neighbour table with per-pair J (no window shifts)")
    ap.add_argument("--demag", action="store_true",
                    help="switch the demagnetising field on (Eq. (6)-(7): coarse-graining + FFT convolution per stage)")
    ap.add_argument("--demag-every", type=int, default=0,
                    help="0: demag field recomputed in every Heun stage; P >= 1: every P-th step, held in between")
    ap.add_argument("--kernel", default="auto", choices=["auto", "general", "fast", "tma", "fused"],
                    help="stage-kernel variant (asd_set_kernel); auto = the library's choice")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
