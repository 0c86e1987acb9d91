"""Two parallel tracks written one after the other on the GPU (sec. III / Fig. 4; SURVEY.md 8(f)
item 4), read back with the Gaussian-footprint scan that stands in for the TMR head.

    python -m paper_2502_02236_b200.two_track [--lattice sc|l10] [--nz 27] [--bits 10] [--shift-every 5000] [--whole-window]

Pass 0 centres the laser spot on the bottom track and writes bit pattern A starting from a uniformly magnetised
track; pass 1 starts from the track pass 0 has written (asd_track_end_pass / asd_track_begin_pass), centres the spot on
the top track and writes pattern B.  Prints one JSON record: the patterns, the read-back value at the centre of every
bit the freezing point has swept, the number of bits read back with the wrong sign, how far pass 1 changed the bottom
track, and the throughput of the whole run (shifts, field uploads and scans included).  Everything runs through the C
ABI; there is no CPU path.
"""
from __future__ import annotations

import argparse
import json
import time

import numpy as np

import asd_inputs as ai
from . import binding as asd


def run(lattice: int = ai.SC, nz: int = 27, n_bits: int = 10, shift_every: int = 5000, length_nm: float = 120.0,
        width_nm: float = 80.0, periods=None, device: str = "cuda:0", whole_window: bool = False, demag_every: int = 1) -> dict:
    import torch
    tt = ai.two_track_film(lattice, length_nm=length_nm, width_nm=width_nm, nz=nz, n_bits=n_bits,
                           shift_every=shift_every)
    w = tt.w
    ctx = asd.context_from_workload(w, device=device)
    if whole_window:
        # everything P:33 puts on the window: its own demagnetising field (held, refreshed every demag_every Heun steps),
        # the frozen track's stray field (recomputed at every shift) and ends exchange coupled to the frozen track
        ctx.enable_demag([a * 1e-9 for a in w.spacing_nm])
        ctx.set_demag_every(demag_every)
        ctx.enable_track_stray(True, 0)
        ctx.enable_track_exchange(True)
    up = lambda sim, T: sim.set_fields_host(T=T)
    periods = tt.n_periods if periods is None else periods
    wb = tt.written_bits(periods)
    rec = {"workload": w.name, "window": ("P:33: demagnetising field every %d Heun steps + track stray field + coupled ends"
                                          % demag_every) if whole_window else "exchange, anisotropy, head field, thermal field",
           "sites": w.n_sites, "track_planes": w.track_nx, "bits_per_track": n_bits,
           "bit_planes": tt.bit_planes, "periods_per_pass": periods, "heun_steps_per_period": shift_every,
           "track_centres_sites": list(tt.track_y), "reader_sigma_sites": list(tt.reader_sigma),
           "bits_swept": wb.tolist(), "pattern": [b.astype(int).tolist() for b in tt.bits], "passes": []}
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    steps = 0
    reads = []
    for p in (0, 1):
        steps += ai.drive_pass(ctx, tt, p, up, periods=periods)
        r = ai.read_tracks(ctx, tt)                      # synchronises
        reads.append(r)
        rec["passes"].append({"pass": p, "spot_on_track": p, "read_back": np.round(r, 4).tolist()})
    dt = time.perf_counter() - t0
    rec["seconds"] = dt
    rec["spin_updates_per_s"] = steps * w.n_sites / dt
    rec["gpu_launches"] = ctx.launch_count()
    # figure of merit: sign of the read-back at the centre of every swept bit against the pattern written there
    err0 = int(np.sum(np.sign(reads[0][0][wb]) != tt.bits[0][wb]))
    err_bottom = int(np.sum(np.sign(reads[1][0][wb]) != tt.bits[0][wb]))
    err_top = int(np.sum(np.sign(reads[1][1][wb]) != tt.bits[1][wb]))
    rec["bit_errors"] = {"bottom_after_pass0": err0, "bottom_after_pass1": err_bottom, "top_after_pass1": err_top,
                         "of": int(len(wb))}
    rec["bottom_track_change_by_pass1"] = float(np.abs(reads[1][0][wb] - reads[0][0][wb]).max()) if len(wb) else None
    rec["top_track_before_pass1"] = np.round(reads[0][1][wb], 4).tolist()
    ctx.destroy()
    return rec


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--lattice", choices=["sc", "l10"], default="sc")
    ap.add_argument("--nz", type=int, default=27)
    ap.add_argument("--bits", type=int, default=10)
    ap.add_argument("--shift-every", type=int, default=5000)
    ap.add_argument("--length-nm", type=float, default=120.0)
    ap.add_argument("--width-nm", type=float, default=80.0)
    ap.add_argument("--periods", type=int, default=None)
    ap.add_argument("--whole-window", action="store_true",
                    help="with the window's demagnetising field, the frozen track's stray field and track-coupled ends (P:33)")
    ap.add_argument("--demag-every", type=int, default=1, help="with --whole-window: Heun steps per refresh of the held field")
    a = ap.parse_args()
    print(json.dumps(run(ai.SC if a.lattice == "sc" else ai.L10, a.nz, a.bits, a.shift_every, a.length_nm, a.width_nm,
                         a.periods, whole_window=a.whole_window, demag_every=a.demag_every)))


if __name__ == "__main__":
    main()
