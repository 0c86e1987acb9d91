"""Writing a bit sequence with the multiscale window on the GPU, next to the fully atomistic window (the comparison of
the paper's Fig. 3 and P:120 in miniature).

    python -m paper_2502_02236_b200.multiscale_write [--lattice sc|l10] [--bits 8] [--mesh-cells 24] [--every 20]

Two runs over the same granular track, bit pattern, laser spot, head field and schedule (the window moves by one 2.1 nm
macrocell at a time at 1 nm per 5000 Heun steps):
  "multiscale"  [micromagnetic LLG mesh | atomistic mesh | micromagnetic LLG mesh] (asd_mm_enable)
  "atomistic"   the same atomistic mesh alone (open ends)
Each ends with asd_track_end_pass and is read back with asd_track_read_scan at the bit centres.  Prints one JSON record:
pattern, read-back per bit of both runs, bits with the wrong sign, the largest difference between the two read-backs and
the throughput of each run.  Everything runs through the C ABI; there is no CPU path.
"""
from __future__ import annotations

import argparse
import json
import time

import numpy as np

import asd_inputs as ai
from . import binding as asd


def _one(mw: ai.MultiscaleWrite, with_meshes: bool, cells, device: str) -> dict:
    import torch
    w = mw.ms.w
    ctx = asd.context_from_workload(w, device=device)
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    steps = ai.drive_multiscale_write(ctx, mw, cells=cells, with_meshes=with_meshes)
    c = mw.bit_centres()
    step = float(c[1] - c[0]) if len(c) > 1 else 1.0
    scan = ctx.track_read_scan(mw.track_y, mw.reader_sigma[0], mw.reader_sigma[1], float(c[0]), step, len(c))   # synchronises
    dt = time.perf_counter() - t0
    rec = {"heun_steps": steps, "seconds": dt, "spin_updates_per_s": steps * w.n_sites / dt,
           "gpu_launches": ctx.launch_count(), "read_back": np.round(scan, 4).tolist()}
    ctx.destroy()
    return rec


def run(lattice: int = ai.SC, n_bits: int = 8, mesh_cells: int = 24, every: int = 20, nz: int = 27, cells=None,
        device: str = "cuda:0") -> dict:
    mw = ai.multiscale_write(lattice, n_bits=n_bits, mesh_cells=(mesh_cells, mesh_cells), every=every, nz=nz)
    w = mw.ms.w
    cells = mw.cells_per_pass() if cells is None else cells
    sw = mw.swept_bits(cells)
    rec = {"workload": w.name, "atomistic_sites": w.n_sites, "mesh_cells": [mesh_cells, mesh_cells],
           "mesh_step_every_heun_steps": every, "track_planes": w.track_nx, "bit_cells": mw.bit_cells,
           "cells_per_pass": cells, "heun_steps_per_cell": mw.steps_per_cell, "pattern": mw.bits.astype(int).tolist(),
           "bits_swept": sw.tolist()}
    rec["multiscale"] = _one(mw, True, cells, device)
    rec["atomistic"] = _one(mw, False, cells, device)
    a = np.asarray(rec["multiscale"]["read_back"])[sw]
    b = np.asarray(rec["atomistic"]["read_back"])[sw]
    rec["bit_errors"] = {"multiscale": int(np.sum(np.sign(a) != mw.bits[sw])), "atomistic": int(np.sum(np.sign(b) != mw.bits[sw])),
                         "of": int(len(sw))}
    rec["max_read_back_difference"] = float(np.abs(a - b).max()) if len(sw) else None
    return rec


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--lattice", choices=["sc", "l10"], default="sc")
    ap.add_argument("--bits", type=int, default=8)
    ap.add_argument("--mesh-cells", type=int, default=24)
    ap.add_argument("--every", type=int, default=20)
    ap.add_argument("--nz", type=int, default=27)
    ap.add_argument("--cells", type=int, default=None, help="cells to travel (default: the whole track)")
    a = ap.parse_args()
    print(json.dumps(run(ai.SC if a.lattice == "sc" else ai.L10, a.bits, a.mesh_cells, a.every, a.nz, a.cells)))


if __name__ == "__main__":
    main()
