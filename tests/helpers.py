"""Shared test helpers: build the oracle (and, in GPU tests, the CUDA context) from one Workload."""
from __future__ import annotations

import numpy as np

import asd_inputs as ai
from oracle import asd_oracle as orc


def oracle_spec(w: ai.Workload, **over) -> orc.LatticeSpec:
    d = dict(lattice=w.lattice, nx=w.nx, ny=w.ny, nz=w.nz, pbc=w.pbc, mu_s=w.mu_s, lam=w.lam, gamma=w.gamma,
             dt=w.dt, J=w.J, track_nx=w.track_nx, x0=w.x0, grain_map=w.grain_map,
             grain_ku=w.grain_ku.astype(np.float64), grain_axis=w.grain_axis.astype(np.float64),
             macro=w.macro, seed=w.seed)
    d.update(over)
    return orc.LatticeSpec(**d)


def oracle_from_workload(w: ai.Workload, **over) -> orc.Oracle:
    o = orc.Oracle(oracle_spec(w, **over))
    o.set_spins(w.sx, w.sy, w.sz)
    o.set_fields(w.T, w.Bx, w.By, w.Bz)
    return o


def single_grain_spec(lattice, nx, ny, nz, pbc=(0, 0, 0), ku=0.0, axis=(0.0, 0.0, 1.0), **kw) -> orc.LatticeSpec:
    return orc.LatticeSpec(lattice=lattice, nx=nx, ny=ny, nz=nz, pbc=pbc,
                           grain_map=np.zeros((kw.get("track_nx", nx) or nx, ny), dtype=np.int32),
                           grain_ku=np.array([ku]), grain_axis=np.array([axis], dtype=np.float64), **kw)
