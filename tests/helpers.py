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


# ---------------------------------------------------------------------------------------------
# CUDA side (GPU tests only): the same Workload through the C ABI binding.
# ---------------------------------------------------------------------------------------------
def gpu_desc(w: ai.Workload, **over):
    import paper_2502_02236_b200 as asd
    d = dict(lattice=w.lattice, nx=w.nx, ny=w.ny, nz=w.nz, pbc=w.pbc, mu_s=w.mu_s, lam=w.lam, gamma=w.gamma,
             dt=w.dt, J=w.J, track_nx=w.track_nx, x0=w.x0, grain_map=w.grain_map, n_grains=w.n_grains,
             grain_ku=w.grain_ku, grain_axis=w.grain_axis, macro=w.macro, seed=w.seed)
    d.update(over)
    return asd.LatticeDesc(**d)


def gpu_from_workload(w: ai.Workload, **over):
    import torch
    import paper_2502_02236_b200 as asd
    ctx = asd.Context(gpu_desc(w, **over))
    dev = ctx.device
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).to(dev)
    ctx.set_spins(t(w.sx), t(w.sy), t(w.sz))
    ctx.set_fields(t(w.T), t(w.Bx), t(w.By), t(w.Bz))
    torch.cuda.synchronize()
    return ctx


def max_abs_diff(ctx, o) -> float:
    return float(np.abs(ctx.get_spins_host().astype(np.float64) - o.get_spins()).max())
