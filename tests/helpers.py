"""Shared test helpers: build the oracle (and, in GPU tests, the CUDA context) from one Workload."""
from __future__ import annotations

import numpy as np

import asd_inputs as ai
from oracle import asd_oracle as orc


def oracle_spec(w: ai.Workload, **over) -> orc.LatticeSpec:
    return orc.spec_from_workload(w, **over)


def oracle_from_workload(w: ai.Workload, **over) -> orc.Oracle:
    return orc.from_workload(w, **over)


def single_grain_spec(lattice, nx, ny, nz, pbc=(0, 0, 0), ku=0.0, axis=(0.0, 0.0, 1.0), **kw) -> orc.LatticeSpec:
    return orc.LatticeSpec(lattice=lattice, nx=nx, ny=ny, nz=nz, pbc=pbc,
                           grain_map=np.zeros((kw.get("track_nx", nx) or nx, ny), dtype=np.int32),
                           grain_ku=np.array([ku]), grain_axis=np.array([axis], dtype=np.float64), **kw)


# ---------------------------------------------------------------------------------------------
# CUDA side (GPU tests only): the same Workload through the C ABI binding.
# ---------------------------------------------------------------------------------------------
def gpu_desc(w: ai.Workload, **over):
    import paper_2502_02236_b200 as asd
    return asd.desc_from_workload(w, **over)


def gpu_from_workload(w: ai.Workload, **over):
    import paper_2502_02236_b200 as asd
    return asd.context_from_workload(w, **over)


def max_abs_diff(ctx, o) -> float:
    return float(np.abs(ctx.get_spins_host().astype(np.float64) - o.get_spins()).max())
