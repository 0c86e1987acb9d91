"""Slab decomposition along x, host side: the index plan, and
the decomposition itself with the ORACLE as the ranks -- in one process and as a world_size-2 gloo job -- bit-identical to
the undivided window (the noise is keyed by global site, and every own plane sees exact neighbours)."""
import os
import subprocess
import sys

import numpy as np
import pytest

import asd_inputs as ai
from asd_inputs import slabs as sl
from tests.helpers import oracle_from_workload
from tests.slab_oracle import OracleSlabs

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_slab_plan_indices():
    s = sl.slab_bounds(23, 3, halo=2)
    assert [(a.lo, a.hi, a.glo, a.ghi) for a in s] == [(0, 8, 0, 10), (8, 16, 6, 18), (16, 23, 14, 23)]
    assert [a.own_first for a in s] == [0, 2, 2] and sum(a.n_own for a in s) == 23
    # ghosts are filled from the owners' planes next to the cut: global planes 6, 7 -> slab 1's planes 0, 1; 8, 9 -> slab 0's 8, 9
    assert sl.halo_moves(s, 2) == [(0, 6, 1, 0, 2), (1, 2, 0, 8, 2), (1, 8, 2, 0, 2), (2, 2, 1, 10, 2)]
    # a shift by 3: slab 0's top three own planes (local 5, 6, 7) become slab 1's first three own planes (local 2, 3, 4)
    assert sl.shift_moves(s, 3) == [(1, 2, 0, 5, 3), (2, 2, 1, 7, 3)]
    with pytest.raises(ValueError):
        sl.slab_bounds(9, 4, halo=4)
    with pytest.raises(ValueError):
        sl.slab_bounds(20, 2, halo=3)
    w = ai.small_film(ai.SC, 23, 8, 3, extra_track=6)
    ws = sl.slab_workload(w, s[1])
    assert (ws.nx, ws.x0, ws.track_nx) == (12, 6, w.track_nx)
    assert np.array_equal(ws.T, w.T[6 * 24:18 * 24]) and np.array_equal(ws.sz, w.sz[6 * 24:18 * 24])


@pytest.mark.parametrize("lattice", [ai.SC, ai.L10])
@pytest.mark.parametrize("nslabs,halo", [(2, 2), (3, 2), (2, 4)])
def test_oracle_slabs_are_bit_identical_to_the_whole_window(lattice, nslabs, halo):
    w = ai.small_film(lattice, 24, 12, 4, extra_track=10, tilt_deg=20.0, dt=1e-16)
    whole = oracle_from_workload(w)
    parts = OracleSlabs(w, nslabs, halo)
    plane = w.ny * w.nz

    def same():
        S = whole.get_spins()
        for r, s in enumerate(parts.slabs):
            assert np.array_equal(parts.own(r), S[:, s.lo * plane:s.hi * plane])
    for sim in (whole, parts):
        sim.step_heun(3)
    same()
    for sim in (whole, parts):
        sim.set_field_scale(-0.5); sim.shift_window(3); sim.step_heun(2); sim.shift_window(4); sim.step_heun(3)
    same()
    # what left the window went to slab 0's track store, exactly as to the whole window's
    _, cnt_w, sum_w = whole.track_get()
    _, cnt_0, sum_0 = parts.o[0].track_get()
    assert np.array_equal(cnt_w, cnt_0) and np.array_equal(sum_w, sum_0)


_WORKER = r"""
import os, sys
import numpy as np
import torch.distributed as dist
sys.path.insert(0, {root!r})
import asd_inputs as ai
from tests.helpers import oracle_from_workload
from tests.slab_oracle import OracleSlabs
dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
w = ai.small_film(ai.L10, 20, 12, 3, extra_track=8, tilt_deg=20.0, dt=1e-16)
parts = OracleSlabs(w, world, halo=2, mine=[rank], dist=dist)
parts.step_heun(2); parts.shift_window(3); parts.step_heun(3)
own = parts.own(rank)
if rank == 0:
    import torch
    pieces = [own]
    for r in range(1, world):
        s = parts.slabs[r]
        buf = torch.empty((3, s.n_own * w.ny * w.nz), dtype=torch.float64)
        dist.recv(buf, src=r)
        pieces.append(buf.numpy())
    whole = oracle_from_workload(w)
    whole.step_heun(2); whole.shift_window(3); whole.step_heun(3)
    ok = np.array_equal(np.concatenate(pieces, axis=1), whole.get_spins())
    print("SLABS_BIT_IDENTICAL" if ok else "SLABS_DIFFER", flush=True)
else:
    import torch
    dist.send(torch.from_numpy(own.copy()), dst=0)
dist.barrier()
dist.destroy_process_group()
"""


def test_two_rank_gloo_slab_decomposition(tmp_path):
    script = tmp_path / "slab_worker.py"
    script.write_text(_WORKER.format(root=ROOT))
    port = 29500 + (os.getpid() % 2000)
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr",
           "127.0.0.1", "--master-port", str(port), str(script)]
    env = dict(os.environ, OMP_NUM_THREADS="2")
    r = subprocess.run(cmd, capture_output=True, text=True, timeout=300, env=env)
    assert r.returncode == 0, r.stdout[-2000:] + r.stderr[-2000:]
    assert "SLABS_BIT_IDENTICAL" in r.stdout, r.stdout[-2000:] + r.stderr[-2000:]
