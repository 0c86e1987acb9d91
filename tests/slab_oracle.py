"""The oracle as the ranks of a slab decomposition (test harness): the same index plan as the CUDA slab runner
(asd_inputs.slabs), planes moved as fp64 numpy arrays -- in one process, or between processes over torch.distributed."""
from __future__ import annotations

import numpy as np

from asd_inputs import slabs as sl
from oracle import asd_oracle as orc


class OracleSlabs:
    def __init__(self, w, nslabs, halo=2, mine=None, dist=None):
        self.w, self.halo, self.dist = w, halo, dist
        self.slabs = sl.slab_bounds(w.nx, nslabs, halo)
        self.mine = list(range(nslabs)) if mine is None else list(mine)
        self.o = {r: orc.from_workload(sl.slab_workload(w, self.slabs[r])) for r in self.mine}
        self.plane = w.ny * w.nz
        self.fresh = 0

    def _get(self, r, p0, n):
        return self.o[r].get_spins()[:, p0 * self.plane:(p0 + n) * self.plane].copy()

    def _put(self, r, p0, block):
        S = self.o[r].get_spins()
        S[:, p0 * self.plane:p0 * self.plane + block.shape[1]] = block
        self.o[r].set_spins_f64(S)

    def _fetch(self, moves):
        """-> {(dst_rank, dst_plane): block} for the moves whose destination lives here."""
        import torch
        got = {}
        for (sr, sp, dr, dp, n) in moves:
            if sr in self.o and dr in self.o:
                got[(dr, dp)] = self._get(sr, sp, n)
            elif sr in self.o:
                self.dist.send(torch.from_numpy(self._get(sr, sp, n)), dst=dr)
            elif dr in self.o:
                buf = torch.empty((3, n * self.plane), dtype=torch.float64)
                self.dist.recv(buf, src=sr)
                got[(dr, dp)] = buf.numpy()
        return got

    def exchange(self):
        for (dr, dp), block in self._fetch(sl.halo_moves(self.slabs, self.halo)).items():
            self._put(dr, dp, block)
        self.fresh = self.halo // 2

    def step_heun(self, n=1):
        while n > 0:
            if self.fresh == 0:
                self.exchange()
            k = min(n, self.fresh)
            for o in self.o.values():
                o.step_heun(k)
            self.fresh -= k
            n -= k

    def set_field_scale(self, s):
        for o in self.o.values():
            o.set_field_scale(s)

    def shift_window(self, p):
        staged = self._fetch(sl.shift_moves(self.slabs, p))
        for o in self.o.values():
            assert o.shift_window(p) == 0
        for (dr, dp), block in staged.items():
            self._put(dr, dp, block)
        self.fresh = 0

    def own(self, r):
        s = self.slabs[r]
        return self._get(r, s.own_first, s.n_own)
