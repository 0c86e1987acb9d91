"""One window cut into x-slabs across devices.

Every slab is an ordinary `Context` over its own planes plus `halo` ghost planes towards each neighbour; between Heun
steps the owners' planes are copied over the ghosts.  Nothing here computes: the copies are device-to-device copies of
the library's own plane storage (asd_planes_view), between the contexts of one process (`SlabWindow.local`: all slabs
on one device, for testing the decomposition on a single GPU) or between ranks with torch.distributed send / recv over
NCCL -- NVLink peer traffic on an NVSwitch node (`SlabWindow.distributed`: one slab per rank).  Because the noise is keyed
by global site, the result is bit-identical to the undivided window's as long as every slab runs the same kernel variant.
"""
from __future__ import annotations

from typing import List, Optional

import numpy as np

import asd_inputs as ai
from asd_inputs import slabs as sl
from . import binding as asd


class SlabWindow:
    def __init__(self, w: ai.Workload, slabs: List[sl.Slab], mine: List[int], halo: int, device: str, dist=None,
                 kernel: Optional[int] = None):
        self.w, self.slabs, self.mine, self.halo, self.dist = w, slabs, mine, halo, dist
        self.ctx = {r: asd.context_from_workload(sl.slab_workload(w, slabs[r]), device=device) for r in mine}
        if kernel is not None:
            for c in self.ctx.values():
                c.set_kernel(kernel)
        self.fresh = 0                      # Heun steps the ghost planes are still good for

    # ---- construction ----
    @classmethod
    def local(cls, w: ai.Workload, nslabs: int, halo: int = 2, device: str = "cuda:0", kernel: Optional[int] = None):
        slabs = sl.slab_bounds(w.nx, nslabs, halo)
        return cls(w, slabs, list(range(nslabs)), halo, device, None, kernel)

    @classmethod
    def distributed(cls, w: ai.Workload, dist, halo: int = 2, device: str = "cuda:0", kernel: Optional[int] = None):
        slabs = sl.slab_bounds(w.nx, dist.get_world_size(), halo)
        return cls(w, slabs, [dist.get_rank()], halo, device, dist, kernel)

    # ---- plane traffic ----
    def _move(self, moves):
        """Carries out (src_rank, src_plane, dst_rank, dst_plane, n) plane copies, all three components."""
        import torch
        ops, keep = [], []
        for (sr, sp, dr, dp, n) in moves:
            for comp in range(3):
                if sr in self.ctx and dr in self.ctx:
                    self.ctx[dr].planes_view(comp, dp, n).copy_(self.ctx[sr].planes_view(comp, sp, n))
                elif sr in self.ctx:
                    ops.append(self.dist.P2POp(self.dist.isend, self.ctx[sr].planes_view(comp, sp, n), dr))
                elif dr in self.ctx:
                    ops.append(self.dist.P2POp(self.dist.irecv, self.ctx[dr].planes_view(comp, dp, n), sr))
        if ops:
            for req in self.dist.batch_isend_irecv(ops):
                req.wait()

    def exchange(self):
        self._move(sl.halo_moves(self.slabs, self.halo))
        self.fresh = self.halo // 2

    # ---- the library's calls, slab-wise ----
    def step_heun(self, n: int = 1):
        while n > 0:
            if self.fresh == 0:
                self.exchange()
            k = min(n, self.fresh)
            for c in self.ctx.values():
                c.step_heun(k)
            self.fresh -= k
            n -= k

    def set_field_scale(self, s: float):
        for c in self.ctx.values():
            c.set_field_scale(s)

    def shift_window(self, p: int):
        """Slab r's top p own planes come from slab r + 1 (pre-shift values, staged through a copy because the source
        slab shifts too); slab 0's outgoing planes go to the track, the last slab's incoming planes come from it."""
        import torch
        moves = sl.shift_moves(self.slabs, p)
        staged = {}
        ops = []
        for (sr, sp, dr, dp, n) in moves:
            for comp in range(3):
                if sr in self.ctx and dr in self.ctx:
                    staged[(dr, comp)] = self.ctx[sr].planes_view(comp, sp, n).clone()
                elif sr in self.ctx:
                    ops.append(self.dist.P2POp(self.dist.isend, self.ctx[sr].planes_view(comp, sp, n).clone(), dr))
                elif dr in self.ctx:
                    buf = torch.empty_like(self.ctx[dr].planes_view(comp, dp, n))
                    staged[(dr, comp)] = buf
                    ops.append(self.dist.P2POp(self.dist.irecv, buf, sr))
        if ops:
            for req in self.dist.batch_isend_irecv(ops):
                req.wait()
        for c in self.ctx.values():
            c.shift_window(p)
        for (sr, sp, dr, dp, n) in moves:
            if dr in self.ctx:
                for comp in range(3):
                    self.ctx[dr].planes_view(comp, dp, n).copy_(staged[(dr, comp)])
        self.fresh = 0

    def magnetisation(self):
        """Mean spin over the magnetic sites of the whole window (own planes of every slab; all-reduced across ranks)."""
        tot = np.zeros(4)
        for r, c in self.ctx.items():
            s = self.slabs[r]
            v, cnt = c.magnetisation_planes(s.own_first, s.n_own)
            tot[:3] += v; tot[3] += cnt
        if self.dist is not None:
            import torch
            t = torch.from_numpy(tot).to(next(iter(self.ctx.values())).device)
            self.dist.all_reduce(t)
            tot = t.cpu().numpy()
        return tot[:3] / max(tot[3], 1.0), tot[3]

    def own_spins_host(self):
        """{rank: [3, n_own * plane]} of the slabs held here."""
        plane = self.w.ny * self.w.nz
        out = {}
        for r, c in self.ctx.items():
            s = self.slabs[r]
            out[r] = c.get_spins_host()[:, s.own_first * plane:(s.own_first + s.n_own) * plane]
        return out

    def gather_spins_host(self) -> np.ndarray:
        """[3, N] spins of the whole window (local mode)."""
        own = self.own_spins_host()
        return np.concatenate([own[r] for r in sorted(own)], axis=1)
