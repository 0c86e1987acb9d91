"""Cutting one window into x-slabs: pure index arithmetic and array slicing, shared
by the CUDA slab runner (paper_2502_02236_b200/slab.py) and by the tests that run the oracle as the ranks.

A slab holds its own planes [lo, hi) of the window plus `halo` ghost planes towards each neighbour (none at the window's
two ends).  One Heun step spoils two ghost planes from the outside in, so `halo` planes last halo // 2 steps.
"""
from __future__ import annotations

import copy
from dataclasses import dataclass
from typing import List, Tuple

import numpy as np

from . import workloads as wl


@dataclass
class Slab:
    rank: int
    lo: int          # first own plane (window-local index of the whole window)
    hi: int          # one past the last own plane
    glo: int         # first plane held (own or ghost)
    ghi: int         # one past the last plane held

    @property
    def own_first(self) -> int:
        """Local index of the first own plane."""
        return self.lo - self.glo

    @property
    def n_own(self) -> int:
        return self.hi - self.lo

    @property
    def n_held(self) -> int:
        return self.ghi - self.glo


def slab_bounds(nx: int, world: int, halo: int = 2) -> List[Slab]:
    """Even split of nx planes over `world` slabs (the first nx % world slabs take one plane more)."""
    if halo < 2 or halo % 2:
        raise ValueError("halo must be an even number of planes >= 2")
    base, extra = divmod(nx, world)
    if base < halo:
        raise ValueError("every slab must own at least `halo` planes")
    out, lo = [], 0
    for r in range(world):
        hi = lo + base + (1 if r < extra else 0)
        out.append(Slab(rank=r, lo=lo, hi=hi, glo=max(0, lo - halo), ghi=min(nx, hi + halo)))
        lo = hi
    return out


def slab_workload(w: wl.Workload, s: Slab) -> wl.Workload:
    """The workload of one slab: planes [glo, ghi) of every per-site array; same track, grains and seed; the window
    origin moves with it, so global site ids (the Philox counters) are those of the whole window."""
    c = copy.copy(w)
    plane = w.ny * w.nz
    c.nx = s.n_held
    c.x0 = w.x0 + s.glo
    c.name = f"{w.name}[slab {s.rank}: planes {s.glo}..{s.ghi - 1}]"
    for name in ("T", "Bx", "By", "Bz", "sx", "sy", "sz"):
        setattr(c, name, getattr(w, name)[s.glo * plane:s.ghi * plane].copy())
    return c


def halo_moves(slabs: List[Slab], halo: int) -> List[Tuple[int, int, int, int, int]]:
    """(src_rank, src_local_plane, dst_rank, dst_local_plane, n_planes): the owners' planes that overwrite the ghosts."""
    mv = []
    for a, b in zip(slabs[:-1], slabs[1:]):
        mv.append((a.rank, a.hi - halo - a.glo, b.rank, 0, halo))                       # a's top own planes -> b's left ghosts
        mv.append((b.rank, b.own_first, a.rank, a.hi - a.glo, halo))                    # b's bottom own planes -> a's right ghosts
    return mv


def shift_moves(slabs: List[Slab], p: int) -> List[Tuple[int, int, int, int, int]]:
    """Before every slab shifts by p planes, slab r needs the first p own planes of slab r + 1 (their pre-shift values):
    after its own shift they are its top p own planes.  (src_rank, src_local_plane, dst_rank, dst_local_plane, n)."""
    mv = []
    for a, b in zip(slabs[:-1], slabs[1:]):
        if p > b.n_own or p > a.n_own:
            raise ValueError("a shift cannot be longer than a slab")
        mv.append((b.rank, b.own_first, a.rank, a.hi - p - a.glo, p))
    return mv


def assemble(slabs: List[Slab], pieces: List[np.ndarray], plane: int) -> np.ndarray:
    """[3, N] spins of the whole window from the slabs' [3, n_held * plane] arrays (own planes only)."""
    return np.concatenate([pc[:, s.own_first * plane:(s.own_first + s.n_own) * plane] for s, pc in zip(slabs, pieces)], axis=1)
