"""Pins P10 and P11 for the oracle's moving-window shift (Eq. (6) P:64-66,
cone thermalisation P:68).

P10  indexing: with integer-valued "spins" every move and every macrocell sum is exact, so the oracle is compared
     bit for bit with an independent numpy formulation written here from the definitions (array slicing for the
     move, np.add.at over floor-divided coordinates for Eq. (6)); two shifts p1, p2 == one shift p1 + p2.
P11  seeding: the distribution P:68 states (polar angle uniform on [0, theta_max] about M, free azimuth) and its
     stated purpose (the slab reproduces |M|/M_S^0 = m); theta_max against sin(t)/t = m and against the paper's
     radicand with the prefactor its own Taylor series gives (sqrt(10), S3).
"""
import math

import numpy as np
import pytest
from scipy import stats

import asd_inputs as ai
from oracle import asd_oracle as orc
from tests.helpers import oracle_from_workload


def _integer_valued(w):
    N = w.n_sites
    g = np.arange(N, dtype=np.int64)
    mag = w.magnetic_mask().reshape(-1)
    w.sx = ((g % 4093) * mag).astype(np.float32)
    w.sy = ((g // 4093) * mag).astype(np.float32)
    w.sz = ((g % 977 + 1) * mag).astype(np.float32)
    return w


def _numpy_shift(S, gm, x0, p, macro, track_sum, track_cnt):
    """Independent statement of O5 for the outgoing slab and the move.  S: [3, nx, nz, ny]."""
    _, nx, nz, ny = S.shape
    mx, my, mz = macro
    i, k, j = np.meshgrid(np.arange(p), np.arange(nz), np.arange(ny), indexing="ij")
    magnetic = gm[x0 + i, j] >= 0
    cx, cy, cz = (x0 + i) // mx, j // my, k // mz
    for a in range(3):
        np.add.at(track_sum[a], (cx[magnetic], cy[magnetic], cz[magnetic]), S[a, :p][magnetic])
    np.add.at(track_cnt, (cx[magnetic], cy[magnetic], cz[magnetic]), 1)
    return S[:, p:].copy()          # the block that stays, now at planes 0 .. nx-p-1


@pytest.mark.parametrize("lattice,dims,macro", [(ai.SC, (24, 20, 9), (7, 7, 7)), (ai.L10, (19, 28, 7), (7, 7, 5)),
                                                (ai.SC, (10, 9, 4), (3, 2, 3))])
def test_p10_shift_indexing_exact(lattice, dims, macro):
    nx, ny, nz = dims
    w = _integer_valued(ai.small_film(lattice, nx, ny, nz, extra_track=30, macro=macro))
    o = oracle_from_workload(w)
    ncx, ncy, ncz = o.track_dims()
    assert (ncx, ncy, ncz) == (-(-w.track_nx // macro[0]), -(-ny // macro[1]), -(-nz // macro[2]))
    tsum, tcnt = np.zeros((3, ncx, ncy, ncz)), np.zeros((ncx, ncy, ncz), dtype=np.int64)
    x0 = 0
    for p in (3, 4, 1, 7, 2):
        S = o.get_spins().reshape(3, nx, nz, ny)
        kept = _numpy_shift(S, w.grain_map, x0, p, macro, tsum, tcnt)
        assert o.shift_window(p) == 0
        x0 += p
        S2 = o.get_spins().reshape(3, nx, nz, ny)
        assert np.array_equal(S2[:, :nx - p], kept)
        _, cnt, sm = o.track_get()
        assert np.array_equal(cnt.reshape(ncx, ncy, ncz), tcnt)
        assert np.array_equal(sm.reshape(ncx, ncy, ncz, 3), np.moveaxis(tsum, 0, -1))
        # incoming planes: vacant columns 0, magnetic sites unit vectors
        tail = S2[:, nx - p:]
        vac = np.broadcast_to((w.grain_map[x0 + nx - p:x0 + nx, :] < 0)[:, None, :], tail.shape[1:])
        assert np.all(tail[:, vac] == 0.0)
        assert np.allclose(np.sqrt((tail[:, ~vac] ** 2).sum(axis=0)), 1.0, atol=1e-14)
        c = o.counters()
        assert c["x0"] == x0
    assert o.counters()["shift"] == 5
    # every magnetic site that left the window was counted exactly once
    left = np.broadcast_to((w.grain_map[:x0, :] >= 0)[:, None, :], (x0, nz, ny)).sum()
    assert tcnt.sum() == left


def test_p10_two_shifts_equal_one():
    w = _integer_valued(ai.small_film(ai.SC, 20, 12, 6, extra_track=20, macro=(7, 7, 7)))
    a, b = oracle_from_workload(w), oracle_from_workload(w)
    a.shift_window(3); a.shift_window(5)
    b.shift_window(8)
    nkeep = (20 - 8) * 12 * 6
    assert np.array_equal(a.get_spins()[:, :nkeep], b.get_spins()[:, :nkeep])
    ma, ca, sa = a.track_get()
    mb, cb, sb = b.track_get()
    assert np.array_equal(ca, cb) and np.array_equal(sa, sb)
    assert a.counters()["x0"] == b.counters()["x0"] == 8
    # the seeded planes are a pure function of (seed, pass, global site): same atoms, same spins
    assert np.array_equal(a.get_spins()[:, nkeep + 3 * 72:], b.get_spins()[:, nkeep + 3 * 72:])


def test_shift_rejects_bad_arguments():
    w = ai.small_film(ai.SC, 8, 8, 3, extra_track=2)
    o = oracle_from_workload(w)
    assert o.shift_window(0) != 0
    assert o.shift_window(9) != 0
    assert o.shift_window(3) != 0          # past the end of the track
    assert o.shift_window(2) == 0


@pytest.mark.parametrize("m", [0.999, 0.9, 0.7, 0.5, 0.2, 0.05])
def test_p11_theta_max_reproduces_m(m):
    """<cos theta> of a polar angle uniform on [0, theta_max] is sin(theta_max)/theta_max: that must equal m."""
    t = orc.theta_max(m)
    assert 0.0 < t < math.pi
    assert abs(math.sin(t) / t - m) < 1e-12
    # numerical mean of cos over the uniform polar angle (the stated distribution), midpoint rule
    th = (np.arange(200000) + 0.5) / 200000 * t
    assert abs(np.cos(th).mean() - m) < 1e-9


def test_p11_theta_max_limits_and_paper_series():
    assert orc.theta_max(1.0) == 0.0
    assert abs(orc.theta_max(0.0) - math.pi) < 1e-12
    # P:68 prints theta_max = (5 pi/9) sqrt(1 - sqrt(1 + 6 (m - 1)/5)).  Inverting the Taylor series of
    # sin(t)/t = 1 - t^2/6 + t^4/120 gives exactly that radicand with prefactor sqrt(10); it agrees with the
    # root to O((1-m)^2.5) and the printed prefactor 5 pi/9 does not (S3).
    for m in (0.999, 0.99, 0.95):
        rad = math.sqrt(1.0 - math.sqrt(1.0 + 6.0 * (m - 1.0) / 5.0))
        series = math.sqrt(10.0) * rad
        printed = (5.0 * math.pi / 9.0) * rad
        t = orc.theta_max(m)
        assert abs(series / t - 1.0) < 0.3 * (1.0 - m) ** 2 + 1e-9
        assert abs(printed / t - 1.0) > 0.4


def test_p11_seeded_slab_distribution_and_magnitude():
    nx, ny, nz = 12, 48, 12
    w = ai.small_film(ai.SC, nx, ny, nz, extra_track=nx, macro=(nx, ny, nz), pitch_nm=50.0, boundary_nm=0.0)
    assert np.all(w.grain_map >= 0)                      # one magnetic block: every incoming site is seeded
    rng = np.random.default_rng(3)
    for m, n in ((0.8, (0.0, 0.0, 1.0)), (0.55, (1.0, 0.0, 0.0)), (0.3, tuple(rng.standard_normal(3)))):
        n = np.asarray(n) / np.linalg.norm(n)
        o = oracle_from_workload(w)
        ncell = int(np.prod(o.track_dims()))
        o.track_set_init(np.tile((m * n).astype(np.float32), (ncell, 1)))
        assert o.shift_window(nx) == 0                    # the whole window is new
        S = o.get_spins()
        N = S.shape[1]
        assert np.allclose(np.sqrt((S ** 2).sum(axis=0)), 1.0, atol=1e-14)
        mean = S.mean(axis=1)
        n32 = (m * n).astype(np.float32).astype(np.float64)
        m32 = np.linalg.norm(n32)
        assert abs(np.linalg.norm(mean) - m32) < 3.0 / math.sqrt(N)           # purpose clause of P:68
        assert np.linalg.norm(mean / np.linalg.norm(mean) - n32 / m32) < 4.0 / math.sqrt(N)
        # polar angle about n uniform on [0, theta_max]; azimuth uniform
        c = np.clip((S * (n32 / m32)[:, None]).sum(axis=0), -1.0, 1.0)
        theta = np.arccos(c)
        tmax = orc.theta_max(m32)
        assert theta.max() <= tmax + 1e-9
        assert stats.kstest(theta / tmax, "uniform").pvalue > 1e-3
    # m = 1: all spins exactly n
    o = oracle_from_workload(w)
    o.track_set_init(None, 1.0)
    o.shift_window(nx)
    S = o.get_spins()
    assert np.all(S[2] == 1.0) and np.all(S[0] == 0.0) and np.all(S[1] == 0.0)
