"""Pins for the oracle's passes over the track and its read-back scan (PAPER.md P:122-124 and
P:114; readings T1-T3 of DESIGN.md sec. 13).  All `-m "not gpu"`.

T1 end_pass    integer-valued "spins": the flush of the window into the track is exact and is compared with an
               independent numpy statement (np.add.at over floor-divided coordinates of ALL window planes); a pass
               ended after shifts has counted every magnetic site of planes [0, x0 + nx) exactly once; the committed
               init_mean is sum / count where count > 0 and untouched elsewhere.
T2 begin_pass  the regenerated window is a pure function of (seed, pass, global site): it equals, site for site, what
               shift_window seeds for the same atoms when the pass counter has the same value; magnitudes: the cone
               reproduces |mean| of the track cells (the purpose clause of P:68); pass 1 differs from pass 0.
T3 read_scan   uniform track -> exactly that value; linear in the written store; translation covariance by whole
               cells; a sharp transition read with a fine-celled track follows the closed form
               R(x) = -erf((x - x_t) / (sqrt(2) sigma_x)); a pattern on the other track is suppressed by the Gaussian.
"""
import math

import numpy as np
import pytest

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


def _numpy_flush(S, gm, x0, macro, dims):
    """Eq. (6) over every plane of the window, written from the definition.  S: [3, nx, nz, ny]."""
    _, nx, nz, ny = S.shape
    mx, my, mz = macro
    tsum, tcnt = np.zeros((3,) + dims), np.zeros(dims, dtype=np.int64)
    i, k, j = np.meshgrid(np.arange(nx), np.arange(nz), np.arange(ny), indexing="ij")
    magnetic = gm[x0 + i, j] >= 0
    cx, cy, cz = (x0 + i) // mx, j // my, k // mz
    for a in range(3):
        np.add.at(tsum[a], (cx[magnetic], cy[magnetic], cz[magnetic]), S[a][magnetic])
    np.add.at(tcnt, (cx[magnetic], cy[magnetic], cz[magnetic]), 1)
    return tsum, tcnt


@pytest.mark.parametrize("lattice,dims,macro", [(ai.SC, (17, 20, 9), (7, 7, 7)), (ai.L10, (12, 28, 7), (5, 7, 5))])
def test_t1_end_pass_flushes_the_window_exactly(lattice, dims, macro):
    nx, ny, nz = dims
    w = _integer_valued(ai.small_film(lattice, nx, ny, nz, extra_track=22, macro=macro))
    o = oracle_from_workload(w)
    cd = o.track_dims()
    o.shift_window(3); o.shift_window(5)
    _, cnt0, sum0 = o.track_get()
    S = o.get_spins().reshape(3, nx, nz, ny)
    fs, fc = _numpy_flush(S, w.grain_map, 8, macro, cd)
    init0 = np.full((int(np.prod(cd)), 3), 0.25, dtype=np.float32)
    o.track_set_init(init0)
    assert o.track_end_pass() == 0
    mean, cnt, sm = o.track_get()
    assert np.array_equal(cnt.reshape(cd), cnt0.reshape(cd) + fc)
    assert np.array_equal(sm.reshape(cd + (3,)), sum0.reshape(cd + (3,)) + np.moveaxis(fs, 0, -1))
    # every magnetic site of planes [0, x0 + nx) was counted exactly once
    covered = np.broadcast_to((w.grain_map[:8 + nx, :] >= 0)[:, None, :], (8 + nx, nz, ny)).sum()
    assert cnt.sum() == covered
    # what lies ahead of the next pass: the mean spin of written cells, the old value elsewhere.  Seen through a
    # begin_pass over a stretch of track that holds both kinds of cell: integer-valued sums have |mean| > 1, so m = 1 and
    # a written cell's sites are seeded exactly along its mean; unwritten cells keep v = (1/4, 1/4, 1/4).
    assert np.any(cnt == 0) and np.any(cnt > 0)
    x1 = 8 + nx - nx // 2                                       # straddles the end of what was written
    assert o.track_begin_pass(x1) == 0
    R = o.get_spins().reshape(3, nx, nz, ny)
    mx, my, mz = macro
    cntg, meang = cnt.reshape(cd), mean.reshape(cd + (3,))
    i, k, j = np.meshgrid(np.arange(nx), np.arange(nz), np.arange(ny), indexing="ij")
    cell = ((x1 + i) // mx, j // my, k // mz)
    magnetic = w.grain_map[x1 + i, j] >= 0
    written = magnetic & (cntg[cell] > 0)
    fresh = magnetic & (cntg[cell] == 0)
    assert written.sum() > 200 and fresh.sum() > 200
    v = meang[cell]                                             # [nx, nz, ny, 3]
    nhat = v / np.maximum(np.linalg.norm(v, axis=-1, keepdims=True), 1e-300)
    assert np.allclose(np.moveaxis(R, 0, -1)[written], nhat[written], atol=1e-13)
    got = np.moveaxis(R, 0, -1)[fresh].mean(axis=0)
    assert np.linalg.norm(got - 0.25) < 4.0 / math.sqrt(fresh.sum())
    assert np.all(np.moveaxis(R, 0, -1)[~magnetic] == 0.0)


def test_t1_t2_commit_and_regenerate_reproduce_the_written_magnetisation():
    """A window with a known mean spin per cell is flushed; the next pass's window, regenerated from the track at the
    same place, has that mean per cell within the sampling error of the cone (P:68 purpose clause), and other spins."""
    nx, ny, nz = 12, 48, 12
    w = ai.small_film(ai.SC, nx, ny, nz, extra_track=0, macro=(6, 24, 12), pitch_nm=50.0, boundary_nm=0.0)
    assert np.all(w.grain_map >= 0)
    # four cells (2 along x, 2 across): uniform spin directions with different tilts => |mean| of a cell is 1; mix two
    # directions inside each cell to get |mean| < 1
    rng = np.random.default_rng(5)
    S = np.zeros((3, nx, nz, ny))
    target = {}
    for cx in range(2):
        for cy in range(2):
            a = rng.standard_normal(3); a /= np.linalg.norm(a)
            b = rng.standard_normal(3); b /= np.linalg.norm(b)
            blk = S[:, cx * 6:(cx + 1) * 6, :, cy * 24:(cy + 1) * 24]
            half = blk.shape[3] // 2
            blk[:, :, :, :half] = a[:, None, None, None]
            blk[:, :, :, half:] = b[:, None, None, None]
            target[(cx, cy)] = 0.5 * (a.astype(np.float32).astype(float) + b.astype(np.float32).astype(float))
    w.sx, w.sy, w.sz = (S[a].reshape(-1).astype(np.float32) for a in range(3))
    o = oracle_from_workload(w)
    assert o.track_end_pass() == 0
    mean, cnt, _ = o.track_get()
    mean = mean.reshape(2, 2, 1, 3)
    for (cx, cy), t in target.items():
        assert np.allclose(mean[cx, cy, 0], t, atol=1e-12)
    before = o.get_spins().copy()
    assert o.counters()["pass"] == 0
    assert o.track_begin_pass(0) == 0
    c = o.counters()
    assert c["pass"] == 1 and c["x0"] == 0
    _, cnt2, sm2 = o.track_get()
    assert not cnt2.any() and not sm2.any()                     # the written store starts empty
    R = o.get_spins().reshape(3, nx, nz, ny)
    assert np.allclose(np.sqrt((R ** 2).sum(axis=0)), 1.0, atol=1e-14)
    assert not np.array_equal(R.reshape(3, -1), before)
    n_cell = 6 * 12 * 24
    for (cx, cy), t in target.items():
        got = R[:, cx * 6:(cx + 1) * 6, :, cy * 24:(cy + 1) * 24].reshape(3, -1).mean(axis=1)
        assert np.linalg.norm(got - t) < 4.0 / math.sqrt(n_cell)


def test_t2_regenerated_window_is_what_a_shift_seeds_for_the_same_atoms():
    """Seeding is a pure function of (seed, pass, global site, track cell): begin_pass(x0) gives plane x0 + i the spins
    that shift_window gives it when it enters a window whose pass counter has the same value."""
    nx, ny, nz = 10, 16, 6
    w = ai.small_film(ai.L10, nx, ny, nz, extra_track=14, macro=(3, 4, 2))
    rng = np.random.default_rng(11)
    a = oracle_from_workload(w)
    ncell = int(np.prod(a.track_dims()))
    init = (0.2 + 0.7 * rng.random((ncell, 1))) * _unit(rng.standard_normal((ncell, 3)))
    init = init.astype(np.float32)
    a.track_set_init(init)
    assert a.track_begin_pass(9) == 0                             # pass 0 -> 1, window over planes 9..18
    A = a.get_spins().reshape(3, nx, nz, ny)
    b = oracle_from_workload(w)
    b.track_set_init(init)
    b.set_counters(0, 0, 1)                                       # same pass counter, window still at plane 0
    assert b.shift_window(nx) == 0 and b.shift_window(4) == 0     # planes 10..19, then 14..23
    B = b.get_spins().reshape(3, nx, nz, ny)
    assert np.array_equal(A[:, 5:], B[:, :5])                     # global planes 14..18 on both
    # and pass 0 seeds other spins for the same atoms
    c = oracle_from_workload(w)
    c.track_set_init(init)
    c.shift_window(nx); c.shift_window(4)
    assert not np.array_equal(c.get_spins().reshape(3, nx, nz, ny)[:, :5], B[:, :5])
    assert a.track_begin_pass(15) != 0                            # past the end of the track
    assert a.track_begin_pass(-1) != 0


def _unit(v):
    return v / np.linalg.norm(v, axis=-1, keepdims=True)


def _written_track(track_nx, ny, nz, macro, sz_of_site):
    """An oracle whose written store holds sz_of_site(gx, j) on every site of a fully magnetic track (through the public
    calls: set_spins + end_pass with a window as long as the track)."""
    w = ai.small_film(ai.SC, track_nx, ny, nz, extra_track=0, macro=macro, pitch_nm=500.0, boundary_nm=0.0)
    assert np.all(w.grain_map >= 0)
    gx, k, j = np.meshgrid(np.arange(track_nx), np.arange(nz), np.arange(ny), indexing="ij")
    w.sz = sz_of_site(gx, j).astype(np.float32).reshape(-1)
    w.sx = np.zeros_like(w.sz); w.sy = np.zeros_like(w.sz)
    o = oracle_from_workload(w)
    assert o.track_end_pass() == 0
    return o


def test_t3_uniform_track_reads_its_value_and_scan_is_linear():
    o1 = _written_track(40, 24, 4, (4, 4, 2), lambda gx, j: np.full(gx.shape, 0.625))
    r = o1.track_read_scan(11.0, 3.0, 5.0, 2.0, 1.5, 20)
    assert np.allclose(r, 0.625, atol=1e-15)
    f = lambda gx, j: np.sin(0.3 * gx) * np.cos(0.2 * j)
    g = lambda gx, j: ((gx // 8) % 2) * 2.0 - 1.0
    a = _written_track(40, 24, 4, (4, 4, 2), f).track_read_scan(11.0, 3.0, 5.0, 2.0, 1.5, 20)
    b = _written_track(40, 24, 4, (4, 4, 2), g).track_read_scan(11.0, 3.0, 5.0, 2.0, 1.5, 20)
    ab = _written_track(40, 24, 4, (4, 4, 2), lambda gx, j: 0.5 * f(gx, j) - 0.25 * g(gx, j)).track_read_scan(
        11.0, 3.0, 5.0, 2.0, 1.5, 20)
    assert np.allclose(ab, 0.5 * a - 0.25 * b, atol=1e-7)          # fp32 inputs
    # an unwritten track reads 0
    w = ai.small_film(ai.SC, 8, 8, 3, extra_track=4)
    assert not oracle_from_workload(w).track_read_scan(3.0, 2.0, 2.0, 0.0, 1.0, 5).any()


def test_t3_translation_covariance_by_whole_cells():
    pat = lambda s: (lambda gx, j: np.where(((gx - s) // 12) % 2 == 0, 0.8, -0.7) * (np.abs(j - 10) < 6))
    a = _written_track(120, 24, 2, (4, 4, 2), pat(0)).track_read_scan(10.0, 5.0, 4.0, 40.0, 1.0, 30)
    b = _written_track(120, 24, 2, (4, 4, 2), pat(8)).track_read_scan(10.0, 5.0, 4.0, 48.0, 1.0, 30)
    assert np.allclose(a, b, atol=1e-9)        # far from the track ends: the footprint sees the same cells


def test_t3_sharp_transition_follows_the_error_function():
    """Cells of one site (macro 1): the scan across a step from +1 to -1 at plane x_t is the Gaussian-smoothed step,
    R(x) = -erf((x - x_t) / (sqrt 2 sigma_x)), up to the midpoint-rule error of summing unit cells."""
    x_t, sig = 60, 6.0
    o = _written_track(120, 8, 1, (1, 1, 1), lambda gx, j: np.where(gx < x_t, 1.0, -1.0))
    xs = 40.0 + np.arange(41)
    r = o.track_read_scan(4.0, sig, 3.0, 40.0, 1.0, 41)
    ref = np.array([-math.erf((x - x_t) / (math.sqrt(2.0) * sig)) for x in xs])
    assert np.abs(r - ref).max() < 2e-3
    assert abs(r[20]) < 1e-12                  # reader centred on the transition: antisymmetric => 0
    # coarser cells: same curve within O((cell / sigma)^2)
    o4 = _written_track(120, 8, 1, (4, 1, 1), lambda gx, j: np.where(gx < x_t, 1.0, -1.0))
    r4 = o4.track_read_scan(4.0, sig, 3.0, 40.0, 1.0, 41)
    assert np.abs(r4 - ref).max() < 0.06


def test_t3_other_track_is_suppressed_by_the_footprint():
    """Two bit rows 30 sites apart, reader sigma_y = 5: the far row enters with weight exp(-30^2 / 50) ~ 1.5e-8."""
    rows = lambda gx, j: np.where(np.abs(j - 15) < 6, 1.0, 0.0) * 0.9 - np.where(np.abs(j - 45) < 6, 1.0, 0.0) * 0.9
    o = _written_track(60, 60, 2, (3, 3, 2), rows)
    lo = o.track_read_scan(15.0, 4.0, 2.0, 30.0, 1.0, 1)[0]
    hi = o.track_read_scan(45.0, 4.0, 2.0, 30.0, 1.0, 1)[0]
    assert lo > 0.85 and hi < -0.85 and abs(lo + hi) < 1e-6


def test_two_track_workload_recipe():
    tt = ai.two_track_film(ai.SC, length_nm=12.0, width_nm=12.0, nz=4, n_bits=3, bit_nm=3.0, separation_nm=2.0,
                           bit_width_nm=4.0, pitch_nm=3.0, boundary_nm=0.6, shift_every=4, batch=2, macro=(3, 3, 2))
    w = tt.w
    assert w.ny % 4 == 0 and w.track_nx == w.nx + 3 * tt.bit_planes
    # spot centres: bottom / top track, 6 nm apart, symmetric about the film's centre line
    T0 = tt.T_pass[0].reshape(w.nx, w.nz, w.ny); T1 = tt.T_pass[1].reshape(w.nx, w.nz, w.ny)
    j0, j1 = np.unravel_index(T0[:, 0, :].argmax(), (w.nx, w.ny))[1], np.unravel_index(T1[:, 0, :].argmax(), (w.nx, w.ny))[1]
    assert abs((j0 + 0.5) - tt.track_y[0]) <= 0.5 and abs((j1 + 0.5) - tt.track_y[1]) <= 0.5
    assert abs((tt.track_y[1] - tt.track_y[0]) * w.spacing_nm[1] - 6.0) < 1e-9
    assert np.allclose(T0[:, :, ::-1], T1, atol=1e-3)
    # spot diameter above 710 K = the bit width
    hot = (T0[:, 0, :] > 710.0)
    assert abs(hot.any(axis=0).sum() * w.spacing_nm[1] - 4.0) <= 2 * w.spacing_nm[1]
    assert set(np.unique(np.concatenate(tt.bits))) <= {-1.0, 1.0} and not np.array_equal(tt.bits[0], tt.bits[1])
    # a full pass ends with the window at the end of the track
    assert sum(ai.planes_for_shift(q, w.spacing_nm[0]) for q in range(1, tt.n_periods + 1)) <= w.track_nx - w.nx


def test_two_passes_through_the_driver_oracle_side():
    """The call sequence of drive_pass on the oracle: counters, coverage, and the second pass starts from the first
    pass's written track."""
    tt = ai.two_track_film(ai.SC, length_nm=6.0, width_nm=9.6, nz=3, n_bits=2, bit_nm=3.0, separation_nm=1.8,
                           bit_width_nm=3.0, pitch_nm=3.0, boundary_nm=0.6, shift_every=3, batch=2, macro=(3, 3, 3),
                           dt=1e-16)
    w = tt.w
    o = oracle_from_workload(w)
    up = lambda sim, T: sim.set_fields(T=T)
    n0 = ai.drive_pass(o, tt, 0, up)
    assert n0 == tt.n_periods * 3
    mean0, cnt0, _ = o.track_get()
    x_end = o.counters()["x0"]
    covered = np.broadcast_to((w.grain_map[:x_end + w.nx, :] >= 0)[:, None, :], (x_end + w.nx, w.nz, w.ny)).sum()
    assert cnt0.sum() == covered
    r0 = ai.read_tracks(o, tt)
    assert r0.shape == (2, 2) and np.all(np.abs(r0) <= 1.0) and np.all(r0 > 0.5)    # 18 cold-ish steps: still +z
    ai.drive_pass(o, tt, 1, up)
    c = o.counters()
    assert c["pass"] == 1 and c["step"] == 2 * n0 and c["shift"] == 2 * tt.n_periods and c["x0"] == x_end
    mean1, cnt1, _ = o.track_get()
    assert np.array_equal(cnt0, cnt1)                       # the same atoms were read out in both passes
    assert not np.array_equal(mean0, mean1)
