"""Pin P12: the oracle's demagnetising field (Eq. (6)-(7)).

The tensor N of two equal cuboids (Newell et al. 1993, the paper's ref. [28]) and the cell field B_c = -mu_0 sum N M are
checked against things that are not the oracle's formula:
  * the interaction of two separated cells by direct Gauss-Legendre quadrature of the point-dipole kernel over both
    volumes (no closed form involved) -- every component, with sign;
  * textbook values: a cube demagnetises itself with N = 1/3 per axis; tr N = 1 for a cell on itself and 0 between
    different cells; the point-dipole limit at distance;
  * the sum rule: a block of n cells, uniformly magnetised, IS one big cuboid, so the average over its cells of
    sum_c' N(c' - c) must equal the self-tensor of the big cuboid -- pins the offset bookkeeping of the cell sum;
  * the thin-film limit: an extended film magnetised along its normal has B_d -> -mu_0 M at its centre, and -> 0 in plane.
"""
import numpy as np
import pytest

import asd_inputs as ai

from oracle import asd_oracle as orc
from tests.helpers import single_grain_spec

MU0 = 4e-7 * np.pi


def _quad_tensor(cell, R, order=8):
    """N_ab = (1/V) int_V d3r int_V' d3r' (1/4pi) (delta_ab/rho^3 - 3 rho_a rho_b/rho^5), rho = R + r' - r."""
    x, w = np.polynomial.legendre.leggauss(order)
    pts = [0.5 * c * x for c in cell]
    wts = [0.5 * c * w for c in cell]
    g = np.meshgrid(*pts, indexing="ij"); gw = np.meshgrid(*wts, indexing="ij")
    P = np.stack([a.ravel() for a in g], axis=1); W = (gw[0] * gw[1] * gw[2]).ravel()
    rho = np.asarray(R)[None, None, :] + P[None, :, :] - P[:, None, :]
    r2 = (rho ** 2).sum(-1); r5 = r2 ** 2.5
    ww = W[:, None] * W[None, :]
    V = float(np.prod(cell))
    out = np.zeros((3, 3))
    for a in range(3):
        for b in range(3):
            k = ((a == b) * r2 - 3.0 * rho[..., a] * rho[..., b]) / r5 / (4.0 * np.pi)
            out[a, b] = (k * ww).sum() / V
    return np.array([out[0, 0], out[1, 1], out[2, 2], out[0, 1], out[0, 2], out[1, 2]])


def test_p12_tensor_matches_direct_quadrature_of_the_dipole_kernel():
    cell = (2.1e-9, 1.9e-9, 1.4e-9)
    for R in [(2, 0, 0), (0, 2, 0), (0, 0, 3), (2, 1, 0), (2, -1, 1), (-2, 2, -1), (3, 2, 2), (-3, -2, 1)]:
        Rm = [r * c for r, c in zip(R, cell)]
        got, want = orc.newell_tensor(cell, Rm), _quad_tensor(cell, Rm)
        assert np.allclose(got, want, rtol=2e-5, atol=2e-8), (R, got, want)


def test_p12_textbook_values_and_symmetries():
    N = orc.newell_tensor
    assert np.allclose(N((1, 1, 1), (0, 0, 0)), [1 / 3, 1 / 3, 1 / 3, 0, 0, 0], atol=1e-12)
    s = N((3.0, 1.0, 0.4), (0, 0, 0))
    assert abs(s[:3].sum() - 1.0) < 1e-12 and s[0] < s[1] < s[2]          # the short axis demagnetises most
    for R in [(1, 0, 0), (1, 1, 0), (2, -1, 3), (0, 0, 1)]:
        t = N((1.0, 0.8, 0.6), (R[0] * 1.0, R[1] * 0.8, R[2] * 0.6))
        assert abs(t[:3].sum()) < 1e-12                                       # no self-term between different cells
        assert np.allclose(t, N((1.0, 0.8, 0.6), (-R[0] * 1.0, -R[1] * 0.8, -R[2] * 0.6)), atol=1e-14)   # N(-R) = N(R)
    a, b = N((1, 1, 1), (2, 1, 3)), N((1, 1, 1), (-2, 1, 3))
    assert np.allclose(a[[0, 1, 2, 5]], b[[0, 1, 2, 5]], atol=1e-14) and np.allclose(a[[3, 4]], -b[[3, 4]], atol=1e-14)
    # point-dipole limit, on both sides of the switch-over radius (reading D2)
    for scale in (6.0, 11.0, 25.0):
        R = np.array([1.0, 0.7, -0.4]) * scale
        r = np.linalg.norm(R); c = 1.0 / (4 * np.pi * r ** 3)
        dip = np.array([c * (1 - 3 * R[0] ** 2 / r ** 2), c * (1 - 3 * R[1] ** 2 / r ** 2), c * (1 - 3 * R[2] ** 2 / r ** 2),
                        -3 * c * R[0] * R[1] / r ** 2, -3 * c * R[0] * R[2] / r ** 2, -3 * c * R[1] * R[2] / r ** 2])
        assert np.allclose(N((1, 1, 1), R), dip, rtol=0.02, atol=2e-3 * c)


def _uniform_film(nx, ny, nz, macro, spacing, direction):
    spec = single_grain_spec(0, nx, ny, nz, macro=macro, mu_s=3.23 * orc.MU_B, J=(0.0, 0.0, 0.0))
    o = orc.Oracle(spec)
    N = nx * ny * nz
    d = np.asarray(direction, float)
    o.set_spins(np.full(N, d[0]), np.full(N, d[1]), np.full(N, d[2]))
    o.enable_demag(spacing)
    return o


def test_p12_sum_rule_block_of_cells_is_one_big_cuboid():
    a = 0.3e-9
    macro, cells = (2, 3, 2), (4, 3, 2)
    nx, ny, nz = [m * c for m, c in zip(macro, cells)]
    big = [n * a for n in (nx, ny, nz)]
    Ms = 3.23 * orc.MU_B / a ** 3
    Nbig = orc.newell_tensor(big, (0, 0, 0))
    for axis in range(3):
        e = np.zeros(3); e[axis] = 1.0
        B = _uniform_film(nx, ny, nz, macro, (a, a, a), e).demag_cells()
        assert B.shape[:3] == (cells[0] + 1, cells[1], cells[2])            # one spare cell for unaligned windows
        mean = B[:cells[0]].reshape(-1, 3).mean(axis=0)
        want = -MU0 * Ms * np.array([Nbig[[0, 3, 4]], Nbig[[3, 1, 5]], Nbig[[4, 5, 2]]])[axis]
        assert np.allclose(mean, want, rtol=1e-9, atol=1e-12), (axis, mean, want)
        assert np.all(B[cells[0]:] == 0.0)


def test_p12_thin_film_limit():
    a = 0.3e-9
    nx = ny = 60; nz = 3
    Ms = 3.23 * orc.MU_B / a ** 3
    B = _uniform_film(nx, ny, nz, (3, 3, 3), (a, a, a), (0, 0, 1)).demag_cells()
    centre = B[10, 10, 0]
    assert abs(centre[2] / (-MU0 * Ms) - 1.0) < 0.05 and np.all(np.abs(centre[:2]) < 1e-6 * MU0 * Ms)
    B = _uniform_film(nx, ny, nz, (3, 3, 3), (a, a, a), (1, 0, 0)).demag_cells()
    assert abs(B[10, 10, 0][0]) < 0.04 * MU0 * Ms


def test_p12_field_enters_the_effective_field_and_the_step():
    """B_eff with demag - B_eff without = the cell field of the site's macrocell; partial cells use the full cell volume."""
    import asd_inputs as ai
    from tests.helpers import oracle_from_workload
    w = ai.small_film(ai.SC, 10, 12, 4, tilt_deg=40.0, macro=(3, 4, 2))
    w.x0 = 0
    o0, o1 = oracle_from_workload(w), oracle_from_workload(w)
    o1.enable_demag([a * 1e-9 for a in w.spacing_nm])
    cells = o1.demag_cells()
    d = (o1.field() - o0.field()).reshape(3, w.nx, w.nz, w.ny)
    mag = w.magnetic_mask().reshape(w.nx, w.nz, w.ny)
    for (i, k, j) in [(0, 0, 0), (4, 1, 5), (9, 3, 11), (3, 2, 8)]:
        if mag[i, k, j]:
            assert np.allclose(d[:, i, k, j], cells[i // 3, j // 4, k // 2], rtol=1e-12, atol=1e-15)
    assert np.abs(cells).max() > 1e-3                          # it is not nothing: ~0.1 T scale
    o0.step_heun(1); o1.step_heun(1)
    assert np.abs(o1.get_spins() - o0.get_spins()).max() > 1e-9


# ---------------------------------------------------------------------------------------------------------------
# Stray field of the frozen track (reading D4): pinned to the window demagnetising field above
# (itself pinned by P12) through the identity  "a window's own field + the field of everything outside it = the field
# of the whole track", with the whole track held by a second oracle whose window IS the track.
# ---------------------------------------------------------------------------------------------------------------
def _cellwise_track(track_nx, ny, nz, macro, seed):
    """A granular track whose spins are uniform inside every macrocell (one random direction per cell), so that a cell's
    mean spin describes any part of it exactly."""
    w = ai.small_film(ai.SC, track_nx, ny, nz, extra_track=0, macro=macro, pitch_nm=3.0, boundary_nm=0.6)
    rng = np.random.default_rng(seed)
    mx, my, mz = macro
    ncx, ncy, ncz = -(-track_nx // mx), -(-ny // my), -(-nz // mz)
    d = rng.standard_normal((ncx, ncy, ncz, 3)); d /= np.linalg.norm(d, axis=-1, keepdims=True)
    d = d.astype(np.float32).astype(np.float64)
    i, k, j = np.meshgrid(np.arange(track_nx), np.arange(nz), np.arange(ny), indexing="ij")
    S = np.moveaxis(d[i // mx, j // my, k // mz], -1, 0) * w.magnetic_mask()[None]
    return w, d, S                                            # S: [3, track_nx, nz, ny]


@pytest.mark.parametrize("start,shifts", [(0, (4, 6)), (4, (3, 5, 2)), (8, ())])
def test_d4_track_stray_field_completes_the_window_field_to_the_whole_track_field(start, shifts):
    track_nx, ny, nz, macro, nx = 40, 8, 4, (4, 4, 2), 12
    wt, d, S = _cellwise_track(track_nx, ny, nz, macro, seed=5)
    sp = [a * 1e-9 for a in wt.spacing_nm]
    whole = orc.from_workload(wt)
    whole.set_spins_f64(S.reshape(3, -1))
    whole.enable_demag(sp)
    B_full = whole.demag_cells()                              # [10, 2, 2, 3]
    # the window: the same track, 12 planes long, walked from `start` by the given shifts; after every shift its spins are
    # put back to the track's (a shift seeds the incoming planes at random), so what has left it is exactly the track
    import copy
    ww = copy.copy(wt)
    ww.nx, ww.x0 = nx, start
    plane = ny * nz
    for name in ("T", "Bx", "By", "Bz", "sx", "sy", "sz"):
        setattr(ww, name, getattr(wt, name)[:nx * plane].copy())
    o = orc.from_workload(ww)
    o.track_set_init(d.reshape(-1, 3).astype(np.float32))     # what lies ahead (and behind, where the window never was)
    x0 = start
    o.set_spins_f64(S[:, x0:x0 + nx].reshape(3, -1))
    for p in shifts:
        assert o.shift_window(p) == 0
        x0 += p
        o.set_spins_f64(S[:, x0:x0 + nx].reshape(3, -1))
    o.enable_demag(sp)
    assert o.enable_track_stray(True, 0) == 0
    own, stray = o.demag_cells(), o.stray_cells()
    c0 = x0 // macro[0]
    ncw = (x0 + nx - 1) // macro[0] - c0 + 1
    total = own[:ncw] + stray[:ncw]
    assert np.abs(stray[:ncw]).max() > 1e-3                   # tens of millitesla: not a small correction
    assert np.abs(total - B_full[c0:c0 + ncw]).max() < 1e-9 * max(1.0, np.abs(B_full).max()) + 1e-10
    assert not stray[ncw:].any()
    # a range that covers the track changes nothing; a short range drops the far cells (a smaller field, same sign structure)
    assert o.enable_track_stray(True, 10) == 0
    assert np.array_equal(o.stray_cells(), stray)
    assert o.enable_track_stray(True, 1) == 0
    near = o.stray_cells()
    assert 0.0 < np.abs(near - stray).max() < np.abs(stray).max()


def test_d4_stray_field_enters_the_effective_field_and_follows_the_window():
    track_nx, ny, nz, macro, nx = 40, 8, 4, (4, 4, 2), 12
    wt, d, S = _cellwise_track(track_nx, ny, nz, macro, seed=6)
    import copy
    ww = copy.copy(wt)
    ww.nx, ww.x0 = nx, 8
    plane = ny * nz
    for name in ("T", "Bx", "By", "Bz", "sx", "sy", "sz"):
        setattr(ww, name, getattr(wt, name)[:nx * plane].copy())
    sp = [a * 1e-9 for a in wt.spacing_nm]
    a, b = orc.from_workload(ww), orc.from_workload(ww)
    for o in (a, b):
        o.track_set_init(d.reshape(-1, 3).astype(np.float32))
        o.set_spins_f64(S[:, 8:20].reshape(3, -1))
        o.enable_demag(sp)
    assert orc.from_workload(ww).enable_track_stray(True, 0) == 4          # needs the demagnetising field's cells
    b.enable_track_stray(True, 0)
    # every site sees its cell's stray field on top of the rest of the effective field
    diff = (b.field() - a.field()).reshape(3, nx, nz, ny)
    st = b.stray_cells()
    i, k, j = np.meshgrid(np.arange(nx), np.arange(nz), np.arange(ny), indexing="ij")
    want = np.moveaxis(st[(8 + i) // macro[0] - 2, j // macro[1], k // macro[2]], -1, 0) * ww.magnetic_mask()[None]
    assert np.abs(diff - want).max() < 1e-12
    # ... in both Heun stages, and it is recomputed when the window moves
    a.step_heun(1); b.step_heun(1)
    assert np.abs(a.get_spins() - b.get_spins()).max() > 1e-9
    before = b.stray_cells().copy()
    b.shift_window(4)
    assert np.abs(b.stray_cells() - before).max() > 1e-6
