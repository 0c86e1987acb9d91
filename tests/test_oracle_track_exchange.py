"""Pins for reading E1 ("the ends of the simulation window are exchange coupled to the track"): the
neighbour spins beyond the first / last plane of a purely atomistic window are the frozen track's directions.

E1a  no surface: a uniformly magnetised single-grain window inside a uniformly magnetised track has, on its first and
     last plane, exactly the exchange field of its interior (full coordination); without the coupling those planes miss
     J (SC) or J1 + 2 J3 (L1_0).
E1b  definition: field(with) - field(without) is non-zero on the two end planes only and equals Eq. (2) over the
     neighbours beyond the window, written here from distances, the same-grain rule and the track cell lookup (written
     store behind the window, init state ahead of it), on a granular film after shifts.
"""
import math

import numpy as np
import pytest

import asd_inputs as ai
from oracle import asd_oracle as orc


@pytest.mark.parametrize("lattice", [ai.SC, ai.L10])
def test_e1a_uniform_window_in_a_uniform_track_has_no_surface(lattice):
    J = ai.workloads.J_SC if lattice == ai.SC else ai.workloads.J_L10
    nx, ny, nz = 6, 8, 4
    spec = orc.LatticeSpec(lattice=lattice, nx=nx, ny=ny, nz=nz, J=J, track_nx=nx + 8, x0=4, macro=(3, 3, 2),
                           grain_map=np.zeros((nx + 8, ny), dtype=np.int32), grain_ku=np.zeros(1),
                           grain_axis=np.array([[0.0, 0.0, 1.0]]))
    o = orc.Oracle(spec)
    N = nx * ny * nz
    o.set_spins(np.zeros(N), np.zeros(N), np.ones(N))
    mu_s = spec.mu_s
    missing = J[0] if lattice == ai.SC else J[0] + 2.0 * J[2]
    B = o.field().reshape(3, nx, nz, ny)
    inner = B[2, 2, 1, 3]
    assert abs(B[2, 0, 1, 3] - (inner - missing / mu_s)) < 1e-9 * inner        # open ends: one shell short
    o.enable_track_exchange(True)
    B = o.field().reshape(3, nx, nz, ny)
    assert abs(B[2, 0, 1, 3] - inner) < 1e-12 * inner and abs(B[2, nx - 1, 1, 3] - inner) < 1e-12 * inner
    assert np.allclose(B[2, 0], B[2, 2], rtol=1e-12) and np.allclose(B[2, nx - 1], B[2, 2], rtol=1e-12)
    o.step_heun(3)                                                              # ... and nothing moves
    assert np.array_equal(o.get_spins()[2], np.ones(N))


@pytest.mark.parametrize("lattice", [ai.SC, ai.L10])
def test_e1b_track_directions_stand_in_for_the_neighbours_beyond_the_window(lattice):
    w = ai.small_film(lattice, 14, 24, 5, extra_track=20, macro=(4, 5, 2), tilt_deg=25.0)
    a, b = orc.from_workload(w), orc.from_workload(w)
    rng = np.random.default_rng(12)
    ncx, ncy, ncz = a.track_dims()
    v = rng.standard_normal((ncx * ncy * ncz, 3)).astype(np.float32)
    for o in (a, b):
        o.track_set_init(v)
        o.shift_window(3); o.shift_window(4)                  # x0 = 7: unaligned; cells behind hold what was written
    S = a.get_spins()
    b.set_spins_f64(S)
    b.enable_track_exchange(True)
    d = (b.field() - a.field()).reshape(3, w.nx, w.nz, w.ny)
    assert not d[:, 1:-1].any()
    mean, cnt, sm = a.track_get()
    sm, cnt = sm.reshape(ncx, ncy, ncz, 3), cnt.reshape(ncx, ncy, ncz)
    init = v.astype(np.float64).reshape(ncx, ncy, ncz, 3)
    sp = np.asarray(w.spacing_nm)
    shells = [(sp[0], w.J[0])] if lattice == ai.SC else [(sp[0], w.J[0]), (math.hypot(sp[0], sp[1]), w.J[2])]
    x0 = 7
    mx, my, mz = w.macro
    for i, gxn in ((0, x0 - 1), (w.nx - 1, x0 + w.nx)):
        ref = np.zeros((3, w.nz, w.ny))
        for j in range(w.ny):
            g = w.grain_map[x0 + i, j]
            if g < 0:
                continue
            for dj in (-1, 0, 1):
                jj = j + dj
                if jj < 0 or jj >= w.ny or w.grain_map[gxn, jj] != g:
                    continue
                Jij = [Jv for (r, Jv) in shells if abs(r - math.hypot(sp[0], dj * sp[1])) < 1e-9]
                if not Jij:
                    continue
                for k in range(w.nz):
                    c = (gxn // mx, jj // my, k // mz)
                    vec = sm[c] if cnt[c] > 0 else init[c]
                    ref[:, k, j] += Jij[0] / w.mu_s * vec / np.linalg.norm(vec)
        assert np.abs(ref).max() > 1.0
        assert np.abs(d[:, i] - ref).max() < 1e-12 * np.abs(ref).max()
