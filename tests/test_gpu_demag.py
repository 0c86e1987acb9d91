"""GPU parity of the demagnetising field (csrc/asd_demag.cu) against the oracle's Eq. (6)-(7) (pinned by P12):
the per-macrocell field itself (FFT convolution vs the oracle's direct sum) and Heun steps with the field on, for both
lattices, the film and the general kernel, a window whose origin is not aligned with the macrocells, and across a shift."""
import numpy as np
import pytest

import asd_inputs as ai
from tests.helpers import gpu_from_workload, max_abs_diff, oracle_from_workload

pytestmark = pytest.mark.gpu


def _film(lattice, nx, ny, nz, macro, x0, tilt, **kw):
    """small_film whose window starts at global plane x0 (spins re-masked for the columns it then covers)."""
    w = ai.small_film(lattice, nx, ny, nz, extra_track=8, macro=macro, **kw)
    w.x0 = x0
    sx, sy, sz = ai.tilted_spins(w.n_sites, tilt, seed=21)
    mag = w.magnetic_mask().reshape(-1)
    w.sx, w.sy, w.sz = (sx * mag).astype(np.float32), (sy * mag).astype(np.float32), (sz * mag).astype(np.float32)
    return w


def _pair(w):
    sp = [a * 1e-9 for a in w.spacing_nm]
    o, g = oracle_from_workload(w), gpu_from_workload(w)
    o.enable_demag(sp); g.enable_demag(sp)
    return o, g


@pytest.mark.parametrize("lattice", [ai.SC, ai.L10])
@pytest.mark.parametrize("dims,macro,x0", [((24, 28, 6), (3, 3, 3), 0), ((21, 40, 7), (4, 5, 2), 2), ((40, 132, 9), (7, 7, 5), 5)])
def test_cell_field_matches_oracle(lattice, dims, macro, x0):
    nx, ny, nz = dims
    w = _film(lattice, nx, ny, nz, macro, x0, 35.0)
    o, g = _pair(w)
    Bo, Bg = o.demag_cells(), g.demag_field()
    assert Bo.shape == Bg.shape
    scale = np.abs(Bo).max()
    assert scale > 1e-3                                            # Tesla: a real field, not zeros
    assert np.abs(Bg - Bo).max() <= 2e-6 * max(scale, 1.0) + 1e-7  # fp32 FFT convolution vs fp64 direct sum


@pytest.mark.parametrize("lattice", [ai.SC, ai.L10])
@pytest.mark.parametrize("kernel", ["general", "fast"])
def test_heun_steps_with_demag(lattice, kernel):
    import paper_2502_02236_b200 as asd
    w = _film(lattice, 24, 40, 6, (4, 5, 2), 1, 25.0, dt=1e-16)
    o, g = _pair(w)
    g.set_kernel({"general": asd.KERNEL_GENERAL, "fast": asd.KERNEL_FAST}[kernel])
    o.step_heun(1); g.step_heun(1)
    assert max_abs_diff(g, o) <= 1e-5
    o.step_heun(3); g.step_heun(3)
    assert max_abs_diff(g, o) <= 5e-5
    o.shift_window(3); g.shift_window(3)                           # window origin moves: other cells, other alignment
    assert np.abs(g.demag_field() - o.demag_cells()).max() <= 5e-6
    o.step_heun(2); g.step_heun(2)
    assert max_abs_diff(g, o) <= 1e-4


@pytest.mark.parametrize("lattice", [ai.SC, ai.L10])
@pytest.mark.parametrize("every", [1, 3])
def test_fused_step_with_the_held_field(lattice, every):
    """The one-kernel Heun step takes the demagnetising field in the held-field scheme (the field of S serves both
    stages): same tolerances as the stage kernels; the per-stage scheme is refused."""
    import paper_2502_02236_b200 as asd
    w = _film(lattice, 24, 40, 6, (4, 5, 2), 1, 25.0, dt=1e-16)
    o, g = _pair(w)
    with pytest.raises(asd.AsdError):
        g.set_kernel(asd.KERNEL_FUSED)                               # per-stage scheme: the field of S~ is a global quantity
    o.set_demag_every(every); g.set_demag_every(every)
    g.set_kernel(asd.KERNEL_FUSED)
    o.step_heun(1); g.step_heun(1)
    assert max_abs_diff(g, o) <= 1e-5
    o.step_heun(4); g.step_heun(4)
    assert max_abs_diff(g, o) <= 5e-5
    o.shift_window(3); g.shift_window(3)
    o.step_heun(2); g.step_heun(2)
    assert max_abs_diff(g, o) <= 1e-4
    # and it is the stage kernels' held-field result up to rounding
    h = gpu_from_workload(w)
    h.enable_demag([a * 1e-9 for a in w.spacing_nm]); h.set_demag_every(every); h.set_kernel(asd.KERNEL_FAST)
    h.step_heun(5); h.shift_window(3); h.step_heun(2)
    assert np.abs(h.get_spins_host() - g.get_spins_host()).max() <= 2e-5


@pytest.mark.parametrize("lattice", [ai.SC, ai.L10])
@pytest.mark.parametrize("dims,macro,x0,every", [((24, 40, 6), (4, 5, 2), 1, 1), ((40, 132, 9), (7, 7, 5), 5, 1),
                                                 ((21, 40, 7), (4, 5, 2), 2, 2), ((36, 64, 8), (1, 3, 1), 0, 1),
                                                 ((30, 36, 5), (9, 4, 5), 4, 3)])
def test_cell_sums_from_the_fused_corrector(lattice, dims, macro, x0, every):
    """Eq. (6) behind a refresh of the held field is accumulated by the corrector of the fused step before it (integer
    cell sums): the field the next step holds is the oracle's field of those spins, and the film kernel's (whose cell
    sums come from a pass of their own), before and after a shift that leaves stale sums behind."""
    import paper_2502_02236_b200 as asd
    nx, ny, nz = dims
    w = _film(lattice, nx, ny, nz, macro, x0, 30.0, dt=1e-16)
    o, g = _pair(w)
    h = gpu_from_workload(w); h.enable_demag([a * 1e-9 for a in w.spacing_nm])
    for c in (o, g, h):
        c.set_demag_every(every)
    g.set_kernel(asd.KERNEL_FUSED); h.set_kernel(asd.KERNEL_FAST)
    n = 2 * every + 1                                               # steps 1, every + 1, 2 every + 1 refresh
    for leg in range(2):
        o.step_heun(n - 1)
        Bo = o.demag_cells()                                        # field of the spins step n starts from
        o.step_heun(1)
        g.step_heun(n); h.step_heun(n)
        Bg, Bh = g.demag_held_field(), h.demag_held_field()
        scale = np.abs(Bo).max()
        assert scale > 1e-3
        assert np.abs(Bg - Bo).max() <= 1e-4 * scale                # spins differ by <= 5e-5 by then
        assert np.abs(Bg - Bh).max() <= 3e-5 * scale
        assert max_abs_diff(g, o) <= 1e-4
        if leg == 0:
            if every > 1:                                           # end on a step that armed the sums
                g.step_heun(every - 1); h.step_heun(every - 1); o.step_heun(every - 1)
            assert o.shift_window(3) == 0
            g.shift_window(3); h.shift_window(3)


@pytest.mark.parametrize("every", [1, 3])
def test_held_field_update_period(every):
    """asd_set_demag_every(P): field from S at every P-th step, held for both stages in between; a shift re-arms it."""
    w = _film(ai.L10, 24, 40, 6, (4, 5, 2), 1, 25.0, dt=1e-16)
    o, g = _pair(w)
    o.set_demag_every(every); g.set_demag_every(every)
    o.step_heun(4); g.step_heun(4)
    assert max_abs_diff(g, o) <= 5e-5
    o.shift_window(2); g.shift_window(2)
    o.step_heun(2); g.step_heun(2)
    assert max_abs_diff(g, o) <= 1e-4
    # and it is a different scheme from the per-stage default (the corrector sees B_d(S), not B_d(S~))
    o2, _g2 = _pair(w)
    o2.step_heun(4)
    o3, _g3 = _pair(w); o3.set_demag_every(every); o3.step_heun(4)
    assert np.abs(o2.get_spins() - o3.get_spins()).max() > 0.0


def test_demag_changes_the_dynamics_and_tma_is_refused():
    import paper_2502_02236_b200 as asd
    w = ai.small_film(ai.SC, 24, 40, 6, tilt_deg=25.0, dt=1e-15)
    a, b = gpu_from_workload(w), gpu_from_workload(w)
    b.enable_demag([x * 1e-9 for x in w.spacing_nm])
    a.step_heun(5); b.step_heun(5)
    assert np.abs(a.get_spins_host() - b.get_spins_host()).max() > 1e-7
    b.set_kernel(asd.KERNEL_TMA)
    with pytest.raises(asd.AsdError):
        b.step_heun(1)


# ---- stray field of the frozen track (reading D4) ----
def _stray_pair(lattice, x0=3, **kw):
    """A window in the middle of a longer track with a non-trivial track state on both sides: what lies ahead is a random
    mean spin per cell, what lies behind has been written by two shifts."""
    w = ai.small_film(lattice, 21, 40, 6, extra_track=30, macro=(4, 5, 2), tilt_deg=30.0, dt=1e-16, **kw)
    w.x0 = x0
    sx, sy, sz = ai.tilted_spins(w.n_sites, 30.0, seed=23)
    mag = w.magnetic_mask().reshape(-1)
    w.sx, w.sy, w.sz = (sx * mag).astype(np.float32), (sy * mag).astype(np.float32), (sz * mag).astype(np.float32)
    o, g = _pair(w)
    rng = np.random.default_rng(31)
    ncell = int(np.prod(o.track_dims()))
    v = rng.standard_normal((ncell, 3)); v *= rng.uniform(0.5, 1.0, (ncell, 1)) / np.linalg.norm(v, axis=1, keepdims=True)
    v = v.astype(np.float32)
    o.track_set_init(v); g.track_set_init(v)
    for p in (3, 4):
        assert o.shift_window(p) == 0
        g.shift_window(p)
    return w, o, g


@pytest.mark.parametrize("lattice", [ai.SC, ai.L10])
@pytest.mark.parametrize("rng_cells", [0, 3])
def test_track_stray_field_matches_oracle(lattice, rng_cells):
    w, o, g = _stray_pair(lattice)
    assert o.enable_track_stray(True, rng_cells) == 0
    g.enable_track_stray(True, rng_cells)
    Bo, Bg = o.stray_cells(), g.stray_cells()
    scale = np.abs(Bo).max()
    assert scale > 1e-3
    assert np.abs(Bg - Bo).max() <= 3e-6 * max(scale, 1.0) + 1e-7
    # the total cell field the kernels add = own demagnetising field + the track's
    tot = g.demag_field()
    assert np.abs(tot - (o.demag_cells() + Bo)).max() <= 5e-6 * max(scale, 1.0) + 2e-7
    # recomputed when the window moves and when the track state changes
    assert o.shift_window(2) == 0
    g.shift_window(2)
    assert np.abs(g.stray_cells() - o.stray_cells()).max() <= 3e-6 * max(scale, 1.0) + 1e-7
    o.track_set_init(None, 0.7); g.track_set_init(None, 0.7)
    Bo2 = o.stray_cells()
    assert np.abs(Bo2 - Bo).max() > 1e-4
    assert np.abs(g.stray_cells() - Bo2).max() <= 3e-6 * max(scale, 1.0) + 1e-7


@pytest.mark.parametrize("lattice", [ai.SC, ai.L10])
@pytest.mark.parametrize("kernel,every", [("general", 0), ("fast", 0), ("fast", 2), ("fused", 1)])
def test_heun_steps_with_the_track_stray_field(lattice, kernel, every):
    import paper_2502_02236_b200 as asd
    w, o, g = _stray_pair(lattice)
    o.enable_track_stray(True, 0); g.enable_track_stray(True, 0)
    o.set_demag_every(every); g.set_demag_every(every)
    g.set_kernel({"general": asd.KERNEL_GENERAL, "fast": asd.KERNEL_FAST, "fused": asd.KERNEL_FUSED}[kernel])
    o.step_heun(1); g.step_heun(1)
    assert max_abs_diff(g, o) <= 1e-5
    o.step_heun(3); g.step_heun(3)
    assert max_abs_diff(g, o) <= 5e-5
    o.shift_window(3); g.shift_window(3)
    o.step_heun(2); g.step_heun(2)
    assert max_abs_diff(g, o) <= 1e-4


def test_track_stray_needs_demag():
    import paper_2502_02236_b200 as asd
    w = ai.small_film(ai.SC, 12, 16, 4, extra_track=8)
    g = gpu_from_workload(w)
    with pytest.raises(asd.AsdError) as e:
        g.demag_held_field()
    assert e.value.status == 4
    with pytest.raises(asd.AsdError) as e:
        g.enable_track_stray(True, 0)
    assert e.value.status == 4
