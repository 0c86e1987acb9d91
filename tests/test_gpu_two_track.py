"""GPU parity for the passes over the track and the read-back scan (
DESIGN.md sec. 13): asd_track_end_pass / asd_track_begin_pass / asd_track_read_scan against the oracle, then the whole
two-track workload (two passes through asd_inputs.drive_pass) on both sides."""
import numpy as np
import pytest

import asd_inputs as ai
from tests.helpers import gpu_from_workload, oracle_from_workload

pytestmark = pytest.mark.gpu


def _integer_valued(w):
    N = w.n_sites
    g = np.arange(N, dtype=np.int64)
    mag = w.magnetic_mask().reshape(-1)
    w.sx = ((g % 4093) * mag).astype(np.float32)
    w.sy = ((g // 4093) * mag).astype(np.float32)
    w.sz = ((g % 977 + 1) * mag).astype(np.float32)
    return w


@pytest.mark.parametrize("lattice,dims,macro", [(ai.SC, (24, 20, 9), (7, 7, 7)), (ai.L10, (19, 28, 7), (7, 7, 5)),
                                                (ai.SC, (10, 12, 4), (3, 2, 3))])
def test_end_pass_store_bit_exact_and_scan(lattice, dims, macro):
    nx, ny, nz = dims
    w = _integer_valued(ai.small_film(lattice, nx, ny, nz, extra_track=30, macro=macro))
    o, g = oracle_from_workload(w), gpu_from_workload(w)
    for p in (3, 4):
        o.shift_window(p); g.shift_window(p)
    assert o.track_end_pass() == 0
    g.track_end_pass()
    _, cnt_o, sum_o = o.track_get()
    sum_g, cnt_g = g.track_get()
    assert np.array_equal(cnt_o, cnt_g) and np.array_equal(sum_o, sum_g)
    # the scan of identical stores: only the order of the fp64 sums differs
    for (y, sx, sy) in ((ny / 3.0, 4.0, 3.0), (0.8 * ny, 9.5, 1.7)):
        a = o.track_read_scan(y, sx, sy, -2.0, 0.75, 57)
        b = g.track_read_scan(y, sx, sy, -2.0, 0.75, 57)
        assert np.abs(a - b).max() <= 1e-12 * np.abs(a).max()
    # integer-valued sums have |mean| >= 1 => m = 1: the regenerated window lies exactly along the cell means
    assert o.track_begin_pass(5) == 0
    g.track_begin_pass(5)
    assert g.counters() == o.counters()
    so, sg = o.get_spins(), g.get_spins_host().astype(np.float64)
    assert np.abs(so - sg).max() < 3e-6
    sum_g, cnt_g = g.track_get()
    assert not sum_g.any() and not cnt_g.any()


def test_begin_pass_regenerates_the_window_from_a_written_track():
    """Real spins: flush, commit, regenerate.  theta_max of a written cell is taken from an fp32 mean on the device and
    an fp64 one in the oracle: 3e-5 covers d(theta_max)/dm at the m = 0.9-0.99 of a thermal film."""
    w = ai.small_film(ai.L10, 20, 24, 6, extra_track=12, macro=(4, 4, 3), tilt_deg=25.0, dt=1e-16)
    o, g = oracle_from_workload(w), gpu_from_workload(w)
    o.step_heun(2); g.step_heun(2)
    o.shift_window(3); g.shift_window(3)
    assert o.track_end_pass() == 0
    g.track_end_pass()
    _, cnt_o, sum_o = o.track_get()
    sum_g, cnt_g = g.track_get()
    assert np.array_equal(cnt_o, cnt_g)
    assert np.abs(sum_o - sum_g).max() < 1e-4
    for x0 in (0, 7):
        assert o.track_begin_pass(x0) == 0
        g.track_begin_pass(x0)
        assert np.abs(o.get_spins() - g.get_spins_host()).max() < 3e-5
    assert g.counters()["pass"] == 2
    # and the dynamics go on from there
    o.step_heun(1); g.step_heun(1)
    assert np.abs(o.get_spins() - g.get_spins_host()).max() < 4e-5


def test_error_paths():
    import paper_2502_02236_b200 as asd
    w = ai.small_film(ai.SC, 8, 8, 3, extra_track=4)
    g = gpu_from_workload(w)
    for bad in (-1, 5):
        with pytest.raises(asd.AsdError) as e:
            g.track_begin_pass(bad)
        assert e.value.status == 1
    with pytest.raises(asd.AsdError):
        g.track_read_scan(1.0, 0.0, 1.0, 0.0, 1.0, 4)
    g.track_begin_pass(4)                                   # the last admissible origin
    assert g.counters()["x0"] == 4


@pytest.mark.parametrize("lattice", [ai.SC, ai.L10])
def test_two_track_workload_two_passes(lattice):
    """The whole second workload at a size the oracle finishes in seconds: pass 0 with the spot on the bottom track,
    pass 1 started from the written track with the spot on the top track.  Few Heun steps per shift period (thermal
    trajectories of the two precisions separate after ~1e2 steps, Q18), so spins, track store and read-back
    are compared directly."""
    tt = ai.two_track_film(lattice, length_nm=7.2, width_nm=10.8, nz=4, n_bits=2, bit_nm=2.4, separation_nm=2.0,
                           bit_width_nm=3.4, pitch_nm=3.0, boundary_nm=0.6, shift_every=2, batch=2,
                           macro=(3, 3, 2), dt=1e-16, t_peak=500.0)
    w = tt.w
    o, g = oracle_from_workload(w), gpu_from_workload(w)
    up_o = lambda sim, T: sim.set_fields(T=T)
    up_g = lambda sim, T: sim.set_fields_host(T=T)
    for p in (0, 1):
        n_o = ai.drive_pass(o, tt, p, up_o)
        n_g = ai.drive_pass(g, tt, p, up_g)
        assert n_o == n_g and g.counters() == o.counters()
        assert np.abs(o.get_spins() - g.get_spins_host()).max() < 1e-4
        _, cnt_o, sum_o = o.track_get()
        sum_g, cnt_g = g.track_get()
        assert np.array_equal(cnt_o, cnt_g)
        assert np.abs(sum_o - sum_g).max() < 2e-3            # sums over <= 18 sites of spins that agree to 1e-4
        ro, rg = ai.read_tracks(o, tt), ai.read_tracks(g, tt)
        assert ro.shape == (2, 2) and np.abs(ro - rg).max() < 1e-4
    assert o.counters()["pass"] == 1


def test_full_size_two_track_window_flush_and_scan():
    """The two-track window at the demo's size (SC 400 x 268 x 27, 2.89 M sites; macrocells (7, 7, 7)): a shift, the flush
    of the whole window, the committed track and the read-back scan against the oracle -- store bit-exact on
    integer-valued spins, scan to 1e-12, regenerated window to 3e-6."""
    tt = ai.two_track_film(ai.SC, n_bits=2)
    w = _integer_valued(tt.w)
    o, g = oracle_from_workload(w), gpu_from_workload(w)
    o.shift_window(3); g.shift_window(3)
    assert o.track_end_pass() == 0
    g.track_end_pass()
    _, cnt_o, sum_o = o.track_get()
    sum_g, cnt_g = g.track_get()
    assert np.array_equal(cnt_o, cnt_g) and np.array_equal(sum_o, sum_g)
    c = tt.bit_centres()
    for y in tt.track_y:
        a = o.track_read_scan(y, tt.reader_sigma[0], tt.reader_sigma[1], float(c[0]), 5.0, 40)
        b = g.track_read_scan(y, tt.reader_sigma[0], tt.reader_sigma[1], float(c[0]), 5.0, 40)
        assert np.abs(a - b).max() <= 1e-12 * np.abs(a).max()
    assert o.track_begin_pass(0) == 0
    g.track_begin_pass(0)
    assert np.abs(o.get_spins() - g.get_spins_host()).max() <= 3e-6
