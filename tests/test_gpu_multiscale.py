"""GPU parity for the multiscale window: micromagnetic meshes either side of
the atomistic mesh, through asd_mm_* and asd_step_heun / asd_shift_window, against the oracle."""
import numpy as np
import pytest

import asd_inputs as ai
import paper_2502_02236_b200 as asd
from tests.helpers import gpu_from_workload, oracle_from_workload

pytestmark = pytest.mark.gpu


def _pair(lattice, every=2, **kw):
    args = dict(atom_cells=4, mesh_cells=(3, 4), width_nm=7.2, nz=5, extra_cells=5, macro=(3, 4, 2), pitch_nm=3.0,
                boundary_nm=0.6, fwhm_nm=4.0, every=every, tilt_deg=20.0, dt=2e-16)
    args.update(kw)
    ms = ai.multiscale_film(lattice, **args)
    o, g = oracle_from_workload(ms.w), gpu_from_workload(ms.w)
    ai.apply_multiscale(o, ms)
    ai.apply_multiscale(g, ms)
    # tilted mesh directions, so that every term of the mesh field and both couplings are live
    rng = np.random.default_rng(21)
    for side in (0, 1):
        v = np.array([0.0, 0.0, 1.0]) + 0.35 * rng.standard_normal(o.mm_shape(side) + (3,))
        v = (v / np.linalg.norm(v, axis=-1, keepdims=True)).astype(np.float32)
        o.mm_set_m(side, v); g.mm_set_m(side, v)
    return ms, o, g


def _mesh_diff(o, g):
    return max(float(np.abs(o.mm_get_m(s) - g.mm_get_m(s)).max()) for s in (0, 1))


@pytest.mark.parametrize("lattice", [ai.SC, ai.L10])
def test_enable_initial_state_and_shapes(lattice):
    ms = ai.multiscale_film(lattice, atom_cells=4, mesh_cells=(3, 4), width_nm=7.2, nz=5, extra_cells=5,
                            macro=(3, 4, 2), pitch_nm=3.0, boundary_nm=0.6)
    o, g = oracle_from_workload(ms.w), gpu_from_workload(ms.w)
    rng = np.random.default_rng(2)
    init = rng.standard_normal((int(np.prod(o.track_dims())), 3)).astype(np.float32)
    o.track_set_init(init); g.track_set_init(init)
    ai.apply_multiscale(o, ms); ai.apply_multiscale(g, ms)
    for side in (0, 1):
        assert g.mm_shape(side) == o.mm_shape(side)
        a, b = o.mm_get_m(side), g.mm_get_m(side)
        assert np.abs(a - b).max() < 2e-7
        assert (np.linalg.norm(b, axis=-1) == 0).any()             # empty cells over the grain boundaries


@pytest.mark.parametrize("lattice", [ai.SC, ai.L10])
@pytest.mark.parametrize("kernel", ["general", "fast", "fused"])
def test_coupled_steps_match_the_oracle(lattice, kernel):
    ms, o, g = _pair(lattice, every=2)
    g.set_kernel({"general": asd.KERNEL_GENERAL, "fast": asd.KERNEL_FAST, "fused": asd.KERNEL_FUSED}[kernel])
    o.step_heun(1); g.step_heun(1)                                  # mesh step + boundary exchange + one Heun step
    assert np.abs(o.get_spins() - g.get_spins_host()).max() <= 1e-5
    assert _mesh_diff(o, g) <= 1e-5
    o.step_heun(4); g.step_heun(4)                                  # two more mesh steps, held data in between
    assert np.abs(o.get_spins() - g.get_spins_host()).max() <= 4e-5
    assert _mesh_diff(o, g) <= 2e-5
    # the coupling is live: without the meshes the boundary planes end up elsewhere
    plain = gpu_from_workload(ms.w)
    plain.set_kernel(asd.KERNEL_GENERAL)
    plain.step_heun(5)
    d = np.abs(plain.get_spins_host() - g.get_spins_host()).reshape(3, ms.w.nx, ms.w.nz, ms.w.ny)
    assert d[:, 0].max() > 1e-3 and d[:, -1].max() > 1e-3


@pytest.mark.parametrize("lattice", [ai.SC, ai.L10])
def test_field_scale_and_fields_reach_the_meshes(lattice):
    ms, o, g = _pair(lattice, every=1, t_peak=650.0)
    for sim in (o, g):
        sim.set_field_scale(-0.5)
    o.step_heun(3); g.step_heun(3)
    assert np.abs(o.get_spins() - g.get_spins_host()).max() <= 3e-5
    assert _mesh_diff(o, g) <= 1e-5


@pytest.mark.parametrize("lattice", [ai.SC, ai.L10])
def test_whole_cell_shift_matches_the_oracle(lattice):
    ms, o, g = _pair(lattice, every=2)
    w = ms.w
    rng = np.random.default_rng(6)
    init = (0.3 + 0.6 * rng.random((int(np.prod(o.track_dims())), 1))) * np.array([[0.28, -0.2, 0.94]])
    init = init.astype(np.float32)
    o.track_set_init(init); g.track_set_init(init)
    o.step_heun(2); g.step_heun(2)
    for pc in (1, 2):
        p = pc * w.macro[0]
        assert o.shift_window(p) == 0
        g.shift_window(p)
        assert g.counters() == o.counters()
        assert _mesh_diff(o, g) <= 1e-5
        assert np.abs(o.get_spins() - g.get_spins_host()).max() <= 3e-5
        _, cnt_o, sum_o = o.track_get()
        sum_g, cnt_g = g.track_get()
        assert np.array_equal(cnt_o, cnt_g)
        assert np.abs(sum_o - sum_g).max() <= 1e-4 * max(1, cnt_o.max())
        o.step_heun(3); g.step_heun(3)
        assert np.abs(o.get_spins() - g.get_spins_host()).max() <= 6e-5
        assert _mesh_diff(o, g) <= 3e-5


def test_error_paths():
    ms = ai.multiscale_film(ai.SC, atom_cells=4, mesh_cells=(3, 3), width_nm=7.2, nz=5, extra_cells=2,
                            macro=(3, 4, 2), pitch_nm=3.0, boundary_nm=0.6)
    g = gpu_from_workload(ms.w)
    with pytest.raises(asd.AsdError) as e:
        g.mm_set_m(0, np.zeros((3, 6, 3, 3), dtype=np.float32))
    assert e.value.status == 4                                        # not enabled
    with pytest.raises(asd.AsdError):
        g.mm_enable((4, 3), ms.every, ms.Ms0, ms.A0, ms.K0, ms.Tc, ms.cell_grain, ms.spacing_m)   # before the track
    ai.apply_multiscale(g, ms)
    for bad in (4, 12):                                               # not whole cells; longer than a mesh
        with pytest.raises(asd.AsdError) as e:
            g.shift_window(bad)
        assert e.value.status == 1
    with pytest.raises(asd.AsdError) as e:
        g.set_kernel(asd.KERNEL_TMA)
    assert e.value.status == 5
    with pytest.raises(asd.AsdError) as e:
        g.track_begin_pass(10)                                        # not on a whole cell
    assert e.value.status == 1
    g.shift_window(6)
    with pytest.raises(asd.AsdError) as e:
        g.shift_window(3)                                             # leading mesh would leave the track
    assert e.value.status == 4


@pytest.mark.parametrize("lattice", [ai.SC, ai.L10])
def test_passes_over_the_track_with_the_meshes(lattice):
    """asd_track_end_pass / asd_track_begin_pass on a multiscale window (readings T1', T2'): meshes and atoms to the track,
    then the next pass's window (atoms regenerated, meshes along the track) one cell further along."""
    ms, o, g = _pair(lattice, every=2, t_peak=450.0)
    w = ms.w
    o.step_heun(2); g.step_heun(2)
    assert o.shift_window(w.macro[0]) == 0
    g.shift_window(w.macro[0])
    o.step_heun(2); g.step_heun(2)
    assert o.track_end_pass() == 0
    g.track_end_pass()
    _, cnt_o, sum_o = o.track_get()
    sum_g, cnt_g = g.track_get()
    assert np.array_equal(cnt_o, cnt_g)
    assert np.abs(sum_o - sum_g).max() <= 1e-4 * max(1, cnt_o.max())
    x1 = w.x0 + 2 * w.macro[0]
    assert o.track_begin_pass(x1) == 0
    g.track_begin_pass(x1)
    assert g.counters() == o.counters()
    assert _mesh_diff(o, g) <= 2e-6
    assert np.abs(o.get_spins() - g.get_spins_host()).max() <= 3e-5
    o.step_heun(3); g.step_heun(3)
    assert np.abs(o.get_spins() - g.get_spins_host()).max() <= 6e-5
    assert _mesh_diff(o, g) <= 2e-5


def test_full_size_multiscale_window_one_coupled_step():
    """The bench's multiscale workload at full size ([48-cell mesh | SC 336 x 200 x 27 atoms | 48-cell mesh], 1.81 M sites,
    11 136 cells; the fused step's edge-field instance, as ASD_KERNEL_AUTO runs it): every site and every cell
    against the oracle after one coupled step, then after a whole-cell shift and one more step."""
    ms = ai.multiscale_film(ai.SC, every=1)
    o, g = oracle_from_workload(ms.w), gpu_from_workload(ms.w)
    ai.apply_multiscale(o, ms); ai.apply_multiscale(g, ms)
    rng = np.random.default_rng(3)
    for side in (0, 1):
        v = np.array([0.0, 0.0, 1.0]) + 0.3 * rng.standard_normal(o.mm_shape(side) + (3,))
        v = (v / np.linalg.norm(v, axis=-1, keepdims=True)).astype(np.float32)
        o.mm_set_m(side, v); g.mm_set_m(side, v)
    o.step_heun(1); g.step_heun(1)
    assert np.abs(o.get_spins() - g.get_spins_host()).max() <= 1e-5
    assert _mesh_diff(o, g) <= 1e-5
    assert o.shift_window(7) == 0
    g.shift_window(7)
    o.step_heun(1); g.step_heun(1)
    assert np.abs(o.get_spins() - g.get_spins_host()).max() <= 3e-5
    assert _mesh_diff(o, g) <= 2e-5


@pytest.mark.parametrize("lattice", [ai.SC, ai.L10])
@pytest.mark.parametrize("kernel", ["general", "fast", "fused", "auto"])
def test_multiscale_window_with_the_demagnetising_field(lattice, kernel):
    """Meshes and the window's demagnetising field together (general, film and -- held-field scheme -- fused kernels carry
    both): coupled steps against the oracle, per-stage and held-field schemes."""
    for every_dm in (0, 2, 1):
        if kernel == "fused" and every_dm == 0:
            continue                                                # the one-kernel step takes the held field only
        ms, o, g = _pair(lattice, every=2)
        sp = [a * 1e-9 for a in ms.w.spacing_nm]
        o.enable_demag(sp); g.enable_demag(sp)
        o.set_demag_every(every_dm); g.set_demag_every(every_dm)
        if kernel != "auto":
            g.set_kernel({"general": asd.KERNEL_GENERAL, "fast": asd.KERNEL_FAST, "fused": asd.KERNEL_FUSED}[kernel])
        o.step_heun(1); g.step_heun(1)
        assert np.abs(o.get_spins() - g.get_spins_host()).max() <= 1e-5
        o.step_heun(3); g.step_heun(3)
        assert np.abs(o.get_spins() - g.get_spins_host()).max() <= 4e-5
        assert _mesh_diff(o, g) <= 2e-5
