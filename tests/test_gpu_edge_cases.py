"""GPU parity on the degenerate cases of the method: no steps, no magnetic sites, no damping, no torque, a window
that is replaced whole by one shift, the thinnest and narrowest lattices -- each against the fp64 oracle on the same
inputs, on every kernel variant that takes the lattice (a variant that does not says so with ASD_EUNSUPPORTED)."""
import dataclasses

import numpy as np
import pytest

import asd_inputs as ai
import paper_2502_02236_b200 as asd
from tests.helpers import gpu_from_workload, max_abs_diff, oracle_from_workload

pytestmark = pytest.mark.gpu

KERNELS = {"auto": asd.KERNEL_AUTO, "general": asd.KERNEL_GENERAL, "fast": asd.KERNEL_FAST, "tma": asd.KERNEL_TMA,
           "fused": asd.KERNEL_FUSED, "persistent": asd.KERNEL_PERSISTENT}


def _ctx(w, kernel):
    """Context on kernel variant `kernel`, or None where the variant does not take this lattice."""
    g = gpu_from_workload(w)
    try:
        g.set_kernel(KERNELS[kernel])
        g.step_heun(0)
    except asd.AsdError as e:
        assert e.status in (1, 4, 5), e          # EINVAL / EUNSUPPORTED / ESTATE: refused, not failed
        return None
    return g


def _step_or_skip(g, n):
    try:
        g.step_heun(n)
    except asd.AsdError as e:
        assert "UNSUPPORTED" in str(e) or e.status in (4, 5), e
        pytest.skip("variant does not take this lattice")


@pytest.mark.parametrize("kernel", list(KERNELS))
def test_zero_steps_change_nothing(kernel):
    w = ai.small_film(ai.L10, 12, 16, 4, tilt_deg=20.0)
    g = _ctx(w, kernel)
    if g is None:
        pytest.skip("variant does not take this lattice")
    before, c0, l0 = g.get_spins_host(), g.counters(), g.launch_count()      # (reading the spins back launches a kernel)
    g.step_heun(0)
    assert g.launch_count() == l0 and g.counters() == c0
    assert np.array_equal(g.get_spins_host(), before)


@pytest.mark.parametrize("kernel", list(KERNELS))
@pytest.mark.parametrize("lattice", [ai.SC, ai.L10])
def test_a_window_without_magnetic_sites(lattice, kernel):
    """Every column vacant: zeros stay exact zeros through steps and a shift, and the magnetisation of nothing is 0."""
    w = ai.small_film(lattice, 10, 12, 3, extra_track=6)
    w = dataclasses.replace(w, grain_map=np.full_like(w.grain_map, -1), sx=np.zeros_like(w.sx), sy=np.zeros_like(w.sy),
                            sz=np.zeros_like(w.sz))
    g = _ctx(w, kernel)
    if g is None:
        pytest.skip("variant does not take this lattice")
    _step_or_skip(g, 3)
    assert not g.get_spins_host().any()
    m, n = g.magnetisation()
    assert n == 0 and np.array_equal(m, np.zeros(3))
    assert not np.isnan(g.grain_magnetisation()).any()
    g.shift_window(2)
    _step_or_skip(g, 1)
    assert not g.get_spins_host().any()
    o = oracle_from_workload(w)
    o.step_heun(3); o.shift_window(2); o.step_heun(1)
    assert not o.get_spins().any()


@pytest.mark.parametrize("kernel", list(KERNELS))
@pytest.mark.parametrize("lattice", [ai.SC, ai.L10])
def test_no_damping(lattice, kernel):
    """lambda = 0: Eq. (1) is pure precession and the thermal field vanishes with it (sigma ~ sqrt(lambda))."""
    w = dataclasses.replace(ai.small_film(lattice, 9, 12, 4, tilt_deg=30.0, dt=1e-16), lam=0.0)
    o, g = oracle_from_workload(w), _ctx(w, kernel)
    if g is None:
        pytest.skip("variant does not take this lattice")
    o.step_heun(1); _step_or_skip(g, 1)
    assert max_abs_diff(g, o) <= 1e-5
    o.step_heun(9); g.step_heun(9)
    assert max_abs_diff(g, o) <= 5e-5


@pytest.mark.parametrize("kernel", list(KERNELS))
def test_a_stationary_state_stays_put(kernel):
    """T = 0, a granular film magnetised along its grains' common easy axis and the field: S x B = 0 at every site, the torque is
    zero and 200 steps must leave every spin where it was (to the rounding of the renormalisation)."""
    w = ai.small_film(ai.SC, 12, 16, 4, uniform_T=0.0, spot=False, tilt_deg=0.0)
    mag = w.magnetic_mask().reshape(-1).astype(np.float32)
    w = dataclasses.replace(w, grain_axis=np.tile(np.array([[0.0, 0.0, 1.0]], np.float32), (w.n_grains, 1)),
                            sx=np.zeros_like(w.sx), sy=np.zeros_like(w.sy), sz=mag, Bx=np.zeros_like(w.Bx),
                            By=np.zeros_like(w.By))
    o, g = oracle_from_workload(w), _ctx(w, kernel)
    if g is None:
        pytest.skip("variant does not take this lattice")
    o.step_heun(200); _step_or_skip(g, 200)
    s = g.get_spins_host()
    assert np.abs(s[2] - mag).max() <= 2e-7 and np.abs(s[:2]).max() <= 1e-7
    assert max_abs_diff(g, o) <= 2e-7


@pytest.mark.parametrize("lattice", [ai.SC, ai.L10])
def test_a_shift_that_replaces_the_whole_window(lattice):
    """p = nx: nothing is moved, every plane goes to the track and every plane is seeded from it."""
    nx, ny, nz = 8, 12, 4
    w = ai.small_film(lattice, nx, ny, nz, extra_track=2 * nx, macro=(4, 4, 2), tilt_deg=15.0)
    o, g = oracle_from_workload(w), gpu_from_workload(w)
    o.step_heun(2); g.step_heun(2)
    assert o.shift_window(nx) == 0
    g.shift_window(nx)
    assert g.counters()["x0"] == o.counters()["x0"] == w.x0 + nx
    _, cnt_o, sum_o = o.track_get()
    sum_g, cnt_g = g.track_get()
    assert np.array_equal(cnt_o, cnt_g)
    assert np.abs(sum_o - sum_g).max() <= 1e-4 * max(1.0, np.abs(sum_o).max())
    assert max_abs_diff(g, o) <= 3e-5                      # every site is a seeded one (cone sampling)
    o.step_heun(1); g.step_heun(1)
    assert max_abs_diff(g, o) <= 5e-5
    with pytest.raises(asd.AsdError):
        g.shift_window(nx + 1)                             # more planes than the window has


@pytest.mark.parametrize("dims", [(1, 4, 1), (2, 4, 1), (1, 1, 1), (5, 1, 2), (3, 5, 1)])
@pytest.mark.parametrize("lattice", [ai.SC, ai.L10])
def test_the_thinnest_and_narrowest_lattices(lattice, dims):
    """One plane, one row, one layer, one site: every missing neighbour is an open boundary of Eq. (2)."""
    nx, ny, nz = dims
    w = ai.small_film(lattice, nx, ny, nz, boundary_nm=0.0, tilt_deg=40.0, dt=1e-16)
    o, g = oracle_from_workload(w), gpu_from_workload(w)
    o.step_heun(1); g.step_heun(1)
    assert max_abs_diff(g, o) <= 1e-5
    o.step_heun(5); g.step_heun(5)
    assert max_abs_diff(g, o) <= 5e-5
