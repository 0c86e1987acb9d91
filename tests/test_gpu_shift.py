"""GPU parity for asd_shift_window: indexing bit-exact, seeded slab against the oracle."""
import numpy as np
import pytest

import asd_inputs as ai
from tests.helpers import gpu_from_workload, oracle_from_workload

pytestmark = pytest.mark.gpu


def _integer_valued(w):
    """Spins replaced by integers that encode the global site id: sums and moves are exact in fp32/fp64."""
    N = w.n_sites
    g = np.arange(N, dtype=np.int64)
    mag = w.magnetic_mask().reshape(-1)
    w.sx = ((g % 4093) * mag).astype(np.float32)
    w.sy = ((g // 4093) * mag).astype(np.float32)
    w.sz = ((g % 977 + 1) * mag).astype(np.float32)
    return w


@pytest.mark.parametrize("lattice,dims,macro", [(ai.SC, (24, 20, 9), (7, 7, 7)), (ai.L10, (19, 28, 7), (7, 7, 5)),
                                                (ai.SC, (10, 9, 4), (3, 2, 3))])
def test_shift_indexing_bit_exact(lattice, dims, macro):
    nx, ny, nz = dims
    w = _integer_valued(ai.small_film(lattice, nx, ny, nz, extra_track=30, macro=macro))
    o, g = oracle_from_workload(w), gpu_from_workload(w)
    keep = None
    for p in (3, 4, 1, 7, 2):
        before = g.get_spins_host()
        assert o.shift_window(p) == 0
        g.shift_window(p)
        so, sg = o.get_spins(), g.get_spins_host()
        nkeep = (nx - p) * ny * nz
        # moved block: exactly the old spins p planes ahead, where the new column is... the move itself is unmasked
        assert np.array_equal(sg[:, :nkeep], before[:, p * ny * nz:])
        assert np.array_equal(sg[:, :nkeep].astype(np.float64), so[:, :nkeep])
        # macrocell sums and counts exact
        _, cnt_o, sum_o = o.track_get()
        sum_g, cnt_g = g.track_get()
        assert np.array_equal(cnt_o, cnt_g)
        assert np.array_equal(sum_o, sum_g)
        assert g.counters()["x0"] == o.counters()["x0"]
    assert g.counters()["shift"] == 5


def test_seeded_slab_matches_oracle_and_reproduces_m():
    nx, ny, nz = 16, 24, 8
    w = ai.small_film(ai.SC, nx, ny, nz, extra_track=40, macro=(4, 4, 4))
    o, g = oracle_from_workload(w), gpu_from_workload(w)
    ncx, ncy, ncz = g.track_dims()
    assert (ncx, ncy, ncz) == o.track_dims()
    rng = np.random.default_rng(8)
    v = rng.standard_normal((ncx * ncy * ncz, 3))
    v /= np.linalg.norm(v, axis=1, keepdims=True)
    v *= rng.uniform(0.0, 1.0, size=(v.shape[0], 1))
    v[0] = 0.0                          # degenerate: no direction -> z, theta_max = pi
    v[1] = (1.0, 0.0, 0.0)              # along x: the other frame branch, m = 1 -> exactly n
    v = v.astype(np.float32)
    o.track_set_init(v); g.track_set_init(v)
    for p in (5, 16, 3):
        assert o.shift_window(p) == 0
        g.shift_window(p)
        so, sg = o.get_spins(), g.get_spins_host().astype(np.float64)
        assert np.abs(so - sg).max() < 3e-6
    # default track state: m0 = 1 along +z -> incoming magnetic spins are exactly +z
    o.track_set_init(None, 1.0); g.track_set_init(None, 1.0)
    o.shift_window(6); g.shift_window(6)
    sg = g.get_spins_host()
    tail = sg[:, (nx - 6) * ny * nz:]
    magt = np.abs(tail).sum(axis=0) > 0
    assert np.array_equal(tail[2][magt], np.ones(magt.sum(), dtype=np.float32))
    assert np.all(tail[0] == 0) and np.all(tail[1] == 0)


def test_full_size_cfg4_shift():
    """asd_shift_window at BASELINE cfg4's size (881 x 220 x 27 L1_0, 220 x 27-site planes, macrocells (7, 7, 5)) with the
    schedule's plane counts (p = 3 then 4) and a non-trivial track state: moved block, macrocell sums and counts bit
    exact on integer-valued spins; seeded slabs against the oracle on real spins."""
    w = _integer_valued(ai.make_config(4))
    nx, ny, nz = w.nx, w.ny, w.nz
    o, g = oracle_from_workload(w), gpu_from_workload(w)
    for p in (3, 4):
        before = g.get_spins_host()
        assert o.shift_window(p) == 0
        g.shift_window(p)
        so, sg = o.get_spins(), g.get_spins_host()
        nkeep = (nx - p) * ny * nz
        assert np.array_equal(sg[:, :nkeep], before[:, p * ny * nz:])
        assert np.array_equal(sg[:, :nkeep].astype(np.float64), so[:, :nkeep])
        _, cnt_o, sum_o = o.track_get()
        sum_g, cnt_g = g.track_get()
        assert np.array_equal(cnt_o, cnt_g) and np.array_equal(sum_o, sum_g)
        assert int(cnt_g.sum()) > 0
    assert g.counters()["x0"] == o.counters()["x0"] == 7
    # seeding: track state with random directions and magnitudes, real spins
    w = ai.make_config(4)
    sx, sy, sz = ai.tilted_spins(w.n_sites, 20.0, seed=4)
    mag = w.magnetic_mask().reshape(-1)
    w.sx, w.sy, w.sz = sx * mag, sy * mag, sz * mag
    o, g = oracle_from_workload(w), gpu_from_workload(w)
    ncx, ncy, ncz = g.track_dims()
    rng = np.random.default_rng(8)
    v = rng.standard_normal((ncx * ncy * ncz, 3))
    v /= np.linalg.norm(v, axis=1, keepdims=True)
    v *= rng.uniform(0.0, 1.0, size=(v.shape[0], 1))
    v = v.astype(np.float32)
    o.track_set_init(v); g.track_set_init(v)
    for p in (3, 4):
        assert o.shift_window(p) == 0
        g.shift_window(p)
        so, sg = o.get_spins(), g.get_spins_host().astype(np.float64)
        assert np.abs(so - sg).max() < 3e-6
        slab = sg[:, (nx - p) * ny * nz:]
        n = np.sqrt((slab ** 2).sum(axis=0))
        assert np.all((np.abs(n - 1.0) < 2e-6) | (n == 0.0))       # seeded spins are unit vectors, vacant sites 0
    # one Heun step after the shifts: the window origin, the grain map and the Philox site ids moved along
    o.step_heun(1); g.step_heun(1)
    assert np.abs(o.get_spins() - g.get_spins_host()).max() <= 1e-5


def test_heun_after_shift_uses_new_origin():
    """Noise follows the atom (global site id) and the grain map follows the window after a shift."""
    w = ai.small_film(ai.L10, 20, 24, 5, extra_track=12, tilt_deg=20.0, dt=1e-16)
    o, g = oracle_from_workload(w), gpu_from_workload(w)
    o.step_heun(1); g.step_heun(1)
    o.shift_window(4); g.shift_window(4)
    o.step_heun(2); g.step_heun(2)
    o.shift_window(3); g.shift_window(3)
    o.step_heun(1); g.step_heun(1)
    assert np.abs(o.get_spins() - g.get_spins_host()).max() < 3e-5


def test_shift_errors():
    import paper_2502_02236_b200 as asd
    w = ai.small_film(ai.SC, 8, 8, 3, extra_track=2)
    g = gpu_from_workload(w)
    with pytest.raises(asd.AsdError) as e:
        g.shift_window(0)
    assert e.value.status == 1
    with pytest.raises(asd.AsdError) as e:
        g.shift_window(3)              # past the end of the track
    assert e.value.status == 4
    g.shift_window(2)


def test_option_and_demag_errors():
    """Error behaviour of the option calls (include/asd.h): bad arguments are ASD_EINVAL, demag queries before
    asd_enable_demag are ASD_ESTATE, lattices the demag path does not cover are ASD_EUNSUPPORTED."""
    import paper_2502_02236_b200 as asd
    w = ai.small_film(ai.SC, 8, 8, 3)
    g = gpu_from_workload(w)
    for bad in (lambda: g.set_graph_mode(7), lambda: g.set_kernel(9), lambda: g.set_demag_every(-1),
                lambda: g.demag_field(), lambda: g.enable_demag([0.3e-9, 0.0, 0.3e-9])):
        with pytest.raises(asd.AsdError):
            bad()
    g.step_heun(2)                                        # the context is still usable after the refused calls
    p = ai.make_config(0)                                 # periodic: no demag
    gp = gpu_from_workload(p)
    with pytest.raises(asd.AsdError):
        gp.enable_demag([0.3e-9] * 3)


def test_staged_field_upload_equals_the_direct_one():
    """asd_stage_fields_host + asd_commit_fields (double-buffered upload) must leave exactly the state asd_set_fields_host
    does, including 'NULL = keep', a re-stage while steps are in flight, and a commit with nothing staged."""
    import torch
    w = ai.small_film(ai.L10, 16, 24, 5, tilt_deg=20.0)
    a, b = gpu_from_workload(w), gpu_from_workload(w)
    pin = lambda x: torch.from_numpy(np.ascontiguousarray(x, dtype=np.float32)).pin_memory()
    rng = np.random.default_rng(1)
    T2, Bz2 = pin(w.T * 1.3 + 5.0), pin(rng.standard_normal(w.n_sites))
    T3, Bx3 = pin(w.T * 0.5), pin(rng.standard_normal(w.n_sites))
    a.set_fields_host(T=T2, Bz=Bz2); a.step_heun(3)
    a.set_fields_host(T=T3, Bx=Bx3); a.step_heun(2)

    b.stage_fields_host(T=T2, Bz=Bz2); b.commit_fields(); b.step_heun(3)
    b.stage_fields_host(T=T3, Bx=Bx3)                      # copied while the 3 steps above run
    b.commit_fields(); b.commit_fields()                   # the second commit has nothing to do
    b.step_heun(2)
    assert np.array_equal(a.get_spins_host(), b.get_spins_host())
