"""GPU parity for the persistent-cluster path (csrc/asd_heun_persist.cu; "cfg 0 is launch/latency-bound
... one persistent CTA"): n Heun steps in one launch with the lattice resident in distributed shared memory."""
import numpy as np
import pytest

import asd_inputs as ai
import paper_2502_02236_b200 as asd
from tests.helpers import gpu_from_workload, max_abs_diff, oracle_from_workload

pytestmark = pytest.mark.gpu


def test_cfg0_on_the_persistent_cluster():
    w = ai.make_config(0)
    o, g = oracle_from_workload(w), gpu_from_workload(w)
    g.set_kernel(asd.KERNEL_PERSISTENT)
    o.step_heun(1); g.step_heun(1)
    assert max_abs_diff(g, o) <= 1e-5
    n0 = g.launch_count()
    o.step_heun(9); g.step_heun(9)
    assert g.launch_count() == n0 + 1                       # one launch per call, however many steps
    assert max_abs_diff(g, o) <= 1e-4
    assert g.counters()["step"] == 10
    w0 = ai.make_config(0, uniform_T=0.0)
    o, g = oracle_from_workload(w0), gpu_from_workload(w0)
    g.set_kernel(asd.KERNEL_PERSISTENT)
    o.step_heun(1000); g.step_heun(1000)
    assert max_abs_diff(g, o) <= 1e-4
    s = g.get_spins_host().astype(np.float64)
    assert np.all(np.abs(np.sqrt((s ** 2).sum(axis=0)) - 1.0) < 2e-7)


def test_one_launch_of_n_steps_is_bit_identical_to_n_launches():
    w = ai.make_config(0)
    a, b, c = gpu_from_workload(w), gpu_from_workload(w), gpu_from_workload(w)
    for g in (a, b, c):
        g.set_kernel(asd.KERNEL_PERSISTENT)
    a.step_heun(13)
    for _ in range(13):
        b.step_heun(1)
    c.step_heun(5); c.set_field_scale(1.0); c.step_heun(8)
    sa = a.get_spins_host()
    assert np.array_equal(sa, b.get_spins_host()) and np.array_equal(sa, c.get_spins_host())
    # AUTO takes the same path on a lattice this small
    d = gpu_from_workload(w)
    d.step_heun(13)
    assert np.array_equal(sa, d.get_spins_host())


@pytest.mark.parametrize("lattice", [ai.SC, ai.L10])
@pytest.mark.parametrize("dims,pbc", [((16, 8, 4), (0, 0, 0)), ((8, 16, 6), (0, 0, 0)), ((24, 12, 5), (0, 0, 0)),
                                      ((6, 8, 5), (0, 0, 0)), ((5, 4, 3), (0, 0, 0)), ((32, 32, 8), (0, 0, 0)),
                                      ((32, 64, 12), (0, 0, 0)), ((64, 64, 12), (0, 0, 0))])
def test_open_films_with_grains(lattice, dims, pbc):
    """Granular films (vacant boundaries, several grains, Gaussian spot, head field): clusters of 8, 4, 2 and 1 CTAs,
    one to several planes per CTA, 256-, 512- and 1024-thread slabs, one and four sites per thread."""
    nx, ny, nz = dims
    w = ai.small_film(lattice, nx, ny, nz, tilt_deg=25.0, dt=1e-16)
    o, g = oracle_from_workload(w), gpu_from_workload(w)
    g.set_kernel(asd.KERNEL_PERSISTENT)
    o.step_heun(1); g.step_heun(1)
    assert max_abs_diff(g, o) <= 1e-5
    o.step_heun(4); g.step_heun(4)
    assert max_abs_diff(g, o) <= 5e-5
    s = g.get_spins_host()
    assert np.all(s[:, ~w.magnetic_mask().reshape(-1)] == 0.0)


@pytest.mark.parametrize("lattice", [ai.SC, ai.L10])
@pytest.mark.parametrize("pbc", [(1, 1, 1), (0, 1, 0), (1, 0, 1), (0, 0, 1), (1, 0, 0)])
def test_periodic_wraps(lattice, pbc):
    """One grain, every mix of periodic and open directions; 8 x 12 x 5 sites on a cluster of 8 (one plane per CTA: both x
    neighbours live in other CTAs) and 6 x 8 x 3 on a cluster of 2."""
    from oracle import asd_oracle as orc
    rng = np.random.default_rng(3)
    for (nx, ny, nz) in ((8, 12, 5), (6, 8, 3)):
        N = nx * ny * nz
        J = ai.workloads.J_SC if lattice == ai.SC else ai.workloads.J_L10
        v = rng.standard_normal((N, 3)); v /= np.linalg.norm(v, axis=1, keepdims=True)
        v = v.astype(np.float32)
        T = rng.uniform(0.0, 600.0, N).astype(np.float32)
        B = rng.uniform(-1.0, 1.0, (3, N)).astype(np.float32)
        ax = np.array([[0.6, 0.0, 0.8]], dtype=np.float32)
        spec = orc.LatticeSpec(lattice=lattice, nx=nx, ny=ny, nz=nz, pbc=pbc, dt=1e-16, J=J,
                               grain_map=np.zeros((nx, ny), dtype=np.int32), grain_ku=np.array([9.1e-23]),
                               grain_axis=ax.astype(np.float64), macro=(3, 3, 3), seed=7)
        o = orc.Oracle(spec)
        o.set_spins(v[:, 0], v[:, 1], v[:, 2]); o.set_fields(T, B[0], B[1], B[2])
        d = asd.LatticeDesc(lattice=lattice, nx=nx, ny=ny, nz=nz, pbc=pbc, dt=1e-16, J=J,
                            grain_map=np.zeros((nx, ny), dtype=np.int32), n_grains=1,
                            grain_ku=np.array([9.1e-23], dtype=np.float32), grain_axis=ax, macro=(3, 3, 3), seed=7)
        g = asd.Context(d)
        g.set_spins_host(v[:, 0].copy(), v[:, 1].copy(), v[:, 2].copy())
        g.set_fields_host(T, B[0].copy(), B[1].copy(), B[2].copy())
        g.set_kernel(asd.KERNEL_PERSISTENT)
        o.step_heun(1); g.step_heun(1)
        assert np.abs(o.get_spins() - g.get_spins_host()).max() <= 1e-5
        o.step_heun(3); g.step_heun(3)
        assert np.abs(o.get_spins() - g.get_spins_host()).max() <= 4e-5


def test_auto_takes_the_cluster_where_it_measured_faster():
    """ASD_KERNEL_AUTO (heun_persist_preferred): simple-cubic film slabs up to 2048 sites per CTA, L1_0 up to 1024; beyond
    that the replayed stage kernels.  Same arithmetic per path, so the comparison is bit for bit."""
    for lattice, dims, expect in ((ai.SC, (32, 64, 12), "persistent"), (ai.SC, (64, 64, 12), "fast"),
                                  (ai.L10, (64, 32, 8), "persistent"), (ai.L10, (32, 64, 12), "fast")):
        w = ai.small_film(lattice, *dims, tilt_deg=25.0, dt=1e-16)
        a, b = gpu_from_workload(w), gpu_from_workload(w)
        b.set_kernel(asd.KERNEL_PERSISTENT if expect == "persistent" else asd.KERNEL_FAST)
        n0 = a.launch_count()
        a.step_heun(6); b.step_heun(6)
        n1 = a.launch_count()                                   # before the read-back launches its unpack kernel
        assert np.array_equal(a.get_spins_host(), b.get_spins_host())
        assert (n1 - n0 == 1) == (expect == "persistent")


def test_refused_where_it_does_not_apply():
    w = ai.small_film(ai.SC, 40, 132, 9)                      # a slab does not fit 1024 threads
    g = gpu_from_workload(w)
    with pytest.raises(asd.AsdError) as e:
        g.set_kernel(asd.KERNEL_PERSISTENT)
    assert e.value.status == 5
    w = ai.small_film(ai.SC, 8, 10, 3)                        # ny % 4 != 0
    g = gpu_from_workload(w)
    with pytest.raises(asd.AsdError):
        g.set_kernel(asd.KERNEL_PERSISTENT)
