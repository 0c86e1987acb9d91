"""Slab decomposition on the GPU (paper_2502_02236_b200/slab.py over asd_planes_view): several slabs of one window as
contexts of one process on one device, halo planes copied device to device -- bit-identical to the undivided window for
every kernel variant, across window shifts; the reduction over the slabs' own planes reproduces the magnetisation."""
import numpy as np
import pytest

import asd_inputs as ai
import paper_2502_02236_b200 as asd
from paper_2502_02236_b200.slab import SlabWindow
from tests.helpers import gpu_from_workload

pytestmark = pytest.mark.gpu

KERNELS = {"general": asd.KERNEL_GENERAL, "fast": asd.KERNEL_FAST, "fused": asd.KERNEL_FUSED}


@pytest.mark.parametrize("lattice", [ai.SC, ai.L10])
@pytest.mark.parametrize("kernel", ["general", "fast", "fused"])
@pytest.mark.parametrize("nslabs,halo", [(2, 2), (3, 2), (2, 4)])
def test_slabs_bit_identical_to_the_whole_window(lattice, kernel, nslabs, halo):
    w = ai.small_film(lattice, 36, 40, 6, extra_track=10, tilt_deg=20.0)
    whole = gpu_from_workload(w)
    whole.set_kernel(KERNELS[kernel])
    parts = SlabWindow.local(w, nslabs, halo=halo, kernel=KERNELS[kernel])
    for sim in (whole, parts):
        sim.step_heun(5)
    assert np.array_equal(parts.gather_spins_host(), whole.get_spins_host())
    for sim in (whole, parts):
        sim.set_field_scale(-0.5); sim.shift_window(3); sim.step_heun(4); sim.shift_window(4); sim.step_heun(3)
    assert np.array_equal(parts.gather_spins_host(), whole.get_spins_host())
    m_w, n_w = whole.magnetisation()
    m_p, n_p = parts.magnetisation()
    assert n_w == n_p and np.abs(m_w - m_p).max() < 1e-13
    s0, c0 = parts.ctx[0].track_get()
    sw, cw = whole.track_get()
    assert np.array_equal(c0, cw) and np.array_equal(s0, sw)


def test_planes_view_and_range_magnetisation():
    w = ai.small_film(ai.SC, 12, 16, 5, tilt_deg=30.0)
    g = gpu_from_workload(w)
    S = g.get_spins_host().reshape(3, 12, 5, 16)
    nyp = 16 + 4
    v = g.planes_view(1, 3, 2).cpu().numpy().reshape(2, 5, nyp)
    assert np.array_equal(v[:, :, :16], S[1, 3:5]) and not v[:, :, 16:].any()
    s, cnt = g.magnetisation_planes(3, 4)
    mag = w.magnetic_mask()[3:7]
    assert cnt == mag.sum()
    assert np.abs(s - S[:, 3:7].astype(np.float64).reshape(3, -1).sum(axis=1)).max() < 1e-9
    for bad in ((0, -1, 1), (0, 11, 2), (3, 0, 1)):
        with pytest.raises(asd.AsdError):
            g.planes_view(*bad)
