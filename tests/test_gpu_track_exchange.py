"""GPU parity for asd_enable_track_exchange (reading E1): the ends of a purely atomistic window
exchange coupled to the frozen track, against the oracle -- every Heun kernel, across shifts and track changes."""
import numpy as np
import pytest

import asd_inputs as ai
import paper_2502_02236_b200 as asd
from tests.helpers import gpu_from_workload, max_abs_diff, oracle_from_workload

pytestmark = pytest.mark.gpu

KERNELS = {"general": asd.KERNEL_GENERAL, "fast": asd.KERNEL_FAST, "fused": asd.KERNEL_FUSED, "auto": asd.KERNEL_AUTO}


@pytest.mark.parametrize("lattice", [ai.SC, ai.L10])
@pytest.mark.parametrize("kernel", ["general", "fast", "fused", "auto"])
def test_coupled_ends_match_the_oracle(lattice, kernel):
    w = ai.small_film(lattice, 20, 40, 6, extra_track=24, macro=(4, 5, 2), tilt_deg=25.0, dt=1e-16)
    o, g = oracle_from_workload(w), gpu_from_workload(w)
    rng = np.random.default_rng(4)
    v = rng.standard_normal((int(np.prod(o.track_dims())), 3)).astype(np.float32)
    o.track_set_init(v); g.track_set_init(v)
    o.shift_window(3); g.shift_window(3)                       # x0 = 3: both ends now have track beyond them
    o.enable_track_exchange(True); g.enable_track_exchange(True)
    g.set_kernel(KERNELS[kernel])
    o.step_heun(1); g.step_heun(1)
    assert max_abs_diff(g, o) <= 1e-5
    o.step_heun(3); g.step_heun(3)
    assert max_abs_diff(g, o) <= 5e-5
    o.shift_window(4); g.shift_window(4)                       # the track directions beyond the ends change
    o.step_heun(2); g.step_heun(2)
    assert max_abs_diff(g, o) <= 1e-4
    o.track_set_init(None, 0.9); g.track_set_init(None, 0.9)   # ... and so they do when the track state is replaced
    o.step_heun(1); g.step_heun(1)
    assert max_abs_diff(g, o) <= 1.2e-4
    # it is live: an uncoupled window ends up elsewhere on its end planes (and, through the corrector, a little on the next)
    a, b = gpu_from_workload(w), gpu_from_workload(w)
    for c in (a, b):
        c.track_set_init(v); c.shift_window(3); c.set_kernel(asd.KERNEL_GENERAL)
    b.enable_track_exchange(True)
    a.step_heun(1); b.step_heun(1)
    d = np.abs(a.get_spins_host() - b.get_spins_host()).reshape(3, w.nx, w.nz, w.ny)
    assert d[:, 0].max() > 1e-4 and d[:, -1].max() > 1e-4 and d[:, 1].max() < 1e-4 and not d[:, 2:-2].any()


@pytest.mark.parametrize("lattice", [ai.SC, ai.L10])
@pytest.mark.parametrize("kernel,every", [("general", 0), ("fast", 0), ("fast", 2), ("fused", 1), ("auto", 1)])
def test_the_whole_window_of_p33(lattice, kernel, every):
    """Everything P:33 puts on the window at once: ends exchange coupled to the frozen track, the window's own
    demagnetising field and the track's stray field -- film and fused kernels carry the edge field and the cell field
    together."""
    w = ai.small_film(lattice, 20, 40, 6, extra_track=24, macro=(4, 5, 2), tilt_deg=25.0, dt=1e-16)
    o, g = oracle_from_workload(w), gpu_from_workload(w)
    rng = np.random.default_rng(5)
    v = rng.standard_normal((int(np.prod(o.track_dims())), 3)).astype(np.float32)
    o.track_set_init(v); g.track_set_init(v)
    o.shift_window(3); g.shift_window(3)
    sp = [a * 1e-9 for a in w.spacing_nm]
    for c in (o, g):
        c.enable_demag(sp); c.set_demag_every(every); c.enable_track_stray(True, 0); c.enable_track_exchange(True)
    g.set_kernel(KERNELS[kernel])
    o.step_heun(1); g.step_heun(1)
    assert max_abs_diff(g, o) <= 1e-5
    o.step_heun(4); g.step_heun(4)
    assert max_abs_diff(g, o) <= 6e-5
    o.shift_window(4); g.shift_window(4)
    o.step_heun(3); g.step_heun(3)
    assert max_abs_diff(g, o) <= 1.2e-4


def test_refusals_and_switching_off():
    w = ai.small_film(ai.L10, 16, 24, 4, extra_track=16, macro=(4, 4, 2))
    g = gpu_from_workload(w)
    g.shift_window(4)
    g.enable_track_exchange(True)
    g.step_heun(2)
    with pytest.raises(asd.AsdError) as e:
        g.set_kernel(asd.KERNEL_TMA)
    assert e.value.status == 5
    with pytest.raises(asd.AsdError) as e:
        g.set_kernel(asd.KERNEL_PERSISTENT)
    assert e.value.status == 5
    g.enable_track_exchange(False)
    g.set_kernel(asd.KERNEL_PERSISTENT)
    g.step_heun(2)
