"""CUDA-graph replay of asd_step_heun (csrc/asd_graph.cu): recorded batches must reproduce plain launches bit for bit --
same kernels in the same order; only the way the step index and the field scale reach them differs."""
import numpy as np
import pytest

import asd_inputs as ai
from tests.helpers import gpu_from_workload, max_abs_diff, oracle_from_workload

pytestmark = pytest.mark.gpu


def _run(w, mode, kernel=None):
    import paper_2502_02236_b200 as asd
    g = gpu_from_workload(w)
    g.set_graph_mode(mode)
    if kernel is not None:
        g.set_kernel(kernel)
    g.step_heun(7)                  # one recorded batch of 7
    g.set_field_scale(-0.5)         # the scale is read from device memory by the replay
    g.step_heun(150)                # 64 + 64 + 22
    g.shift_window(3)               # drops the recorded graphs (window origin, buffer roles)
    g.step_heun(7)
    g.step_heun(1)                  # below the graph threshold: plain launches
    return g


@pytest.mark.parametrize("lattice", [ai.SC, ai.L10])
@pytest.mark.parametrize("kernel", ["general", "fast", "tma"])
def test_graph_replay_is_bit_identical_to_plain_launches(lattice, kernel):
    import paper_2502_02236_b200 as asd
    k = {"general": asd.KERNEL_GENERAL, "fast": asd.KERNEL_FAST, "tma": asd.KERNEL_TMA}[kernel]
    w = ai.small_film(lattice, 24, 40, 6, extra_track=8, tilt_deg=20.0)
    a = _run(w, asd.GRAPH_OFF, k)
    b = _run(w, asd.GRAPH_ON, k)
    assert np.array_equal(a.get_spins_host(), b.get_spins_host())
    assert a.counters() == b.counters()
    assert a.launch_count() < b.launch_count() <= a.launch_count() + 8     # + one set_dyn per replay


def test_cfg0_1000_steps_through_graphs_matches_oracle():
    """cfg0 (4096 spins) is launch-bound: ASD_GRAPH_AUTO replays graphs there.  Same tolerance as the plain path."""
    import paper_2502_02236_b200 as asd
    w = ai.make_config(0, uniform_T=0.0)
    o, g = oracle_from_workload(w), gpu_from_workload(w)
    g.set_kernel(asd.KERNEL_GENERAL)         # AUTO would take the persistent cluster (one launch, no graph) on 4096 sites
    n0 = g.launch_count()
    o.step_heun(1000); g.step_heun(1000)
    assert g.launch_count() - n0 >= 2000     # 2000 kernel nodes replayed (+ one set_dyn per replay)
    assert max_abs_diff(g, o) <= 1e-4


@pytest.mark.parametrize("kernel", ["general", "fast"])
def test_dependent_launches_match_serialised_graph_edges_over_many_steps(kernel):
    """The stage kernels are launched with programmatic dependent launch and read what the previous grid wrote through
    the read-only data path after their griddepcontrol.wait.  On a lattice this small three grids
    are co-resident.  Recorded graphs keep plain (fully serialising) edges: 3000 steps of both must agree bit for bit."""
    import paper_2502_02236_b200 as asd
    k = {"general": asd.KERNEL_GENERAL, "fast": asd.KERNEL_FAST}[kernel]
    w = ai.small_film(ai.L10, 16, 32, 6, tilt_deg=20.0)
    a, b = gpu_from_workload(w), gpu_from_workload(w)
    for g, mode in ((a, asd.GRAPH_OFF), (b, asd.GRAPH_ON)):
        g.set_kernel(k); g.set_graph_mode(mode)
        g.step_heun(3000)
    assert np.array_equal(a.get_spins_host(), b.get_spins_host())
