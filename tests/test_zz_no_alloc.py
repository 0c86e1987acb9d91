"""asd_spin_sum_noalloc (csrc/asd_noalloc.cu): the magnetisation reduction for callers that may not allocate.  Its
scratch is a static array in device memory instead of the context's workspace; the existing path it is checked against
is asd_magnetisation_planes (same two-stage fp64 reduction, partials in the caller-owned workspace).

Collected last on purpose (the suite runs with pytest -x): named test_zz_*.  Runs alone in a fresh process as well as
after the other tests -- it depends on no state but the library's own static array, which it exercises twice in a row
(a long call, then a shorter one that must not read the long call's stale rows)."""
import numpy as np
import pytest

import asd_inputs as ai
import paper_2502_02236_b200 as asd

pytestmark = pytest.mark.gpu

# two fp64 sums of the same fp32 values in different orders: |difference| <= N * 2^-52 * max partial sum; the tests of the
# existing path (test_magnetisation_and_grains) hold the MEAN to 1e-6 against the oracle -- this is far inside that
TOL_SUM = 1e-7


def _sums(g, i0, n, out4):
    """(sum S, count) of planes i0 .. i0+n-1 through the no-alloc entry point; views are re-asked (they move per step)."""
    import torch
    v = [g.planes_view(c, i0, n) for c in range(3)]
    asd.spin_sum_noalloc(v[0], v[1], v[2], out4)
    torch.cuda.synchronize()
    r = out4.cpu().numpy()
    return r[:3].copy(), float(r[3])


def test_two_calls_in_a_row_match_the_workspace_reduction():
    import torch
    w = ai.small_film(ai.L10, 30, 44, 6, tilt_deg=35.0)          # grains with vacant boundaries: N_mag != N
    g = asd.context_from_workload(w)
    out4 = torch.full((4,), float("nan"), dtype=torch.float64, device="cuda:0")   # the caller's output, made up front
    g.step_heun(3)

    # call 1: the whole window (30 planes x 6 rows x the padded row stride: a few 4096-element partial rows)
    s_ref, n_ref = g.magnetisation_planes(0, w.nx)
    s1, n1 = _sums(g, 0, w.nx, out4)
    assert n1 == n_ref and 0 < n_ref < w.nx * w.ny * w.nz
    assert np.abs(s1 - s_ref).max() < TOL_SUM
    m_ref, nm = g.magnetisation()
    assert nm == n1 and np.abs(s1 / n1 - m_ref).max() < 1e-12

    # call 2, straight after, on other data and FEWER rows: the first planes only, after more steps -- the static array
    # still holds call 1's rows beyond the ones this call writes; they must not be read
    g.step_heun(2)
    s_ref2, n_ref2 = g.magnetisation_planes(0, 7)
    s2, n2 = _sums(g, 0, 7, out4)
    assert n2 == n_ref2 and n2 < n1
    assert np.abs(s2 - s_ref2).max() < TOL_SUM
    assert np.abs(s2 - s1).max() > 1e-3                          # it really is another result

    # and the whole window again: deterministic, bit for bit, call after call
    a, na = _sums(g, 0, w.nx, out4)
    b, nb = _sums(g, 0, w.nx, out4)
    assert np.array_equal(a, b) and na == nb
    s_ref3, n_ref3 = g.magnetisation_planes(0, w.nx)
    assert na == n_ref3 and np.abs(a - s_ref3).max() < TOL_SUM


def test_plain_arrays_and_a_ragged_tail():
    """No context at all: three arrays whose length is not a multiple of the 4096-element row, with zeros in them."""
    import torch
    rng = np.random.default_rng(5)
    n = 3 * 4096 + 1234
    s = rng.normal(size=(n, 3)); s /= np.linalg.norm(s, axis=1, keepdims=True)
    s[rng.random(n) < 0.2] = 0.0                                  # vacant sites / pads
    s32 = s.astype(np.float32)
    t = [torch.from_numpy(np.ascontiguousarray(s32[:, c])).cuda() for c in range(3)]
    out4 = torch.zeros(4, dtype=torch.float64, device="cuda:0")
    asd.spin_sum_noalloc(t[0], t[1], t[2], out4)
    r = out4.cpu().numpy()
    assert r[3] == float((np.abs(s32).sum(axis=1) > 0).sum())
    assert np.abs(r[:3] - s32.astype(np.float64).sum(axis=0)).max() < TOL_SUM


def test_sizes_beyond_the_static_array_are_refused():
    import torch
    assert asd.NOALLOC_MAX_COUNT == 8388608
    big = torch.zeros(asd.NOALLOC_MAX_COUNT + 1, dtype=torch.float32, device="cuda:0")
    out4 = torch.full((4,), 7.0, dtype=torch.float64, device="cuda:0")
    with pytest.raises(asd.AsdError) as e:
        asd.spin_sum_noalloc(big, big, big, out4)
    assert e.value.status == 1 and "ASD_NOALLOC_MAX_COUNT" in str(e.value) and "8388608" in str(e.value)
    torch.cuda.synchronize()
    assert np.array_equal(out4.cpu().numpy(), np.full(4, 7.0))    # nothing was launched
    ok = big[:asd.NOALLOC_MAX_COUNT]                              # the largest size it takes
    asd.spin_sum_noalloc(ok, ok, ok, out4)
    assert np.array_equal(out4.cpu().numpy(), np.zeros(4))
