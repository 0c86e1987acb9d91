"""GPU parity: libasd (CUDA, fp32) against the fp64 oracle on the same seeded inputs, through the C ABI.

Tolerances (BASELINE.json north_star): max |dS| <= 1e-5 per component after one Heun step; <= 1e-4 after
1000 deterministic T = 0 steps.  |S| = 1 within 2e-7.
"""
import numpy as np
import pytest

import asd_inputs as ai
from tests.helpers import gpu_from_workload, max_abs_diff, oracle_from_workload

pytestmark = pytest.mark.gpu

TOL_1STEP = 1e-5
TOL_T0_1000 = 1e-4


def _check_norm(ctx, w):
    s = ctx.get_spins_host().astype(np.float64)
    mag = w.magnetic_mask().reshape(-1)
    nrm = np.sqrt((s ** 2).sum(axis=0))
    assert np.all(np.abs(nrm[mag] - 1.0) < 2e-7)
    assert np.all(s[:, ~mag] == 0.0)


def test_cfg0_one_thermal_step():
    w = ai.make_config(0)
    o, g = oracle_from_workload(w), gpu_from_workload(w)
    o.step_heun(1); g.step_heun(1)
    assert max_abs_diff(g, o) <= TOL_1STEP
    _check_norm(g, w)


def test_cfg0_thermal_divergence_report():
    """Informational: thermal trajectories diverge chaotically; 10 steps still agree closely."""
    w = ai.make_config(0)
    o, g = oracle_from_workload(w), gpu_from_workload(w)
    o.step_heun(10); g.step_heun(10)
    assert max_abs_diff(g, o) <= 1e-4


def test_cfg0_1000_steps_zero_temperature():
    w = ai.make_config(0, uniform_T=0.0)
    o, g = oracle_from_workload(w), gpu_from_workload(w)
    o.step_heun(1000); g.step_heun(1000)
    assert max_abs_diff(g, o) <= TOL_T0_1000
    _check_norm(g, w)


@pytest.mark.parametrize("lattice", [ai.SC, ai.L10])
@pytest.mark.parametrize("dims", [(21, 40, 7), (13, 37, 5), (9, 4, 3), (3, 3, 3), (1, 8, 1), (40, 132, 9)])
def test_small_film_steps(lattice, dims):
    """Several tiles and a ragged tail; ny % 4 == 0 takes the 128-bit path, odd ny the scalar one."""
    nx, ny, nz = dims
    w = ai.small_film(lattice, nx, ny, nz, tilt_deg=25.0, dt=1e-16)
    o, g = oracle_from_workload(w), gpu_from_workload(w)
    o.step_heun(1); g.step_heun(1)
    assert max_abs_diff(g, o) <= TOL_1STEP
    o.step_heun(4); g.step_heun(4)
    assert max_abs_diff(g, o) <= 5e-5
    _check_norm(g, w)


@pytest.mark.parametrize("lattice", [ai.SC, ai.L10])
@pytest.mark.parametrize("pbc", [(1, 1, 1), (0, 1, 0), (1, 0, 1), (0, 0, 1)])
@pytest.mark.parametrize("dims", [(6, 8, 5), (5, 7, 3)])
def test_adjacent_grains_and_periodic_boundaries(lattice, pbc, dims):
    """Random grain map with touching grains (bonds must be cut between different grains) and every wrap."""
    nx, ny, nz = dims
    rng = np.random.default_rng(5)
    w = ai.small_film(lattice, nx, ny, nz, tilt_deg=30.0, dt=1e-16)
    w.pbc = pbc
    w.grain_map = rng.integers(-1, 3, size=(nx, ny)).astype(np.int32)
    w.grain_ku = (9.1e-23 * (1 + 0.3 * rng.standard_normal(3))).astype(np.float32)
    ax = rng.standard_normal((3, 3)); ax /= np.linalg.norm(ax, axis=1, keepdims=True)
    w.grain_axis = ax.astype(np.float32)
    sx, sy, sz = ai.tilted_spins(w.n_sites, 30.0, seed=9)
    mag = w.magnetic_mask().reshape(-1)
    w.sx, w.sy, w.sz = sx * mag, sy * mag, sz * mag
    o, g = oracle_from_workload(w), gpu_from_workload(w)
    o.step_heun(2); g.step_heun(2)
    assert max_abs_diff(g, o) <= 2e-5
    _check_norm(g, w)


@pytest.mark.parametrize("kernel", ["auto", "general"])
@pytest.mark.parametrize("lattice", [ai.SC, ai.L10])
def test_shell_table_as_ell(lattice, kernel):
    """The built-in shells handed over as an ELL table (asd_inputs.shell_ell_table): the dedicated ELL kernel
    (asd_heun_ell.cu, what AUTO runs) and the general kernel against the oracle driven by the same table."""
    import paper_2502_02236_b200 as asd
    w = ai.small_film(lattice, 21, 38, 7, tilt_deg=25.0, dt=1e-16)
    idx, J = ai.shell_ell_table(w)
    o = oracle_from_workload(w, ell_idx=idx, ell_J=J.astype(np.float64))
    g = gpu_from_workload(w, ell_idx=idx, ell_J=J)
    if kernel == "general":
        g.set_kernel(asd.KERNEL_GENERAL)
    o.step_heun(1); g.step_heun(1)
    assert max_abs_diff(g, o) <= TOL_1STEP
    o.step_heun(4); g.step_heun(4)
    assert max_abs_diff(g, o) <= 5e-5
    _check_norm(g, w)


def test_general_ell_table():
    """User-supplied neighbour table with arbitrary per-pair J (random sparse couplings)."""
    nx, ny, nz = 7, 12, 4
    w = ai.small_film(ai.SC, nx, ny, nz, tilt_deg=30.0, dt=1e-16)
    N, W = w.n_sites, 5
    rng = np.random.default_rng(3)
    idx = rng.integers(-1, N, size=(N, W)).astype(np.int32)
    J = (6e-21 * rng.standard_normal((N, W))).astype(np.float32)
    o = oracle_from_workload(w, ell_idx=idx, ell_J=J.astype(np.float64))
    g = gpu_from_workload(w, ell_idx=idx, ell_J=J)
    o.step_heun(2); g.step_heun(2)
    assert max_abs_diff(g, o) <= 2e-5


def test_magnetisation_and_grains():
    w = ai.small_film(ai.L10, 30, 44, 6, tilt_deg=35.0)
    o, g = oracle_from_workload(w), gpu_from_workload(w)
    o.step_heun(3); g.step_heun(3)
    mo, no = o.magnetisation()
    mg, ng = g.magnetisation()
    assert no == ng
    assert np.abs(mo - mg).max() < 1e-6
    assert np.abs(o.grain_magnetisation() - g.grain_magnetisation()).max() < 1e-6
    mg2, _ = g.magnetisation()
    assert np.array_equal(mg, mg2)                       # deterministic reduction
    assert np.array_equal(g.grain_magnetisation(), g.grain_magnetisation())


def test_counters_resume_bit_exact():
    """Philox is counter based: restoring spins + counters reproduces the trajectory bit for bit."""
    import torch
    w = ai.small_film(ai.SC, 12, 16, 5, tilt_deg=20.0)
    a = gpu_from_workload(w)
    a.step_heun(5)
    snap = a.get_spins_host()
    cnt = a.counters()
    a.step_heun(7)
    ref = a.get_spins_host()
    b = gpu_from_workload(w)
    t = lambda x: torch.from_numpy(np.ascontiguousarray(x)).to(b.device)
    b.set_spins(t(snap[0]), t(snap[1]), t(snap[2]))
    b.set_counters(cnt["step"], cnt["shift"], cnt["pass"])
    b.step_heun(7)
    assert np.array_equal(b.get_spins_host(), ref)


_FULL = {}


def _full_size_workload(cfg):
    w = ai.make_config(cfg)
    sx, sy, sz = ai.tilted_spins(w.n_sites, 20.0, seed=4)
    mag = w.magnetic_mask().reshape(-1)
    w.sx, w.sy, w.sz = sx * mag, sy * mag, sz * mag
    return w


def _full_size_oracle(cfg, w, ell=None):
    """Oracle spins after 1 and after 2 Heun steps of a full-size config (computed once per session, shared by the
    kernel variants; the ELL run has its own entry: it exercises the oracle's table branch)."""
    key = (cfg, ell is not None)
    if key not in _FULL:
        o = oracle_from_workload(w) if ell is None else oracle_from_workload(w, ell_idx=ell[0], ell_J=ell[1].astype(np.float64))
        o.step_heun(1)
        s1 = o.get_spins()
        o.step_heun(1)
        _FULL[key] = (s1, o.get_spins())
    return _FULL[key]


@pytest.mark.parametrize("lattice", [ai.SC, ai.L10])
@pytest.mark.parametrize("dims", [(21, 40, 7), (9, 4, 3), (3, 8, 3), (1, 8, 1), (40, 132, 9), (70, 220, 27), (300, 24, 2)])
def test_staged_tma_kernel(lattice, dims):
    """The TMA-staged film kernel (asd_heun_tma.cu): several strips, chunks of 1..many planes, ragged last strip and
    chunk, against the oracle and bit-for-bit against nothing else (its own arithmetic order)."""
    import paper_2502_02236_b200 as asd
    nx, ny, nz = dims
    w = ai.small_film(lattice, nx, ny, nz, tilt_deg=25.0, dt=1e-16)
    o, g = oracle_from_workload(w), gpu_from_workload(w)
    g.set_kernel(asd.KERNEL_TMA)
    o.step_heun(1); g.step_heun(1)
    assert max_abs_diff(g, o) <= TOL_1STEP
    o.step_heun(3); g.step_heun(3)
    assert max_abs_diff(g, o) <= 5e-5
    _check_norm(g, w)


@pytest.mark.parametrize("lattice", [ai.SC, ai.L10])
@pytest.mark.parametrize("dims", [(21, 40, 7), (9, 4, 3), (3, 8, 3), (1, 8, 1), (40, 132, 9), (70, 220, 27), (300, 24, 2),
                                  (37, 100, 12)])
def test_fused_kernel(lattice, dims):
    """The one-kernel Heun step (asd_heun_fused.cu): several strips, chunks of 1..many planes, ragged last strip and
    chunk, halo columns and halo planes recomputed per CTA; odd and even numbers of steps (the spin buffers swap)."""
    import paper_2502_02236_b200 as asd
    nx, ny, nz = dims
    w = ai.small_film(lattice, nx, ny, nz, tilt_deg=25.0, dt=1e-16)
    o, g = oracle_from_workload(w), gpu_from_workload(w)
    g.set_kernel(asd.KERNEL_FUSED)
    o.step_heun(1); g.step_heun(1)
    assert max_abs_diff(g, o) <= TOL_1STEP
    _check_norm(g, w)
    o.step_heun(3); g.step_heun(3)
    assert max_abs_diff(g, o) <= 5e-5
    _check_norm(g, w)


def test_fused_kernel_matches_two_kernel_step_closely():
    """Fused and two-kernel steps compute the same Heun step in different association orders: they agree to a few ulp,
    and the fused step is bit-reproducible from run to run."""
    import paper_2502_02236_b200 as asd
    w = ai.small_film(ai.L10, 45, 72, 11, tilt_deg=25.0, dt=1e-16)
    a, b, c = gpu_from_workload(w), gpu_from_workload(w), gpu_from_workload(w)
    a.set_kernel(asd.KERNEL_FAST); b.set_kernel(asd.KERNEL_FUSED); c.set_kernel(asd.KERNEL_FUSED)
    a.step_heun(5); b.step_heun(5); c.step_heun(5)
    sa, sb, sc = a.get_spins_host(), b.get_spins_host(), c.get_spins_host()
    assert np.array_equal(sb, sc)
    assert float(np.abs(sa - sb).max()) <= 2e-6


@pytest.mark.parametrize("cfg", [2, 3, 4])
@pytest.mark.parametrize("kernel", ["fast", "tma", "fused", "auto"])
def test_full_size_one_step(cfg, kernel):
    """BASELINE configs at full size in the launch configuration bench.py times: every site against the oracle, at
    north_star's tolerance (1e-5 after ONE step), then a second step.  cfg3 = SC 400x200x27, cfg2 / cfg4 = L1_0."""
    import paper_2502_02236_b200 as asd
    w = _full_size_workload(cfg)
    (o1, o2), g = _full_size_oracle(cfg, w), gpu_from_workload(w)
    if kernel != "auto":
        g.set_kernel({"fast": asd.KERNEL_FAST, "tma": asd.KERNEL_TMA, "fused": asd.KERNEL_FUSED}[kernel])
    g.step_heun(1)
    assert float(np.abs(g.get_spins_host().astype(np.float64) - o1).max()) <= TOL_1STEP
    g.step_heun(1)
    assert float(np.abs(g.get_spins_host().astype(np.float64) - o2).max()) <= 2e-5
    _check_norm(g, w)


@pytest.mark.parametrize("cfg", [3, 4])
def test_full_size_one_step_ell(cfg):
    """The same windows handed over as a general ELL table with per-pair J (asd_inputs.shell_ell_table: W = 6 for SC,
    W = 10 for L1_0) -- the configuration `bench.py --ell` times; every site against the oracle's ELL branch."""
    w = _full_size_workload(cfg)
    idx, J = ai.shell_ell_table(w)
    (o1, o2) = _full_size_oracle(cfg, w, ell=(idx, J))
    g = gpu_from_workload(w, ell_idx=idx, ell_J=J)
    g.step_heun(1)
    assert float(np.abs(g.get_spins_host().astype(np.float64) - o1).max()) <= TOL_1STEP
    g.step_heun(1)
    assert float(np.abs(g.get_spins_host().astype(np.float64) - o2).max()) <= 2e-5
    # and the table says what the built-in shells say (the oracle's two branches, fp32-rounded J apart)
    assert float(np.abs(o2 - _full_size_oracle(cfg, w)[1]).max()) <= 1e-6
    _check_norm(g, w)


def test_near_the_32bit_offset_limit():
    """Maximum size of the film kernel (13 arrays x stride < 2^31 elements): a 147 M-site L1_0 window whose initial state
    is periodic with period 8 in every direction must reproduce, plane for plane and bit for bit, a 24-plane window with
    the same pattern (T = 0: no noise; identical local environments away from the x edges give identical arithmetic).
    Checks every element offset of the large window without the oracle having to hold 147 M fp64 sites."""
    import torch
    import paper_2502_02236_b200 as asd
    ny, nz = 256, 64
    dev = torch.device("cuda", 0)
    free, _ = torch.cuda.mem_get_info()
    nx_big = 8960                                              # 146.8 M sites: 13 * stride = 1.99e9 < 2^31
    if free < 12 * (1 << 30):
        pytest.skip("needs 12 GB of free device memory")

    def run(nx):
        d = asd.LatticeDesc(lattice=ai.L10, nx=nx, ny=ny, nz=nz, J=(5.0e-21, 2.0e-21, 0.8e-21), dt=1e-15, lam=0.1,
                            grain_ku=np.array([9.1e-23], dtype=np.float32),
                            grain_axis=np.array([[0.0, 0.6, 0.8]], dtype=np.float32))
        ctx = asd.Context(d)
        ctx.set_kernel(asd.KERNEL_FAST)
        i = torch.arange(nx, device=dev).view(nx, 1, 1) % 8
        k = torch.arange(nz, device=dev).view(1, nz, 1) % 8
        j = torch.arange(ny, device=dev).view(1, 1, ny) % 8
        th = 0.3 + 0.05 * (i + 2 * k) + 0.02 * j                # polar angle pattern, period 8
        ph = 0.7 * i + 0.4 * j + 0.9 * k
        sx = (torch.sin(th) * torch.cos(ph)).float().reshape(-1).contiguous()
        sy = (torch.sin(th) * torch.sin(ph)).float().reshape(-1).contiguous()
        sz = torch.cos(th).float().reshape(-1).contiguous()
        ctx.set_spins(sx, sy, sz)
        N = nx * ny * nz
        z = torch.zeros(N, device=dev)
        ctx.set_fields(z, z, z, torch.full((N,), 0.5, device=dev))
        ctx.step_heun(2)
        ctx.get_spins(sx, sy, sz)
        torch.cuda.synchronize()
        return torch.stack([sx, sy, sz]).view(3, nx, nz * ny)

    small = run(24)[:, 8:16].clone()                            # planes 8..15: two steps cannot see the x edges
    big = run(nx_big)
    for start in (8, 4480, nx_big - 16):                        # start % 8 == 0: same phase of the pattern
        assert torch.equal(big[:, start:start + 8], small), start
