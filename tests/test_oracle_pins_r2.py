"""Pins for the oracle branches that had none (oracle findings 1-3 and 6), all `-m "not gpu"`:

  * ELL branch of exchange_sum (oracle/asd_oracle.cpp): an ELL table built HERE from distances with random symmetric
    per-pair J, energy and field against a brute-force pair sum; and the shared helper asd_inputs.shell_ell_table
    against the oracle's built-in shells, bit for bit (Eq. (2); S:a2).
  * orc_magnetisation / orc_grain_magnetisation: numpy means over the magnetic mask / per-grain masks on a film with
    vacancies and several grains, N_mag != N (Eq. (6); S:O6).
  * the held-field branch of heun_step (demag_every = P, reading D3): equal, step for step, to the composition
    "demag off; at every P-th step add demag_cells() of the current spins to the per-site B through set_fields".
  * reading D2 (point dipoles beyond 12 cell diagonals): the error the switch-over introduces at cfg4's real offsets
    (7 x 7 x 5-site cells, up to 126 cells apart in x) measured against direct quadrature of the dipole kernel.
"""
import itertools
import math

import numpy as np
import pytest

import asd_inputs as ai
from oracle import asd_oracle as orc
from tests.helpers import oracle_from_workload
from tests.test_oracle_demag import _quad_tensor

MUS = 3.23 * orc.MU_B
MU0 = 4e-7 * np.pi


# ---------------------------------------------------------------------------------------------------------------
# ELL branch
# ---------------------------------------------------------------------------------------------------------------
def _pairs_by_distance(dims, spacing, cutoff, rng, gm):
    """All pairs of magnetic sites closer than `cutoff` (open boundaries), each with its own random J (symmetric)."""
    nx, ny, nz = dims
    coords = [(i, k, j) for i in range(nx) for k in range(nz) for j in range(ny)]        # l = (i*nz + k)*ny + j
    pairs = {}
    for a, b in itertools.combinations(range(len(coords)), 2):
        (i, k, j), (i2, k2, j2) = coords[a], coords[b]
        if gm[i, j] < 0 or gm[i2, j2] < 0:
            continue
        r = math.sqrt(((i2 - i) * spacing[0]) ** 2 + ((j2 - j) * spacing[1]) ** 2 + ((k2 - k) * spacing[2]) ** 2)
        if r < cutoff:
            pairs[(a, b)] = 6e-21 * rng.standard_normal()
    return pairs


def _ell_from_pairs(N, pairs, rng):
    """Site-major ELL table [N, W] from a pair list: slots in random order with -1 holes in between (a site-major /
    slot-major slip or a `break` at the first hole would show)."""
    nb = [[] for _ in range(N)]
    for (a, b), Jab in pairs.items():
        nb[a].append((b, Jab)); nb[b].append((a, Jab))
    W = max(len(x) for x in nb) + 2
    idx = np.full((N, W), -1, dtype=np.int32)
    J = np.zeros((N, W))
    for a in range(N):
        slots = rng.permutation(W)[:len(nb[a])]
        for s, (b, Jab) in zip(slots, nb[a]):
            idx[a, s] = b; J[a, s] = Jab
    return idx, J


@pytest.mark.parametrize("lattice,dims", [(0, (4, 3, 3)), (1, (3, 4, 2))])
def test_ell_branch_energy_and_field_against_brute_force(lattice, dims):
    rng = np.random.default_rng(11 + lattice)
    nx, ny, nz = dims
    N = nx * ny * nz
    spacing = (0.3, 0.3, 0.3) if lattice == 0 else (0.2725, 0.2725, 0.371)
    gm = rng.integers(-1, 2, size=(nx, ny)).astype(np.int32)
    gm[0, 0] = 0; gm[1, 1] = 1
    ku = 9.1e-23 * (1 + 0.3 * rng.standard_normal(2))
    axis = rng.standard_normal((2, 3)); axis /= np.linalg.norm(axis, axis=1, keepdims=True)
    pairs = _pairs_by_distance(dims, spacing, 1.6 * spacing[0], rng, gm)     # beyond the built-in shells on purpose
    idx, Jell = _ell_from_pairs(N, pairs, rng)
    S = rng.standard_normal((N, 3)); S /= np.linalg.norm(S, axis=1, keepdims=True)
    S32, B32 = S.astype(np.float32), rng.standard_normal((N, 3)).astype(np.float32)
    scale = -0.75
    o = orc.Oracle(orc.LatticeSpec(lattice=lattice, nx=nx, ny=ny, nz=nz, mu_s=MUS, J=(1e-21, 2e-21, 3e-21), grain_map=gm,
                                   grain_ku=ku, grain_axis=axis, ell_idx=idx, ell_J=Jell))
    o.set_spins(S32[:, 0], S32[:, 1], S32[:, 2])
    o.set_fields(np.zeros(N), B32[:, 0], B32[:, 1], B32[:, 2])
    o.set_field_scale(scale)
    mag = np.repeat((gm >= 0)[:, None, :], nz, axis=1).reshape(-1)
    Sd = S32.astype(np.float64) * mag[:, None]
    Bd = B32.astype(np.float64)
    gsite = np.repeat(gm[:, None, :], nz, axis=1).reshape(-1)

    def energy(Sx):
        E = -sum(Jab * float(Sx[a] @ Sx[b]) for (a, b), Jab in pairs.items())
        for a in np.nonzero(mag)[0]:
            E -= ku[gsite[a]] * float(Sx[a] @ axis[gsite[a]]) ** 2 + MUS * scale * float(Bd[a] @ Sx[a])
        return E

    E0 = energy(Sd)
    assert abs(o.energy() - E0) <= 1e-12 * abs(E0)
    # the field, term by term from the pair list: B_i = (1/mu_s) sum_j J_ij S_j + (2 k_u/mu_s)(S_i.e)e + s B_app,i
    want = np.zeros((N, 3))
    for (a, b), Jab in pairs.items():
        want[a] += Jab * Sd[b] / MUS; want[b] += Jab * Sd[a] / MUS
    for a in np.nonzero(mag)[0]:
        e = axis[gsite[a]]
        want[a] += 2.0 * ku[gsite[a]] / MUS * float(Sd[a] @ e) * e + scale * Bd[a]
    got = o.field(with_noise=False)
    assert np.allclose(got.T[mag], want[mag], rtol=1e-12, atol=1e-9)
    assert np.all(got[:, ~mag] == 0.0)
    # and it is minus the gradient of that energy
    h = 1e-3
    for a in rng.choice(np.nonzero(mag)[0], size=4, replace=False):
        for c in range(3):
            Sp, Sm = Sd.copy(), Sd.copy()
            Sp[a, c] += h; Sm[a, c] -= h
            g = -(energy(Sp) - energy(Sm)) / (2 * h) / MUS
            assert abs(got[c, a] - g) < 1e-7 * max(1.0, abs(g))


@pytest.mark.parametrize("lattice", [ai.SC, ai.L10])
@pytest.mark.parametrize("touching", [False, True])
def test_shell_ell_table_is_the_builtin_shells_bit_for_bit(lattice, touching):
    """asd_inputs.shell_ell_table (the shared helper the GPU ELL tests and bench.py --ell use) against the oracle's own
    shells: same bonds, same order of summation, so fields, energy and a Heun step agree bit for bit when both sides are
    given the same (fp32-representable) J."""
    w = ai.small_film(lattice, 9, 10, 4, tilt_deg=30.0, dt=1e-16)
    w.J = tuple(float(np.float32(x)) for x in w.J)
    if touching:                                           # grains that touch: bonds must be cut between different grains
        rng = np.random.default_rng(4)
        w.grain_map = rng.integers(-1, 3, size=(w.track_nx, w.ny)).astype(np.int32)
        w.grain_ku = (9.1e-23 * (1 + 0.2 * rng.standard_normal(3))).astype(np.float32)
        ax = rng.standard_normal((3, 3)); ax /= np.linalg.norm(ax, axis=1, keepdims=True)
        w.grain_axis = ax.astype(np.float32)
        sx, sy, sz = ai.tilted_spins(w.n_sites, 30.0, seed=8)
        mag = w.magnetic_mask().reshape(-1)
        w.sx, w.sy, w.sz = sx * mag, sy * mag, sz * mag
    idx, J = ai.shell_ell_table(w)
    a = oracle_from_workload(w)
    b = oracle_from_workload(w, ell_idx=idx, ell_J=J.astype(np.float64))
    assert np.array_equal(a.field(with_noise=False), b.field(with_noise=False))
    assert a.energy() == b.energy()
    a.step_heun(3); b.step_heun(3)
    assert np.array_equal(a.get_spins(), b.get_spins())
    # the table itself: every bond appears from both ends with the same J, no self bonds, none into a vacancy
    mag = w.magnetic_mask().reshape(-1)
    for l in range(w.n_sites):
        for s in range(idx.shape[1]):
            n = idx[l, s]
            if n < 0:
                assert J[l, s] == 0.0
                continue
            assert n != l and mag[l] and mag[n]
            back = np.nonzero(idx[n] == l)[0]
            assert len(back) == 1 and J[n, back[0]] == J[l, s]


# ---------------------------------------------------------------------------------------------------------------
# Magnetisation
# ---------------------------------------------------------------------------------------------------------------
def test_magnetisation_divides_by_the_magnetic_sites_and_bins_by_grain():
    w = ai.small_film(ai.L10, 14, 16, 3, tilt_deg=40.0)
    rng = np.random.default_rng(2)
    w.grain_map = rng.integers(-1, 5, size=(w.track_nx, w.ny)).astype(np.int32)      # grains 0..4, ~1/6 vacant
    w.grain_map[w.grain_map == 3] = -1                                              # grain 3 has no site at all
    w.grain_ku = np.full(5, 9.1e-23, dtype=np.float32)
    w.grain_axis = np.tile(np.array([[0.0, 0.0, 1.0]], dtype=np.float32), (5, 1))
    sx, sy, sz = ai.tilted_spins(w.n_sites, 40.0, seed=3)
    w.sx, w.sy, w.sz = sx, sy, sz                                                   # values on vacant sites must be ignored
    o = oracle_from_workload(w)
    o.step_heun(2)
    S = o.get_spins()                                                               # [3, N], 0 on vacant sites
    gsite = np.repeat(np.asarray(w.grain_map)[w.x0:w.x0 + w.nx][:, None, :], w.nz, axis=1).reshape(-1)
    mag = gsite >= 0
    assert 0 < mag.sum() < w.n_sites
    m, n = o.magnetisation()
    assert n == mag.sum()
    assert np.allclose(m, S[:, mag].mean(axis=1), rtol=0, atol=1e-14)
    assert not np.allclose(m, S.sum(axis=1) / w.n_sites, atol=1e-3)                 # dividing by N would be visible
    gm = o.grain_magnetisation()
    for g in range(5):
        sel = gsite == g
        want = S[:, sel].mean(axis=1) if sel.any() else np.zeros(3)
        assert np.allclose(gm[g], want, rtol=0, atol=1e-14), g


# ---------------------------------------------------------------------------------------------------------------
# Held demagnetising field (reading D3)
# ---------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("lattice,x0", [(ai.SC, 0), (ai.L10, 2)])
def test_held_field_is_demag_cells_added_to_the_applied_field_every_p_steps(lattice, x0):
    P, nsteps = 3, 7
    w = ai.small_film(lattice, 10, 12, 4, extra_track=6, tilt_deg=30.0, dt=1e-16, uniform_T=150.0)
    w.x0 = x0                                                    # window origin not on a macrocell boundary
    sx, sy, sz = ai.tilted_spins(w.n_sites, 30.0, seed=6)
    mag = w.magnetic_mask().reshape(-1)
    w.sx, w.sy, w.sz = sx * mag, sy * mag, sz * mag
    spacing = [a * 1e-9 for a in w.spacing_nm]
    a = oracle_from_workload(w)
    a.enable_demag(spacing)
    a.set_demag_every(P)
    b = oracle_from_workload(w)                                  # demag off: the field is injected through set_fields
    mx, my, mz = w.macro
    i, k, j = np.meshgrid(np.arange(w.nx), np.arange(w.nz), np.arange(w.ny), indexing="ij")
    ci = ((x0 + i) // mx - x0 // mx).reshape(-1); cj = (j // my).reshape(-1); ck = (k // mz).reshape(-1)
    probe = oracle_from_workload(w)
    probe.enable_demag(spacing)
    B0 = [np.asarray(w.Bx, np.float64), np.asarray(w.By, np.float64), np.asarray(w.Bz, np.float64)]
    worst = 0.0
    for n in range(nsteps):
        if n % P == 0:
            s = b.get_spins()
            probe.set_spins(s[0], s[1], s[2])
            cells = probe.demag_cells()                          # [dcx, dcy, dcz, 3], Tesla
            Bd = cells[ci, cj, ck]                               # per site
            b.set_fields(Bx=B0[0] + Bd[:, 0], By=B0[1] + Bd[:, 1], Bz=B0[2] + Bd[:, 2])
        a.step_heun(1); b.step_heun(1)
        worst = max(worst, float(np.abs(a.get_spins() - b.get_spins()).max()))
    # the only difference: set_fields rounds the summed field to fp32 (6e-8 relative of ~1 T => ~1e-11 in S per step)
    assert worst < 2e-10, worst
    # and the held scheme is not the default one (the field of every stage's configuration)
    c = oracle_from_workload(w)
    c.enable_demag(spacing)
    c.step_heun(nsteps)
    assert float(np.abs(a.get_spins() - c.get_spins()).max()) > 1e-8


# ---------------------------------------------------------------------------------------------------------------
# Reading D2 measured at cfg4's offsets
# ---------------------------------------------------------------------------------------------------------------
def test_d2_point_dipole_switch_over_error_at_cfg4_offsets():
    cell = np.array([7 * 0.2725e-9, 7 * 0.2725e-9, 5 * 0.371e-9])       # cfg4 macrocell: 7 x 7 x 5 L1_0 sites
    diag = float(np.linalg.norm(cell))
    # (a) term by term: just beyond the switch-over and out to the far end of the 127-cell window
    worst_rel = 0.0
    for R in [(22, 0, 0), (21, 6, 2), (16, 16, 0), (30, -9, 5), (60, 31, -5), (126, 0, 0), (126, 31, 5), (0, 31, 5), (13, 13, 13)]:
        Rm = np.array(R) * cell
        if np.linalg.norm(Rm) <= 12.0 * diag:
            continue
        got, want = orc.newell_tensor(cell, Rm), _quad_tensor(cell, Rm, order=6)
        scale = np.abs(want).max()
        worst_rel = max(worst_rel, float(np.abs(got - want).max() / scale))
        assert np.abs(want).max() < 2e-5                         # these terms are tiny next to the self term 1/3
    assert worst_rel < 2.5e-3, worst_rel                         # (cell / R)^2-sized quadrupole correction
    # (b) what it does to a cell's field: sum of (dipole - exact) over ALL far cells of the 127 x 32 x 6 window, uniform
    # magnetisation, seen from a centre cell and a corner cell.  Bound: 1e-4 of mu_0 M (the field scale of the film).
    x, wq = np.polynomial.legendre.leggauss(3)
    P = np.stack([a.ravel() for a in np.meshgrid(*[0.5 * c * x for c in cell], indexing="ij")], axis=1)
    Wt = np.prod(np.stack([a.ravel() for a in np.meshgrid(*[0.5 * c * wq for c in cell], indexing="ij")], axis=1), axis=1)
    ww = (Wt[:, None] * Wt[None, :]).ravel()
    dP = (P[None, :, :] - P[:, None, :]).reshape(-1, 3)           # r' - r for all quadrature pairs
    V = float(np.prod(cell))
    for tgt in [(63, 16, 3), (0, 0, 0)]:
        ci, cj, ck = np.meshgrid(np.arange(127), np.arange(32), np.arange(6), indexing="ij")
        Rc = np.stack([ci.ravel() - tgt[0], cj.ravel() - tgt[1], ck.ravel() - tgt[2]], axis=1) * cell
        far = np.linalg.norm(Rc, axis=1) > 12.0 * diag
        Rf = Rc[far]
        r = np.linalg.norm(Rf, axis=1)
        dip = np.zeros(6)                                          # the oracle's far-field formula, summed
        c = V / (4 * np.pi * r ** 3)
        dip[0] = (c * (1 - 3 * Rf[:, 0] ** 2 / r ** 2)).sum(); dip[1] = (c * (1 - 3 * Rf[:, 1] ** 2 / r ** 2)).sum()
        dip[2] = (c * (1 - 3 * Rf[:, 2] ** 2 / r ** 2)).sum(); dip[3] = (-3 * c * Rf[:, 0] * Rf[:, 1] / r ** 2).sum()
        dip[4] = (-3 * c * Rf[:, 0] * Rf[:, 2] / r ** 2).sum(); dip[5] = (-3 * c * Rf[:, 1] * Rf[:, 2] / r ** 2).sum()
        spot = np.array([orc.newell_tensor(cell, R) for R in Rf[:: max(1, len(Rf) // 50)]])
        assert np.all(np.isfinite(spot))
        exact = np.zeros(6)                                        # cuboid-cuboid by quadrature, summed
        for s0 in range(0, len(Rf), 512):
            rho = Rf[s0:s0 + 512, None, :] + dP[None, :, :]
            r2 = (rho ** 2).sum(-1); r5 = r2 ** 2.5
            for q, (a, b) in enumerate([(0, 0), (1, 1), (2, 2), (0, 1), (0, 2), (1, 2)]):
                kern = ((a == b) * r2 - 3.0 * rho[..., a] * rho[..., b]) / r5 / (4.0 * np.pi)
                exact[q] += float((kern * ww[None, :]).sum() / V)
        assert np.abs(dip - exact).max() < 1e-4, (tgt, dip, exact)
