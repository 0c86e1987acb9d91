"""Pins for the oracle's multiscale window (readings M1-M10 of
DESIGN.md sec. 14).  All `-m "not gpu"`.

P13  m_e(T): self-consistency residual; limits T -> 0 and T >= T_C; the closed forms next to T_C from the series of the
     Langevin function (below: m_e^2 = (5/3)(T_C/T - 1)(T/T_C)^3; above, in a field: Curie-Weiss m_e = (h/3)/(1 - T_C/T));
     the value of B(2.1696) SURVEY.md prints.
P14  macrospin: every cell of a uniformly magnetised mesh follows the closed-form damped precession with the
     temperature-dependent damping alpha = lambda (1 - T/3T_C); RK4 error falls 16-fold when the step halves; with
     anisotropy the small-angle frequency is gamma (B + 2 K_0 m_e^2 / M_S^0) / (1 + alpha^2).
P15  standing spin wave along a chain of cells (free ends): omega(k) = gamma [B + (2 A_0 m_e / M_S^0)(2/d^2)(1 - cos kd)]
     -- the stencil, its 1/d^2, the factor 2A/M_S of Eq. (4) and the m_e scaling A(T)/M_S(T) = A_0 m_e / M_S^0.
P16  mesh boundary, atomistic side: the field a mesh adds to the sites of the first / last plane is Eq. (2) with the
     mesh direction in place of the missing neighbour spins -- compared with a brute-force statement written here from
     the neighbour distances; nothing else changes.
P17  mesh boundary, micromagnetic side: the Laplacian's missing neighbour is the direction of the average atomistic
     spin in the stencil cell (and the frozen track's direction at the far end).
P18  a uniformly magnetised window (atoms and cells along the easy axis) at T = 0 does not move.
P19  shift by whole cells: every transfer of Fig. 1 exact on integer-valued spins.
"""
import math

import numpy as np
import pytest

import asd_inputs as ai
from oracle import asd_oracle as orc

G, MUB, KB = orc.GAMMA_E, orc.MU_B, orc.K_B


# ---------------------------------------------------------------------------------------------- P13
@pytest.mark.parametrize("T,Tc,h", [(300.0, 700.0, 0.0), (650.0, 700.0, 0.0), (699.0, 700.0, 0.0), (500.0, 710.0, 0.01),
                                    (800.0, 700.0, 0.05), (50.0, 700.0, 0.0)])
def test_p13_me_is_the_root_of_the_langevin_self_consistency(T, Tc, h):
    m = orc.mm_me(T, Tc, h * KB * T)
    assert 0.0 < m <= 1.0
    x = 3.0 * Tc / T * m + h
    assert abs((1.0 / math.tanh(x) - 1.0 / x) - m) < 1e-12


def test_p13_me_limits_and_closed_forms():
    assert orc.mm_me(0.0, 700.0) == 1.0
    b = 2100.0                                                                # B(x) -> 1 - 1/x: m = 1 - 1/(b m)
    assert abs(orc.mm_me(1.0, 700.0) - (1.0 - 1.0 / b - 1.0 / b ** 2)) < 1e-9
    for T in (700.0, 700.0001, 900.0):
        assert orc.mm_me(T, 700.0) == 0.0
    Ts = np.linspace(10.0, 699.0, 60)
    ms = np.array([orc.mm_me(T, 700.0) for T in Ts])
    assert np.all(np.diff(ms) < 0.0)
    for eps in (1e-3, 3e-3, 1e-2):                                            # just below T_C
        T = 700.0 * (1.0 - eps)
        closed = math.sqrt(5.0 / 3.0 * (700.0 / T - 1.0) * (T / 700.0) ** 3)
        assert abs(orc.mm_me(T, 700.0) / closed - 1.0) < 2.0 * eps
    for h in (1e-4, 1e-3):                                                    # above T_C in a field: Curie-Weiss
        T = 900.0
        assert abs(orc.mm_me(T, 700.0, h * KB * T) / ((h / 3.0) / (1.0 - 700.0 / T)) - 1.0) < 1e-4
    assert abs(orc.langevin(2.1696) - 0.56553) < 1e-5                          # SURVEY.md 8(c) P3's worked value
    assert abs(orc.langevin(1e-5) - (1e-5 / 3.0 - 1e-15 / 45.0)) < 1e-21       # x/3 - x^3/45


# ---------------------------------------------------------------------------------------------- helpers
def _window(lattice=ai.SC, mcx=(3, 3), atom_cells=2, ny=2, nz=2, macro=(2, 2, 2), lam=0.1, dt=1e-15, J=None,
            ku=0.0, decouple=False, every=1, Ms0=1.0e6, A0=1.0e-11, K0=0.0, Tc=700.0, extra_cells=0, n_grains=None):
    """One-grain [mesh | atoms | mesh] window.  decouple: the atomistic cells belong to another grain, so the meshes
    see no neighbour there (and the atoms none in the meshes)."""
    mx, my, mz = macro
    nx = atom_cells * mx
    x0 = mcx[0] * mx
    track_nx = x0 + nx + (mcx[1] + extra_cells) * mx
    gm = np.zeros((track_nx, ny), dtype=np.int32)
    ng = 2 if decouple else 1
    if decouple:
        gm[x0:x0 + nx, :] = 1
    if J is None:
        J = ai.workloads.J_SC if lattice == ai.SC else ai.workloads.J_L10
    spec = orc.LatticeSpec(lattice=lattice, nx=nx, ny=ny, nz=nz, lam=lam, dt=dt, J=J, track_nx=track_nx, x0=x0,
                           grain_map=gm, grain_ku=np.full(ng, ku), grain_axis=np.tile([0.0, 0.0, 1.0], (ng, 1)),
                           macro=macro)
    o = orc.Oracle(spec)
    ncx, ncy, _ = o.track_dims()
    cg = np.zeros((ncx, ncy), dtype=np.int32)
    if decouple:
        cg[x0 // mx:(x0 + nx) // mx, :] = 1
    sp = ai.workloads.A_SC if lattice == ai.SC else ai.workloads.A_L10
    assert o.mm_enable(mcx, every, Ms0, A0, np.full(ng, K0), np.full(ng, Tc), cg, [s * 1e-9 for s in sp]) == 0
    N = nx * ny * nz
    o.set_spins(np.zeros(N), np.zeros(N), np.ones(N))
    return o


def _uniform(o, side, v):
    v = np.asarray(v, dtype=np.float64) / np.linalg.norm(v)
    o.mm_set_m(side, np.broadcast_to(v, o.mm_shape(side) + (3,)))


# ---------------------------------------------------------------------------------------------- P14
def test_p14_macrospin_follows_the_closed_form_with_temperature_dependent_damping():
    lam, T, Tc, B = 0.1, 420.0, 700.0, 2.0
    o = _window(decouple=True, lam=lam, Tc=Tc)
    th0, ph0 = 0.6, 0.3
    v0 = [math.sin(th0) * math.cos(ph0), math.sin(th0) * math.sin(ph0), math.cos(th0)]
    for side in (0, 1):
        _uniform(o, side, v0)
        n = o.mm_shape(side)
        o.mm_set_fields(side, np.full(n, T), np.zeros(n), np.zeros(n), np.full(n, B))
    me, al = o.mm_params(0)
    alpha = lam * (1.0 - T / (3.0 * Tc))
    assert np.allclose(al, alpha, atol=1e-15) and np.allclose(me, orc.mm_me(T, Tc, 3.23 * MUB * B), atol=1e-14)
    h, n = 20e-15, 2000                                                       # the paper's 20 fs
    o.mm_step(n, h)
    t = n * h
    th = 2.0 * math.atan(math.tan(th0 / 2.0) * math.exp(-alpha * G * B * t / (1.0 + alpha ** 2)))
    ph = ph0 + G * B * t / (1.0 + alpha ** 2)
    ref = np.array([math.sin(th) * math.cos(ph), math.sin(th) * math.sin(ph), math.cos(th)])
    for side in (0, 1):
        m = o.mm_get_m(side)
        assert np.abs(m - ref).max() < 1e-9
        assert np.allclose(np.linalg.norm(m, axis=-1), 1.0, atol=1e-14)


def test_p14_rk4_is_fourth_order():
    errs = []
    for n in (25, 50, 100):
        o = _window(decouple=True, lam=0.1)
        _uniform(o, 0, [0.6, 0.2, 0.77])
        sh = o.mm_shape(0)
        o.mm_set_fields(0, np.full(sh, 300.0), np.zeros(sh), np.zeros(sh), np.full(sh, 10.0))
        alpha = 0.1 * (1.0 - 300.0 / 2100.0)
        T_total = 5e-12
        o.mm_step(n, T_total / n)
        v0 = np.array([0.6, 0.2, 0.77]); v0 /= np.linalg.norm(v0)
        th0, ph0 = math.acos(v0[2]), math.atan2(v0[1], v0[0])
        th = 2.0 * math.atan(math.tan(th0 / 2.0) * math.exp(-alpha * G * 10.0 * T_total / (1.0 + alpha ** 2)))
        ph = ph0 + G * 10.0 * T_total / (1.0 + alpha ** 2)
        ref = np.array([math.sin(th) * math.cos(ph), math.sin(th) * math.sin(ph), math.cos(th)])
        errs.append(np.abs(o.mm_get_m(0)[0, 0, 0] - ref).max())
    assert 11.0 < errs[0] / errs[1] < 22.0 and 11.0 < errs[1] / errs[2] < 22.0


def test_p14_anisotropy_field_scales_with_me_squared():
    lam, T, Tc, B, K0, Ms0 = 0.0, 500.0, 700.0, 0.5, 2.2e6, 5.2e5           # the paper's K and M_S
    o = _window(decouple=True, lam=lam, Tc=Tc, K0=K0, Ms0=Ms0)
    eps = 1e-3
    _uniform(o, 0, [eps, 0.0, 1.0])
    sh = o.mm_shape(0)
    o.mm_set_fields(0, np.full(sh, T), np.zeros(sh), np.zeros(sh), np.full(sh, B))
    me = orc.mm_me(T, Tc, 3.23 * MUB * B)
    Bk = 2.0 * K0 * me ** 2 / Ms0                                             # 2K(T)/M_S(T) = 2 K_0 m_e^3 / (M_S^0 m_e)
    f = o.mm_field(0)[1, 0, 0]
    assert abs(f[2] - (B + Bk / math.sqrt(1 + eps ** 2))) < 1e-12 and abs(f[0]) < 1e-15
    h, n = 5e-15, 400
    o.mm_step(n, h)
    m = o.mm_get_m(0)[1, 0, 0]
    assert abs(math.atan2(m[1], m[0]) - G * (B + Bk) * n * h) < 2e-6           # small-angle: omega = gamma (B + B_K)


# ---------------------------------------------------------------------------------------------- P15
@pytest.mark.parametrize("T", [0.0, 520.0])
@pytest.mark.parametrize("mode", [1, 3])
def test_p15_standing_spin_wave_dispersion(T, mode):
    ncell, A0, Ms0, B, Tc = 16, 1.118e-11, 1.109e6, 0.3, 700.0
    o = _window(mcx=(ncell, 2), atom_cells=1, ny=2, nz=2, macro=(2, 2, 2), lam=0.0, decouple=True, A0=A0, Ms0=Ms0, Tc=Tc)
    d = 2 * 0.3e-9
    k = mode * math.pi / (ncell * d)                                          # free ends: cos(k (a + 1/2) d)
    prof = np.cos(k * (np.arange(ncell) + 0.5) * d)
    eps = 1e-4
    m = np.zeros((ncell, 1, 1, 3)); m[..., 2] = 1.0; m[:, 0, 0, 0] = eps * prof
    m /= np.linalg.norm(m, axis=-1, keepdims=True)
    o.mm_set_m(0, m)
    sh = o.mm_shape(0)
    o.mm_set_fields(0, np.full(sh, T), np.zeros(sh), np.zeros(sh), np.full(sh, B))
    me = 1.0 if T == 0.0 else orc.mm_me(T, Tc, 3.23 * MUB * B)
    omega = G * (B + (2.0 * A0 * me / Ms0) * (2.0 / d ** 2) * (1.0 - math.cos(k * d)))
    h = 2e-15
    n = int(0.9 / (omega * h))
    o.mm_step(n, h)
    mt = o.mm_get_m(0)[:, 0, 0, :]
    amp = ((mt[:, 0] + 1j * mt[:, 1]) * prof).sum() / (prof ** 2).sum()
    assert abs(abs(amp) / eps - 1.0) < 1e-5                                   # the mode keeps its shape and amplitude
    assert abs(np.angle(amp) - omega * n * h) < 2e-5
    # nothing leaked into other modes
    assert np.abs((mt[:, 0] + 1j * mt[:, 1]) - amp * prof).max() < 1e-4 * eps


# ---------------------------------------------------------------------------------------------- P16
def _brute_ghost_field(ms, o, side):
    """Eq. (2) restricted to the neighbours that lie in a mesh, from distances: [3, nz, ny] Tesla on plane 0 / nx-1."""
    w = ms.w
    sp = np.asarray(w.spacing_nm)
    m = o.mm_get_m(side)
    col = m[-1] if side == 0 else m[0]                                        # the cell column next to the atoms
    i = 0 if side == 0 else w.nx - 1
    gi = w.x0 + i
    out = np.zeros((3, w.nz, w.ny))
    if w.lattice == ai.SC:
        shells = [(sp[0], w.J[0])]
    else:
        shells = [(sp[0], w.J[0]), (math.hypot(sp[0], sp[1]), w.J[2])]
    for j in range(w.ny):
        g = w.grain_map[gi, j]
        if g < 0:
            continue
        for k in range(w.nz):
            for dj in (-1, 0, 1):
                jj = j + dj
                if jj < 0 or jj >= w.ny:
                    continue
                dist = math.hypot(sp[0], dj * sp[1])
                Jij = [Jv for (r, Jv) in shells if abs(r - dist) < 1e-9]
                if not Jij:
                    continue
                gn = w.grain_map[gi + (-1 if side == 0 else 1), jj]
                if gn != g:
                    continue
                out[:, k, j] += Jij[0] / w.mu_s * col[jj // w.macro[1], k // w.macro[2]]
    return out


@pytest.mark.parametrize("lattice", [ai.SC, ai.L10])
def test_p16_mesh_directions_stand_in_for_the_missing_neighbour_spins(lattice):
    ms = ai.multiscale_film(lattice, atom_cells=3, mesh_cells=(2, 3), width_nm=7.2, nz=5, extra_cells=1,
                            macro=(3, 4, 2), pitch_nm=3.0, boundary_nm=0.6, tilt_deg=20.0)
    w = ms.w
    o = orc.from_workload(w)
    ai.apply_multiscale(o, ms)
    rng = np.random.default_rng(4)
    for side in (0, 1):
        v = rng.standard_normal(o.mm_shape(side) + (3,))
        o.mm_set_m(side, v / np.linalg.norm(v, axis=-1, keepdims=True))
    plain = orc.from_workload(w)
    d = (o.field() - plain.field()).reshape(3, w.nx, w.nz, w.ny)
    assert not d[:, 1:-1].any()                                               # only the two boundary planes feel the meshes
    for side, i in ((0, 0), (1, w.nx - 1)):
        ref = _brute_ghost_field(ms, o, side)
        assert np.abs(ref).max() > 1.0                                        # tens of Tesla of exchange field
        assert np.abs(d[:, i] - ref).max() < 1e-12 * np.abs(ref).max()
    # empty cells (grain boundaries wider than half a cell) have no direction and so add nothing
    m = o.mm_get_m(0)
    empty = ms.cell_grain[w.x0 // w.macro[0] - ms.mcx[0]:w.x0 // w.macro[0], :] < 0
    assert empty.any() and not m[empty].any()


# ---------------------------------------------------------------------------------------------- P17
def test_p17_micromagnetic_side_sees_the_average_atomistic_direction_and_the_track():
    A0, Ms0, Tc = 1.118e-11, 1.109e6, 700.0
    o = _window(mcx=(3, 2), atom_cells=2, ny=4, nz=2, macro=(2, 2, 2), A0=A0, Ms0=Ms0, Tc=Tc, extra_cells=2)
    for side in (0, 1):
        _uniform(o, side, [0.0, 0.0, 1.0])
    N = o.N
    d = 0.6e-9
    u = np.array([0.48, -0.6, 0.64])
    # atoms along u: two opposite tilts inside every stencil cell whose mean direction is u
    t = np.cross(u, [0.0, 0.0, 1.0]); t /= np.linalg.norm(t)
    S = np.zeros((3, 4, 2, 4))
    S[:, :, :, 0::2] = (0.8 * u + 0.6 * t)[:, None, None, None]
    S[:, :, :, 1::2] = (0.8 * u - 0.6 * t)[:, None, None, None]
    o.set_spins(*[S[a].reshape(-1) for a in range(3)])
    u32 = S.astype(np.float32).astype(np.float64)[:, 0, 0, :2].sum(axis=1); u32 /= np.linalg.norm(u32)
    z = np.array([0.0, 0.0, 1.0])
    pref = 2.0 * A0 * 1.0 / Ms0 / d ** 2                                      # T = 0: m_e = 1
    BL, BR = o.mm_field(0), o.mm_field(1)
    assert np.abs(BL[-1] - pref * (u32 - z)).max() < 1e-9 * pref              # trailing mesh, cells next to the atoms
    assert np.abs(BR[0] - pref * (u32 - z)).max() < 1e-9 * pref               # leading mesh, likewise
    assert not BL[:-1].any() and not BR[1:].any()                             # uniform elsewhere; track ahead is +z too
    # the far end of the leading mesh is coupled to the frozen track ahead
    ncell = int(np.prod(o.track_dims()))
    v = np.tile(np.array([0.3, 0.0, 0.4], dtype=np.float32), (ncell, 1))      # direction (0.6, 0, 0.8), |v| = 0.5
    o.track_set_init(v)
    BR = o.mm_field(1)
    assert np.abs(BR[-1] - pref * (np.array([0.6, 0.0, 0.8]) - z)).max() < 1e-6 * pref
    assert not BR[1:-1].any()
    # the trailing mesh starts at the track's first cell: nothing beyond it
    assert not o.mm_field(0)[0].any()


# ---------------------------------------------------------------------------------------------- P18
def test_p18_uniform_window_along_the_easy_axis_is_stationary():
    o = _window(lattice=ai.L10, mcx=(2, 2), atom_cells=2, ny=4, nz=3, macro=(2, 2, 3), ku=9.1e-23, K0=2.2e6, every=3)
    for side in (0, 1):
        _uniform(o, side, [0.0, 0.0, 1.0])
    S0 = o.get_spins().copy()
    o.step_heun(7)
    assert np.array_equal(o.get_spins(), S0)
    for side in (0, 1):
        m = o.mm_get_m(side)
        assert np.array_equal(m[..., 2], np.ones(m.shape[:-1])) and not m[..., :2].any()
    # and a tilted mesh drags the boundary atoms with it (the coupling is live)
    _uniform(o, 0, [0.3, 0.0, 1.0])
    o.step_heun(3)
    d = np.abs(o.get_spins() - S0).reshape(3, 4, 3, 4)
    assert d[:, 0].max() > 1e-4 and d[:, 0].max() > 20 * d[:, 2].max()


# ---------------------------------------------------------------------------------------------- P19
def test_p19_shift_by_whole_cells_moves_everything_exactly():
    ms = ai.multiscale_film(ai.SC, atom_cells=4, mesh_cells=(3, 3), width_nm=7.2, nz=5, extra_cells=4,
                            macro=(3, 4, 2), pitch_nm=3.0, boundary_nm=0.6, t_peak=0.0, t_ambient=0.0)
    w = ms.w
    mx, my, mz = w.macro
    N = w.n_sites
    gidx = np.arange(N, dtype=np.int64)
    mag = w.magnetic_mask().reshape(-1)
    w.sx = ((gidx % 4093) * mag).astype(np.float32)
    w.sy = ((gidx // 4093) * mag).astype(np.float32)
    w.sz = ((gidx % 977 + 1) * mag).astype(np.float32)
    o = orc.from_workload(w)
    ai.apply_multiscale(o, ms)                                                 # T = 0 everywhere: m_e = 1
    rng = np.random.default_rng(9)
    mL = rng.standard_normal(o.mm_shape(0) + (3,)); mL /= np.linalg.norm(mL, axis=-1, keepdims=True)
    mR = rng.standard_normal(o.mm_shape(1) + (3,)); mR /= np.linalg.norm(mR, axis=-1, keepdims=True)
    o.mm_set_m(0, mL); o.mm_set_m(1, mR)
    mL, mR = o.mm_get_m(0), o.mm_get_m(1)                                      # empty cells zeroed
    ncx, ncy, ncz = o.track_dims()
    init = rng.standard_normal((ncx, ncy, ncz, 3)).astype(np.float32)
    o.track_set_init(init.reshape(-1, 3))
    assert o.shift_window(mx + 1) != 0 and o.shift_window(4 * mx) != 0         # whole cells only; not more than a mesh
    S = o.get_spins().reshape(3, w.nx, w.nz, w.ny)
    pc = 2
    p = pc * mx
    assert o.shift_window(p) == 0
    c = o.counters()
    assert c["x0"] == w.x0 + p and c["shift"] == 1
    S2 = o.get_spins().reshape(3, w.nx, w.nz, w.ny)
    assert np.array_equal(S2[:, :w.nx - p], S[:, p:])                          # the atoms that stay
    L2, R2 = o.mm_get_m(0), o.mm_get_m(1)
    assert np.array_equal(L2[:1], mL[pc:]) and np.array_equal(R2[:1], mR[pc:])  # the cells that stay
    cxL, cxA, cxR = 0, w.x0 // mx, (w.x0 + w.nx) // mx
    gm = w.grain_map
    # trailing mesh -> track: (m_e = 1) m times the number of magnetic sites of the cell
    _, cnt, sm = o.track_get()
    cnt, sm = cnt.reshape(ncx, ncy, ncz), sm.reshape(ncx, ncy, ncz, 3)
    for a in range(pc):
        for b in range(ncy):
            for cz in range(ncz):
                cols = (gm[(cxL + a) * mx:(cxL + a + 1) * mx, b * my:(b + 1) * my] >= 0).sum()
                n = cols * (min((cz + 1) * mz, w.nz) - cz * mz) if ms.cell_grain[cxL + a, b] >= 0 else 0
                assert cnt[cxL + a, b, cz] == n
                assert np.allclose(sm[cxL + a, b, cz], mL[a, b, cz] * n, atol=1e-12)
    assert cnt[pc:].sum() == 0
    # outgoing atoms -> trailing mesh: direction of the Eq. (6) sum
    for a in range(pc):
        for b in range(ncy):
            for cz in range(ncz):
                blk = S[:, a * mx:(a + 1) * mx, cz * mz:(cz + 1) * mz, b * my:(b + 1) * my].reshape(3, -1).sum(axis=1)
                got = L2[3 - pc + a, b, cz]
                if ms.cell_grain[cxA + a, b] < 0:
                    assert not got.any()
                else:
                    assert np.allclose(got, blk / np.linalg.norm(blk), atol=1e-14)
    # leading mesh -> incoming atoms: |m_e m| = 1, so every magnetic site lies exactly along its cell's direction;
    # a magnetic site over an empty cell has M = 0 to reproduce: theta_max = pi, any direction (reading S3)
    n_free = 0
    for i in range(w.nx - p, w.nx):
        a = (i - (w.nx - p)) // mx
        for j in range(w.ny):
            vac = gm[w.x0 + p + i, j] < 0
            for k in range(w.nz):
                want = np.zeros(3) if vac else mR[a, j // my, k // mz]
                if not vac and not want.any():
                    assert abs(np.linalg.norm(S2[:, i, k, j]) - 1.0) < 1e-14
                    n_free += 1
                    continue
                assert np.allclose(S2[:, i, k, j], want, atol=1e-14)
    assert n_free < 0.2 * p * w.ny * w.nz
    # track ahead -> leading mesh
    for a in range(pc):
        for b in range(ncy):
            for cz in range(ncz):
                got = R2[3 - pc + a, b, cz]
                if ms.cell_grain[cxR + 3 + a, b] < 0:
                    assert not got.any()
                else:
                    v = init[cxR + 3 + a, b, cz].astype(np.float64)
                    assert np.allclose(got, v / np.linalg.norm(v), atol=1e-14)


def test_mm_enable_rejects_misaligned_windows_and_recipe_is_consistent():
    spec = orc.LatticeSpec(lattice=ai.SC, nx=8, ny=4, nz=2, track_nx=40, x0=7, macro=(4, 2, 2),
                           grain_map=np.zeros((40, 4), dtype=np.int32), grain_ku=np.zeros(1),
                           grain_axis=np.array([[0.0, 0.0, 1.0]]))
    o = orc.Oracle(spec)
    cg = np.zeros((10, 2), dtype=np.int32)
    args = (1, 1e6, 1e-11, np.zeros(1), np.full(1, 700.0), cg, [3e-10] * 3)
    assert o.mm_enable((1, 1), *args) == 1                                     # x0 not on a cell boundary
    spec.x0 = 8
    o = orc.Oracle(spec)
    assert o.mm_enable((3, 1), *args) == 1                                     # trailing mesh starts before the track
    assert o.mm_enable((2, 7), *args) == 1                                     # leading mesh ends after it
    assert o.mm_enable((2, 6), *args) == 0
    # the recipe: continuum limits of Eq. (9)-(10)
    Ms0, A, K = ai.multiscale.continuum_parameters(ai.SC, (6.71e-21, 0, 0), (0.3, 0.3, 0.3), 3.23 * MUB, np.array([9.1e-23]))
    assert abs(A[0] - 6.71e-21 / 0.6e-9) < 1e-20 and A[0] == A[1] == A[2]      # A_SC = J / 2a
    assert abs(Ms0 - 3.23 * MUB / 2.7e-29) < 1.0 and abs(K[0] - 9.1e-23 / 2.7e-29) < 1e-3
    J = 3.77e-21
    _, A, _ = ai.multiscale.continuum_parameters(ai.L10, (J, J, J), (0.2725, 0.2725, 0.371), 3.23 * MUB, np.array([0.0]))
    assert abs(A[0] - 3.0 * J / (2.0 * 0.371e-9)) < 1e-20                      # Eq. (10) with a -> the plane spacing
    cgm = ai.multiscale.cell_grain_map(np.array([[0, 0, -1, 1], [0, -1, -1, 1], [2, 2, 2, -1], [2, 2, -1, -1]]), (2, 2, 1))
    assert cgm.tolist() == [[0, -1], [2, -1]] or cgm.tolist() == [[0, 1], [2, -1]]


def test_passes_over_the_track_with_a_multiscale_window():
    """Readings T1' / T2': at the end of a pass the cells of both meshes go to the track as m_e m on
    their magnetic sites, next to the atoms' Eq. (6) sums; the next pass starts with the meshes along the track they lie
    over and the atoms regenerated from it.  Integer-valued atoms, T = 0 (m_e = 1): exact."""
    ms = ai.multiscale_film(ai.SC, atom_cells=3, mesh_cells=(2, 3), width_nm=7.2, nz=5, extra_cells=3,
                            macro=(3, 4, 2), pitch_nm=3.0, boundary_nm=0.6, t_peak=0.0, t_ambient=0.0)
    w = ms.w
    mx, my, mz = w.macro
    gidx = np.arange(w.n_sites, dtype=np.int64)
    mag = w.magnetic_mask().reshape(-1)
    w.sx = ((gidx % 61) * mag).astype(np.float32)
    w.sy = ((gidx // 61 % 7) * mag).astype(np.float32)
    w.sz = ((gidx % 13 + 1) * mag).astype(np.float32)
    o = orc.from_workload(w)
    ai.apply_multiscale(o, ms)
    rng = np.random.default_rng(17)
    mesh = []
    for side in (0, 1):
        v = rng.standard_normal(o.mm_shape(side) + (3,)); v /= np.linalg.norm(v, axis=-1, keepdims=True)
        o.mm_set_m(side, v)
        mesh.append(o.mm_get_m(side))
    ncx, ncy, ncz = o.track_dims()
    S = o.get_spins().reshape(3, w.nx, w.nz, w.ny)
    assert o.track_end_pass() == 0
    mean, cnt, sm = o.track_get()
    cnt, sm = cnt.reshape(ncx, ncy, ncz), sm.reshape(ncx, ncy, ncz, 3)
    gm = w.grain_map
    cxA = w.x0 // mx
    for side, cx0 in ((0, cxA - 2), (1, cxA + 3)):
        for a in range(ms.mcx[side]):
            for b in range(ncy):
                for cz in range(ncz):
                    cols = (gm[(cx0 + a) * mx:(cx0 + a + 1) * mx, b * my:(b + 1) * my] >= 0).sum()
                    n = cols * (min((cz + 1) * mz, w.nz) - cz * mz) if ms.cell_grain[cx0 + a, b] >= 0 else 0
                    assert cnt[cx0 + a, b, cz] == n
                    assert np.allclose(sm[cx0 + a, b, cz], mesh[side][a, b, cz] * n, atol=1e-12)
    for a in range(3):                                     # the atoms' cells: Eq. (6) sums, exact
        for b in range(ncy):
            for cz in range(ncz):
                blk = S[:, a * mx:(a + 1) * mx, cz * mz:(cz + 1) * mz, b * my:(b + 1) * my].reshape(3, -1).sum(axis=1)
                assert np.array_equal(sm[cxA + a, b, cz], blk)
    assert cnt[cxA + 6:].sum() == 0 and cnt[:cxA - 2].sum() == 0
    # next pass, one cell further along: the meshes lie along the committed track (or what lay ahead where nothing was written)
    x1 = w.x0 + mx
    assert o.track_begin_pass(x1 + 1) == 1                 # whole cells only
    assert o.track_begin_pass(x1) == 0
    c = o.counters()
    assert c["pass"] == 1 and c["x0"] == x1
    _, cnt2, _ = o.track_get()
    assert not cnt2.any()
    mean = mean.reshape(ncx, ncy, ncz, 3)
    for side, cx0 in ((0, x1 // mx - 2), (1, (x1 + w.nx) // mx)):
        m = o.mm_get_m(side)
        for a in range(ms.mcx[side]):
            for b in range(ncy):
                for cz in range(ncz):
                    if ms.cell_grain[cx0 + a, b] < 0:
                        assert not m[a, b, cz].any()
                    elif cnt[cx0 + a, b, cz] > 0:
                        v = mean[cx0 + a, b, cz]
                        assert np.allclose(m[a, b, cz], v / np.linalg.norm(v), atol=1e-6)   # init_mean is fp64 here; exact up to the division
                    else:
                        assert np.array_equal(m[a, b, cz], [0.0, 0.0, 1.0])                 # the default track ahead: +z
    R = o.get_spins().reshape(3, w.nx, w.nz, w.ny)
    assert np.allclose(np.linalg.norm(R, axis=0)[np.broadcast_to((gm[x1:x1 + w.nx] >= 0)[:, None, :], R.shape[1:])], 1.0, atol=1e-14)
    # the dynamics go on
    o.step_heun(2)


# ---------------------------------------------------------------------------------------------- M9 (who steps when)
def test_m9_mesh_takes_one_step_of_every_dt_per_every_heun_steps():
    """Cadence and step length from a closed form: a decoupled, uniformly magnetised mesh in a field is a macrospin
    (P14); after n Heun steps with `every` = P it has precessed by gamma B / (1 + alpha^2) x ceil(n / P) P dt."""
    lam, T, Tc, B, dt = 0.1, 300.0, 700.0, 5.0, 1e-15
    for every, n in ((1, 7), (4, 9), (5, 10), (20, 1)):
        o = _window(decouple=True, lam=lam, Tc=Tc, every=every, dt=dt)
        th0 = 0.5
        for side in (0, 1):
            _uniform(o, side, [math.sin(th0), 0.0, math.cos(th0)])
            sh = o.mm_shape(side)
            o.mm_set_fields(side, np.full(sh, T), np.zeros(sh), np.zeros(sh), np.full(sh, B))
        o.step_heun(n)
        alpha = lam * (1.0 - T / (3.0 * Tc))
        t = -(-n // every) * every * dt
        m = o.mm_get_m(0)[1, 0, 0]
        assert abs(math.atan2(m[1], m[0]) - G * B * t / (1.0 + alpha ** 2)) < 1e-9, (every, n)
        th = 2.0 * math.atan(math.tan(th0 / 2.0) * math.exp(-alpha * G * B * t / (1.0 + alpha ** 2)))
        assert abs(math.acos(m[2]) - th) < 1e-9


def test_m9_atoms_see_the_mesh_directions_of_the_exchange_instant():
    """The boundary data go both ways from the configurations at the exchange instant, BEFORE the meshes step: during the
    following Heun steps the atoms see m(t_n), not m(t_n + every dt).  A window whose meshes rotate a lot in one step
    (30 T on the cells only) and a twin whose meshes cannot move (no field there) leave the atoms identical."""
    def make(mesh_field):
        o = _window(lattice=ai.SC, mcx=(2, 2), atom_cells=2, ny=4, nz=2, macro=(2, 2, 2), every=3, K0=0.0, A0=0.0)
        for side in (0, 1):
            _uniform(o, side, [0.5, 0.2, 0.84])
            sh = o.mm_shape(side)
            o.mm_set_fields(side, np.zeros(sh), np.zeros(sh), np.full(sh, mesh_field), np.zeros(sh))
        rng = np.random.default_rng(2)
        v = rng.standard_normal((o.N, 3)); v /= np.linalg.norm(v, axis=1, keepdims=True)
        o.set_spins(v[:, 0], v[:, 1], v[:, 2])
        return o
    a, b = make(30.0), make(0.0)
    m0 = b.mm_get_m(0).copy()
    a.step_heun(3); b.step_heun(3)                                             # one exchange, one mesh step, three Heun steps
    assert np.abs(a.mm_get_m(0) - m0).max() > 5e-3                             # a's meshes did turn ...
    assert np.array_equal(b.mm_get_m(0), m0)
    assert np.array_equal(a.get_spins(), b.get_spins())                        # ... and its atoms never saw it
    a.step_heun(1); b.step_heun(1)                                             # next exchange: now they do
    assert np.abs(a.get_spins() - b.get_spins()).max() > 1e-6
