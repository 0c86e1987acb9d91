"""Pins P2, P3, P4, P6, P7 for the oracle's dynamics (Eq. (1)-(3), (8)-(11)).

Each test compares the oracle with a closed form the paper or textbook mathematics fixes -- never
with a re-typed copy of the oracle's own formula.
"""
import math

import numpy as np
import pytest

from oracle import asd_oracle as orc
from tests.helpers import single_grain_spec

G = orc.GAMMA_E
MUS = 3.23 * orc.MU_B


def _single_spin(theta0, B, lam, dt, nsteps, start=None):
    o = orc.Oracle(single_grain_spec(0, 1, 1, 1, lam=lam, dt=dt, J=(0, 0, 0), mu_s=MUS))
    if start is None:
        start = (math.sin(theta0), 0.0, math.cos(theta0))
    o.set_spins([start[0]], [start[1]], [start[2]])
    o.set_fields(T=[0.0], Bx=[0.0], By=[0.0], Bz=[B])
    o.step_heun(nsteps)
    s = o.get_spins()[:, 0]
    return s


def test_p2_single_spin_damped_precession_closed_form():
    """Eq. (1), T = 0, B || z: phi(t) = +gamma B t/(1+lam^2); tan(theta/2) = tan(theta0/2) exp(-lam gamma B t/(1+lam^2))."""
    B, lam = 10.0, 0.1
    start = (0.6, 0.0, 0.8)                 # the oracle takes fp32 inputs: use the angle of the ROUNDED start
    s32 = np.array(start, dtype=np.float32).astype(np.float64)
    theta0 = math.atan2(s32[0], s32[2])
    t_end = 2.0e-12
    errs = []
    for nsteps in (1000, 2000, 4000):
        dt = t_end / nsteps
        s = _single_spin(theta0, B, lam, dt, nsteps, start=start)
        gp = G / (1.0 + lam * lam)
        phi = gp * B * t_end
        th = 2.0 * math.atan(math.tan(theta0 / 2.0) * math.exp(-lam * gp * B * t_end))
        exact = np.array([math.sin(th) * math.cos(phi), math.sin(th) * math.sin(phi), math.cos(th)])
        errs.append(np.abs(s - exact).max())
        assert abs(np.linalg.norm(s) - 1.0) < 1e-14
    assert errs[0] < 8e-6
    # Heun is second order: halving dt divides the global error by 4
    assert 3.6 < errs[0] / errs[1] < 4.4
    assert 3.6 < errs[1] / errs[2] < 4.4


def test_p2_sense_of_precession():
    """At S = x, B = B z: dS/dt = +gamma' B y  (Eq. (1) with gamma > 0)."""
    s = _single_spin(math.pi / 2, 1.0, 0.0, 1e-15, 1)
    assert s[1] > 0 and abs(s[1] - G * 1e-15) < 1e-8
    # damping pulls towards +B
    s = _single_spin(math.pi / 2, 1.0, 0.5, 1e-15, 1)
    assert s[2] > 0


@pytest.mark.parametrize("lam", [0.1, 1.0])
def test_p3_langevin_equilibrium(lam):
    """Isolated spins in B at temperature T: <cos theta> = coth x - 1/x, x = mu_s B / kB T  (B(x) of P:38).
    lam = 1 discriminates the sigma normalisation and the same-noise-in-both-stages rule
    (wrong variants give ~0.77 instead of 0.5655)."""
    B, T = 10.0, 10.0
    x = MUS * B / (orc.K_B * T)
    L = 1.0 / math.tanh(x) - 1.0 / x
    nx, ny, nz = 32, 32, 24
    dt = 2e-15 if lam >= 1.0 else 1e-14      # O(dt) bias grows with lam
    o = orc.Oracle(single_grain_spec(0, nx, ny, nz, lam=lam, dt=dt, J=(0, 0, 0), mu_s=MUS, seed=11))
    N = nx * ny * nz
    o.set_spins(np.zeros(N), np.zeros(N), np.ones(N))
    o.set_fields(T=np.full(N, T), Bx=np.zeros(N), By=np.zeros(N), Bz=np.full(N, B))
    relax = int(4.0 * (1 + lam * lam) / (lam * G * B * dt))      # 4 relaxation times
    o.step_heun(min(relax, 12000))
    acc, ns = 0.0, 0
    for _ in range(8):
        o.step_heun(max(50, relax // 8))
        acc += o.get_spins()[2].mean()
        ns += 1
    assert abs(acc / ns - L) < 0.004, (acc / ns, L)


def _spin_wave_omega(lattice, dims, J, q, ku, Bz, dt=2e-17, nsteps=1500, eps=1e-3):
    """Measured precession frequency of a plane spin wave with phase advance q = (qx,qy,qz) per site."""
    nx, ny, nz = dims
    o = orc.Oracle(single_grain_spec(lattice, nx, ny, nz, pbc=(1, 1, 1), ku=ku, lam=0.0, dt=dt, J=J, mu_s=MUS))
    i, k, j = np.meshgrid(np.arange(nx), np.arange(nz), np.arange(ny), indexing="ij")
    ph = (q[0] * i + q[1] * j + q[2] * k).reshape(-1)
    N = nx * ny * nz
    o.set_spins(eps * np.cos(ph), eps * np.sin(ph), np.sqrt(1 - eps * eps) * np.ones(N))
    o.set_fields(T=np.zeros(N), Bx=np.zeros(N), By=np.zeros(N), Bz=np.full(N, Bz))
    total, prev = 0.0, 0.0
    for _ in range(nsteps // 50):
        o.step_heun(50)
        s = o.get_spins()
        cur = math.atan2(s[1, 0], s[0, 0])
        d = cur - prev
        d -= 2 * math.pi * round(d / (2 * math.pi))
        total += d
        prev = cur
    return total / (dt * (nsteps // 50) * 50)


def test_p4_spin_wave_dispersion_sc():
    """omega(k) = gamma [B + 2ku/mu_s + (1/mu_s) sum_j J_j (1 - cos k.r_j)]: exchange normalisation (Eq. (2))."""
    J, ku, Bz = 6.71e-21, 9.1e-23, 2.0
    n = 8
    q = (2 * math.pi / n * 1, 2 * math.pi / n * 2, 2 * math.pi / n * 3)
    w = _spin_wave_omega(0, (n, n, n), (J, 0, 0), q, ku, Bz)
    exact = G * (Bz + 2 * ku / MUS + (2 * J / MUS) * sum(1 - math.cos(x) for x in q))
    assert abs(w / exact - 1.0) < 1e-3


def test_p4_spin_wave_dispersion_l10_shells_distinguish_geometry():
    """L1_0 Fe sublattice: J1 on (+-1,0,0),(0,+-1,0); J2 on (0,0,+-1); J3 on (+-1,+-1,0)."""
    J = (5.0e-21, 2.0e-21, 0.8e-21)
    n = 8
    q = (2 * math.pi / n * 1, 2 * math.pi / n * 2, 2 * math.pi / n * 3)
    w = _spin_wave_omega(1, (n, n, n), J, q, 0.0, 1.0)
    ex = (2 * J[0] * ((1 - math.cos(q[0])) + (1 - math.cos(q[1]))) + 2 * J[1] * (1 - math.cos(q[2]))
          + 2 * J[2] * ((1 - math.cos(q[0] + q[1])) + (1 - math.cos(q[0] - q[1]))))
    exact = G * (1.0 + ex / MUS)
    assert abs(w / exact - 1.0) < 1e-3


def test_p4_small_k_limit_matches_paper_exchange_stiffness():
    """Eq. (11): omega - omega0 = lambda_ex gamma M_S k^2, lambda_ex = 2A/(mu0 M_S^2)  (in Tesla: (2A/M_S) k^2),
    with A_SC = J/2a, mu_S = M_S a^3 and A_L10 = 3J/2a, mu_S = M_S a^3/2."""
    J = 3.77e-21
    n = 64
    q = 2 * math.pi / n
    # SC, wave along x, lattice constant a
    a = 0.5e-9
    w = _spin_wave_omega(0, (n, 3, 3), (J, 0, 0), (q, 0, 0), 0.0, 1.0, nsteps=1000)
    Ms = MUS / a ** 3
    A = J / (2 * a)
    k = q / a
    assert abs((w - G * 1.0) / (G * (2 * A / Ms) * k * k) - 1.0) < 2e-3
    # L1_0, uniform J, wave along the cell's [100] = sublattice [110]: phase advance q on both sublattice axes;
    # in-plane spacing a/sqrt2 => k = q*sqrt2/(a/sqrt2)... k.r for a nn step is k a/2 = q  => k = 2q/a
    w = _spin_wave_omega(1, (n, n, 3), (J, J, J), (q, q, 0), 0.0, 1.0, nsteps=1000)
    Ms = MUS / (a ** 3 / 2)
    A = 3 * J / (2 * a)
    k = 2 * q / a
    assert abs((w - G * 1.0) / (G * (2 * A / Ms) * k * k) - 1.0) < 3e-3


def test_p6_p7_energy_monotone_and_unit_norm_at_zero_temperature():
    import asd_inputs as ai
    from tests.helpers import oracle_from_workload
    for lattice in (ai.SC, ai.L10):
        w = ai.small_film(lattice, 14, 12, 5, spot=False, uniform_T=0.0, bz=-0.8, tilt_deg=40.0, dt=1e-15)
        o = oracle_from_workload(w)
        mag = w.magnetic_mask().reshape(-1)
        E = [o.energy()]
        for _ in range(40):
            o.step_heun(5)
            E.append(o.energy())
            s = o.get_spins()
            nrm = np.sqrt((s ** 2).sum(axis=0))
            assert np.all(np.abs(nrm[mag] - 1.0) < 1e-14)
            assert np.all(nrm[~mag] == 0.0)
        E = np.array(E)
        assert np.all(np.diff(E) <= 1e-12 * abs(E[0]))
        assert E[-1] < E[0] - 1e-3 * abs(E[0])
