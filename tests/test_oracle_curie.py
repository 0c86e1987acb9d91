"""Pin P8: the emergent Curie temperature of the oracle's bulk simple-cubic Heisenberg model,
T_C = eps z J / (3 k_B) with eps_SC = 0.72, z = 6  =>  T_C = 1.44 J / k_B   (Eq. (8)).

This is a whole-loop check: noise amplitude, exchange normalisation (Eq. (2)), the same-noise rule and
the integrator all have to be right for the order-disorder transition to sit where the paper says.

Two tiers (P8):
  * always on (about 20 s): the transition is BRACKETED by 0.85 T_C and 1.15 T_C.  A thermal field wrong by a
    factor sqrt(2) or sqrt(1 + lambda^2) in amplitude moves the apparent T_C by a factor 2 and fails this.
  * opt-in (ASD_SLOW=1, about 10 min on 8 cores): T_C from a power-law fit, extrapolated linearly to dt -> 0
    (stochastic Heun has an O(dt) bias of the stationary distribution: +6 % at dt = 1 fs, lambda = 1), within
    3 % of 1.44 J/k_B.  Last recorded result: DESIGN.md sec. 3.
"""
import os

import numpy as np
import pytest

from oracle import asd_oracle as orc
from tests.helpers import single_grain_spec

J = 6.71e-21                      # BASELINE configs[0]
MUS = 3.23 * orc.MU_B
TC_PAPER = 1.44 * J / orc.K_B     # 699.8 K


def _bulk(L, dt, lam=1.0, seed=1):
    N = L ** 3
    o = orc.Oracle(single_grain_spec(0, L, L, L, pbc=(1, 1, 1), lam=lam, dt=dt, J=(J, 0, 0), mu_s=MUS, seed=seed))
    o.set_spins(np.zeros(N), np.zeros(N), np.ones(N))
    return o, N


def _mean_m(o, N, T, n_relax, n_avg, n_samples=16):
    z = np.zeros(N)
    o.set_fields(T=np.full(N, T), Bx=z, By=z, Bz=z)
    o.step_heun(n_relax)
    acc = []
    for _ in range(n_samples):
        o.step_heun(max(1, n_avg // n_samples))
        m, _n = o.magnetisation()
        acc.append(np.linalg.norm(m))
    return float(np.mean(acc))


def test_p8_transition_is_bracketed_by_the_paper_curie_temperature():
    o, N = _bulk(12, 5e-16)
    below = _mean_m(o, N, 0.85 * TC_PAPER, 1500, 1500)
    above = _mean_m(o, N, 1.15 * TC_PAPER, 2500, 1500)
    # 3-D Heisenberg: m(0.85 T_C) ~ 0.15^0.36 ~ 0.5 (+ finite size); far above T_C only the 1/sqrt(N) remnant
    assert 0.42 < below < 0.66, below
    assert above < 0.16, above


@pytest.mark.skipif(os.environ.get("ASD_SLOW") != "1", reason="about 10 minutes; set ASD_SLOW=1")
def test_p8_curie_temperature_extrapolated_to_zero_time_step():
    from scipy.optimize import curve_fit
    temps = np.arange(575.0, 751.0, 25.0)
    tc = []
    for dt, nsteps in ((5e-16, 8000), (2.5e-16, 16000)):
        o, N = _bulk(24, dt)
        m = np.array([_mean_m(o, N, T, nsteps // 2, nsteps // 2) for T in temps])
        sel = m > 0.25
        f = lambda T, Tc, b: np.clip(1.0 - T / Tc, 1e-12, None) ** b
        p, _cov = curve_fit(f, temps[sel], m[sel], p0=(720.0, 0.36))
        print("dt", dt, "m(T)", np.round(m, 4), "fit T_C, beta", p)
        tc.append(p[0])
    tc0 = 2.0 * tc[1] - tc[0]                      # linear extrapolation dt -> 0
    print("T_C(dt->0) =", tc0, "paper", TC_PAPER)
    assert tc[0] > tc[1] > 0.99 * TC_PAPER         # the O(dt) bias raises the apparent T_C
    assert abs(tc0 / TC_PAPER - 1.0) < 0.03
