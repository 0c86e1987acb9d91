"""Ensemble observables for thermal runs (Q16, Q18): trajectories of the fp32 CUDA path and the fp64 oracle
diverge chaotically after ~1e2 steps, so thermal parity is stated on time averages: M(T) = time average (second half
of each temperature's steps) of the grain-averaged |<S>_grain|, and T_C from the fit m = (1 - T/T_C)^beta on the points
with m > 0.25.  The same estimator runs on both sides; nothing here knows which side it is driving.
"""
from __future__ import annotations

import numpy as np


class Side:
    """Adapter: set_uniform_T(T), step(n), grain_m() -> [n_grains, 3]."""

    def __init__(self, sim, n_sites: int, is_gpu: bool):
        self.sim, self.N, self.is_gpu = sim, n_sites, is_gpu

    def set_uniform_T(self, T: float):
        a = np.full(self.N, T, dtype=np.float32)
        if self.is_gpu:
            self.sim.set_fields_host(T=a)
        else:
            self.sim.set_fields(T=a)

    def step(self, n: int):
        self.sim.step_heun(n)

    def grain_m(self) -> np.ndarray:
        return np.asarray(self.sim.grain_magnetisation())


def sweep(side: Side, temps, n_steps: int, n_samples: int = 20, grain_weights=None) -> np.ndarray:
    """State is carried from one temperature to the next (BASELINE configs[1]).  Returns M(T)."""
    out = []
    for T in temps:
        side.set_uniform_T(float(T))
        side.step(n_steps // 2)
        acc = []
        per = max(1, (n_steps - n_steps // 2) // n_samples)
        for _ in range(n_samples):
            side.step(per)
            g = np.linalg.norm(side.grain_m(), axis=1)
            acc.append(float(np.average(g, weights=grain_weights)))
        out.append(np.mean(acc))
    return np.array(out)


def fit_tc(temps, m, m_min: float = 0.25):
    from scipy.optimize import curve_fit
    temps, m = np.asarray(temps, float), np.asarray(m, float)
    sel = m > m_min
    f = lambda T, Tc, b: np.clip(1.0 - T / Tc, 1e-12, None) ** b
    p, _ = curve_fit(f, temps[sel], m[sel], p0=(temps[sel].max() * 1.1, 0.36), maxfev=20000)
    return float(p[0]), float(p[1])
