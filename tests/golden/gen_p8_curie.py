"""Writes tests/golden/p8_curie_record.json: the oracle's bulk simple-cubic Curie temperature (pin P8).

    python tests/golden/gen_p8_curie.py            (about 5-10 minutes on 8 cores; calls only oracle/)

Method (P8): periodic SC lattice, L = 24, J = 6.71e-21 J, mu_s = 3.23 mu_B, lambda = 1, no anisotropy,
no field; temperature sweep 575 ... 750 K in steps of 25 K with the state carried from one temperature to the next;
m(T) = time average of |<S>| over the second half of each temperature's steps; T_C from the fit m = (1 - T/T_C)^beta
(beta free) on the points with m > 0.25; two time steps (0.5 fs, 0.25 fs) and a linear extrapolation to dt -> 0
(stochastic Heun has an O(dt) bias of the stationary distribution).  Expected: T_C = eps z J / (3 k_B) = 1.44 J / k_B
(Eq. (8): eps_SC = 0.72, z = 6).

The record carries the SHA-256 of oracle/asd_oracle.cpp: tests/test_oracle_curie.py refuses a record made by a different
oracle.
"""
import hashlib
import json
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
from oracle import asd_oracle as orc  # noqa: E402

J = 6.71e-21
MUS = 3.23 * orc.MU_B
L = 24
TEMPS = np.arange(575.0, 751.0, 25.0)
RUNS = ((5e-16, 8000), (2.5e-16, 16000))          # (dt, Heun steps per temperature)


def oracle_sha256() -> str:
    return hashlib.sha256(open(os.path.join(ROOT, "oracle", "asd_oracle.cpp"), "rb").read()).hexdigest()


def mean_m(o, N, T, n_relax, n_avg, n_samples=16):
    z = np.zeros(N)
    o.set_fields(T=np.full(N, T), Bx=z, By=z, Bz=z)
    o.step_heun(n_relax)
    acc = []
    for _ in range(n_samples):
        o.step_heun(max(1, n_avg // n_samples))
        m, _n = o.magnetisation()
        acc.append(np.linalg.norm(m))
    return float(np.mean(acc))


def main():
    from scipy.optimize import curve_fit
    t0 = time.time()
    N = L ** 3
    runs = []
    for dt, nsteps in RUNS:
        spec = orc.LatticeSpec(lattice=0, nx=L, ny=L, nz=L, pbc=(1, 1, 1), lam=1.0, dt=dt, J=(J, 0, 0), mu_s=MUS, seed=1,
                               grain_map=np.zeros((L, L), dtype=np.int32), grain_ku=np.array([0.0]),
                               grain_axis=np.array([[0.0, 0.0, 1.0]]))
        o = orc.Oracle(spec)
        o.set_spins(np.zeros(N), np.zeros(N), np.ones(N))
        m = [mean_m(o, N, float(T), nsteps // 2, nsteps // 2) for T in TEMPS]
        m = np.array(m)
        sel = m > 0.25
        f = lambda T, Tc, b: np.clip(1.0 - T / Tc, 1e-12, None) ** b
        p, _cov = curve_fit(f, TEMPS[sel], m[sel], p0=(720.0, 0.36))
        runs.append({"dt": dt, "steps_per_T": nsteps, "m": [float(x) for x in m], "T_C_fit": float(p[0]), "beta_fit": float(p[1])})
        print("dt", dt, "m(T)", np.round(m, 4), "fit", p, flush=True)
    tc0 = 2.0 * runs[1]["T_C_fit"] - runs[0]["T_C_fit"]
    rec = {"pin": "P8", "what": "bulk SC Heisenberg T_C of the oracle, extrapolated to dt -> 0", "L": L, "J": J,
           "mu_s": MUS, "lambda": 1.0, "temps_K": [float(t) for t in TEMPS], "runs": runs, "T_C_dt0": tc0,
           "T_C_paper": 1.44 * J / orc.K_B, "ratio": tc0 / (1.44 * J / orc.K_B),
           "oracle_sha256": oracle_sha256(), "threads": orc.max_threads(), "wall_s": round(time.time() - t0, 1),
           "written_by": "tests/golden/gen_p8_curie.py"}
    out = os.path.join(ROOT, "tests", "golden", "p8_curie_record.json")
    json.dump(rec, open(out, "w"), indent=1)
    print("wrote", out, "T_C(dt->0) =", tc0, "ratio", rec["ratio"])


if __name__ == "__main__":
    main()
