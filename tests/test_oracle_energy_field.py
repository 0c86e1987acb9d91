"""Pin P5: the oracle's field is minus the gradient of an energy computed here by brute force from the
geometric definition of the neighbour shells (pair list built from DISTANCES, not from offset tables):
  E = - sum_{bonds <ij>} J_ij S_i.S_j - sum_i k_u,g (S_i.e_g)^2 - mu_s sum_i s B_i.S_i ,  B_i = -(1/mu_s) dE/dS_i.
SC: |r_ij| = a -> J (6 neighbours).  L1_0 Fe sublattice: in-plane nn at s -> J1, out-of-plane at c -> J2,
in-plane nnn at s*sqrt2 -> J3 ("4 nearest + 6 next nearest").  Bonds need both ends magnetic and in
the same grain ("exchange-decoupled").
"""
import itertools
import math

import numpy as np
import pytest

from oracle import asd_oracle as orc

MUS = 3.23 * orc.MU_B


def _brute_energy(S, lattice, dims, pbc, spacing, J, gm, ku, axis, B, scale):
    nx, ny, nz = dims
    coords = [(i, k, j) for i in range(nx) for k in range(nz) for j in range(ny)]   # l = (i*nz+k)*ny+j
    L = (nx * spacing[0], ny * spacing[1], nz * spacing[2])
    E = 0.0
    for a, (i, k, j) in enumerate(coords):
        ga = gm[i, j]
        if ga < 0:
            continue
        d = float(S[a] @ axis[ga])
        E -= ku[ga] * d * d
        E -= MUS * scale * float(B[a] @ S[a])
    for a, b in itertools.combinations(range(len(coords)), 2):
        (i, k, j), (i2, k2, j2) = coords[a], coords[b]
        if gm[i, j] < 0 or gm[i2, j2] < 0 or gm[i, j] != gm[i2, j2]:
            continue
        # all periodic images that realise a bond (a pair can be bonded through more than one image when n = 3)
        for sx, sy, sz in itertools.product((-1, 0, 1), repeat=3):
            if (sx and not pbc[0]) or (sy and not pbc[1]) or (sz and not pbc[2]):
                continue
            dx = (i2 - i) * spacing[0] + sx * L[0]
            dy = (j2 - j) * spacing[1] + sy * L[1]
            dz = (k2 - k) * spacing[2] + sz * L[2]
            r = math.sqrt(dx * dx + dy * dy + dz * dz)
            Jij = 0.0
            if lattice == 0:
                if abs(r - spacing[0]) < 1e-6:
                    Jij = J[0]
            else:
                s, c = spacing[0], spacing[2]
                inplane = abs(dz) < 1e-9
                if inplane and abs(r - s) < 1e-6:
                    Jij = J[0]
                elif abs(dx) < 1e-9 and abs(dy) < 1e-9 and abs(r - c) < 1e-6:
                    Jij = J[1]
                elif inplane and abs(r - s * math.sqrt(2)) < 1e-6:
                    Jij = J[2]
            if Jij:
                E -= Jij * float(S[a] @ S[b])
    return E


@pytest.mark.parametrize("lattice,dims,pbc", [
    (0, (3, 3, 3), (1, 1, 1)), (0, (4, 3, 2), (0, 0, 0)), (0, (4, 4, 2), (1, 0, 0)),
    (1, (3, 3, 3), (1, 1, 1)), (1, (4, 4, 2), (0, 0, 0)), (1, (3, 4, 3), (0, 1, 1)),
])
def test_p5_energy_and_field_against_brute_force(lattice, dims, pbc):
    rng = np.random.default_rng(7 + lattice)
    nx, ny, nz = dims
    N = nx * ny * nz
    spacing = (0.3, 0.3, 0.3) if lattice == 0 else (0.2725, 0.2725, 0.371)
    J = (6.71e-21, 0, 0) if lattice == 0 else (5.0e-21, 2.0e-21, 0.8e-21)
    gm = rng.integers(-1, 3, size=(nx, ny)).astype(np.int32)          # grains 0..2, some vacant, adjacent grains
    gm[0, 0] = 0
    ku = (9.1e-23 * (1 + 0.3 * rng.standard_normal(3)))
    axis = rng.standard_normal((3, 3))
    axis /= np.linalg.norm(axis, axis=1, keepdims=True)
    S = rng.standard_normal((N, 3))
    S /= np.linalg.norm(S, axis=1, keepdims=True)
    S32 = S.astype(np.float32)
    B32 = rng.standard_normal((N, 3)).astype(np.float32)
    scale = 0.625
    spec = orc.LatticeSpec(lattice=lattice, nx=nx, ny=ny, nz=nz, pbc=pbc, mu_s=MUS, J=J, grain_map=gm,
                           grain_ku=ku, grain_axis=axis)
    o = orc.Oracle(spec)
    o.set_spins(S32[:, 0], S32[:, 1], S32[:, 2])
    o.set_fields(np.zeros(N), B32[:, 0], B32[:, 1], B32[:, 2])
    o.set_field_scale(scale)
    mag = np.repeat((gm >= 0)[:, None, :], nz, axis=1).reshape(-1)
    Sd = S32.astype(np.float64) * mag[:, None]
    Bd = B32.astype(np.float64)
    args = (lattice, dims, pbc, spacing, J, gm, ku, axis, Bd, scale)
    E0 = _brute_energy(Sd, *args)
    assert abs(o.energy() - E0) <= 1e-12 * abs(E0)
    # field = -(1/mu_s) dE/dS by central differences (E is quadratic in each S_i => exact up to rounding)
    Bo = o.field(with_noise=False)
    h = 1e-3
    for a in rng.choice(np.nonzero(mag)[0], size=min(8, int(mag.sum())), replace=False):
        for c in range(3):
            Sp, Sm = Sd.copy(), Sd.copy()
            Sp[a, c] += h
            Sm[a, c] -= h
            g = -(_brute_energy(Sp, *args) - _brute_energy(Sm, *args)) / (2 * h) / MUS
            assert abs(Bo[c, a] - g) < 1e-7 * max(1.0, abs(g)), (a, c, Bo[c, a], g)
    assert np.all(Bo[:, ~mag] == 0.0)
