"""Synthetic workload recipes (BASELINE.json configs[0..4]); see the package docstring.

Site order everywhere: window-local l = (i*nz + k)*ny + j  (x slowest, y fastest), so every
per-site array below has shape [nx, nz, ny] when viewed in 3-D.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field
from typing import Optional, Sequence, Tuple

import numpy as np

GAMMA_E = 1.76085963023e11   # rad s^-1 T^-1
MU_B = 9.2740100783e-24      # J/T
K_B = 1.380649e-23           # J/K
SC, L10 = 0, 1


@dataclass
class Workload:
    name: str
    lattice: int
    nx: int
    ny: int
    nz: int
    pbc: Tuple[int, int, int]
    mu_s: float
    lam: float
    gamma: float
    dt: float
    J: Tuple[float, float, float]
    spacing_nm: Tuple[float, float, float]      # lattice spacing along x, y, z
    track_nx: int
    x0: int
    grain_map: np.ndarray                       # [track_nx, ny] int32, -1 = vacant column
    grain_ku: np.ndarray                        # [G] float32, J per atom
    grain_axis: np.ndarray                      # [G, 3] float32 unit vectors
    macro: Tuple[int, int, int]
    seed: int
    T: np.ndarray                               # [N] float32, K
    Bx: np.ndarray
    By: np.ndarray
    Bz: np.ndarray                              # [N] float32, Tesla
    sx: np.ndarray
    sy: np.ndarray
    sz: np.ndarray                              # [N] float32, 0 on vacant sites
    steps: int = 1000                           # Heun steps the config asks for
    shift_every: int = 0                        # Heun steps between window shifts (0 = never)
    bit_steps: int = 0                          # Heun steps per written bit (0 = static field)
    bit_seed: int = 3
    notes: str = ""

    @property
    def n_sites(self) -> int:
        return self.nx * self.ny * self.nz

    @property
    def n_grains(self) -> int:
        return int(self.grain_ku.shape[0])

    def magnetic_mask(self) -> np.ndarray:
        """[nx, nz, ny] bool: True where the site is magnetic at the current x0."""
        col = self.grain_map[self.x0:self.x0 + self.nx, :] >= 0          # [nx, ny]
        return np.broadcast_to(col[:, None, :], (self.nx, self.nz, self.ny)).copy()


# ----------------------------------------------------------------------------------------------
# Grains: 2-D columnar Voronoi cells from seeds on a jittered hexagonal lattice of
# the given pitch; a column is vacant when it lies within boundary_nm/2 of the bisector of its two
# nearest seeds (=> boundary_nm wide non-magnetic boundaries).  k_u ~ Normal(ku_mean, ku_rel_sigma),
# easy axis polar tilt |Normal(0, tilt_deg)|, azimuth uniform.
# ----------------------------------------------------------------------------------------------
def voronoi_grain_map(track_nx: int, ny: int, ax_nm: float, ay_nm: float, pitch_nm: float = 8.0,
                      boundary_nm: float = 1.0, jitter: float = 0.25, seed: int = 2,
                      ku_mean: float = 9.1e-23, ku_rel_sigma: float = 0.05, tilt_deg: float = 3.0):
    rng = np.random.default_rng(seed)
    Lx, Ly = track_nx * ax_nm, ny * ay_nm
    dy = pitch_nm * math.sqrt(3.0) / 2.0
    pts = []
    r = 0
    y = -pitch_nm
    while y < Ly + pitch_nm:
        x = -pitch_nm + (0.5 * pitch_nm if (r & 1) else 0.0)
        while x < Lx + pitch_nm:
            pts.append((x, y))
            x += pitch_nm
        y += dy
        r += 1
    pts = np.asarray(pts, dtype=np.float64)
    pts += rng.uniform(-jitter * pitch_nm, jitter * pitch_nm, size=pts.shape)
    cx = (np.arange(track_nx) + 0.5) * ax_nm
    cy = (np.arange(ny) + 0.5) * ay_nm
    P = np.stack(np.meshgrid(cx, cy, indexing="ij"), axis=-1).reshape(-1, 2)
    from scipy.spatial import cKDTree
    d, idx = cKDTree(pts).query(P, k=2)
    a, b = pts[idx[:, 0]], pts[idx[:, 1]]
    dist_bisector = (d[:, 1] ** 2 - d[:, 0] ** 2) / (2.0 * np.linalg.norm(a - b, axis=1))
    owner = idx[:, 0].copy()
    owner[dist_bisector < 0.5 * boundary_nm] = -1
    used = np.unique(owner[owner >= 0])
    remap = -np.ones(len(pts), dtype=np.int64)
    remap[used] = np.arange(len(used))
    gm = np.where(owner >= 0, remap[np.maximum(owner, 0)], -1).astype(np.int32).reshape(track_nx, ny)
    G = max(1, len(used))
    ku = (ku_mean * (1.0 + ku_rel_sigma * rng.standard_normal(G))).astype(np.float32)
    polar = np.abs(rng.normal(0.0, math.radians(tilt_deg), G))
    azim = rng.uniform(0.0, 2.0 * math.pi, G)
    axis = np.stack([np.sin(polar) * np.cos(azim), np.sin(polar) * np.sin(azim), np.cos(polar)], axis=1)
    axis = _unit_f32(axis)
    return gm, ku, axis


def _unit_f32(v: np.ndarray) -> np.ndarray:
    """Round to fp32 and renormalise in fp32 a couple of times so |v| = 1 within 1 ulp."""
    v = np.asarray(v, dtype=np.float64)
    v = v / np.linalg.norm(v, axis=-1, keepdims=True)
    return v.astype(np.float32)


def laser_temperature(nx: int, ny: int, nz: int, ax_nm: float, ay_nm: float, fwhm_nm: float = 60.0,
                      t_ambient: float = 300.0, t_peak: float = 800.0,
                      centre: Optional[Tuple[float, float]] = None) -> np.ndarray:
    """Q11: T = T_amb + (T_peak - T_amb) exp(-4 ln2 r^2 / FWHM^2), r in-plane from the window centre."""
    x = (np.arange(nx) + 0.5) * ax_nm
    y = (np.arange(ny) + 0.5) * ay_nm
    cx, cy = centre if centre is not None else (0.5 * nx * ax_nm, 0.5 * ny * ay_nm)
    r2 = (x[:, None] - cx) ** 2 + (y[None, :] - cy) ** 2
    T2 = t_ambient + (t_peak - t_ambient) * np.exp(-4.0 * math.log(2.0) * r2 / fwhm_nm ** 2)
    return np.broadcast_to(T2[:, None, :], (nx, nz, ny)).astype(np.float32).reshape(-1).copy()


def tilted_spins(n: int, tilt_deg: float, seed: int) -> Tuple[np.ndarray, np.ndarray, np.ndarray]:
    """Q12: polar tilt exactly tilt_deg from +z, azimuth uniform (seeded numpy PCG64), fp32."""
    rng = np.random.default_rng(seed)
    phi = rng.uniform(0.0, 2.0 * math.pi, n)
    th = math.radians(tilt_deg)
    v = np.stack([math.sin(th) * np.cos(phi), math.sin(th) * np.sin(phi), np.full(n, math.cos(th))], axis=1)
    v = _unit_f32(v)
    return v[:, 0].copy(), v[:, 1].copy(), v[:, 2].copy()


def _film(name, lattice, nx, ny, nz, spacing, J, lam, dt, extra_track, macro, pitch_nm, boundary_nm,
          grain_seed, seed, uniform_T=None, spot=False, fwhm_nm=60.0, bz=0.0, steps=1000, shift_every=0,
          bit_steps=0, notes="") -> Workload:
    track_nx = nx + extra_track
    gm, ku, axis = voronoi_grain_map(track_nx, ny, spacing[0], spacing[1], pitch_nm=pitch_nm,
                                     boundary_nm=boundary_nm, seed=grain_seed)
    N = nx * ny * nz
    if spot:
        T = laser_temperature(nx, ny, nz, spacing[0], spacing[1], fwhm_nm=fwhm_nm)
    else:
        T = np.full(N, 300.0 if uniform_T is None else uniform_T, dtype=np.float32)
    mag = np.broadcast_to((gm[:nx, :] >= 0)[:, None, :], (nx, nz, ny)).reshape(-1)
    z = np.zeros(N, dtype=np.float32)
    return Workload(name=name, lattice=lattice, nx=nx, ny=ny, nz=nz, pbc=(0, 0, 0), mu_s=3.23 * MU_B,
                    lam=lam, gamma=GAMMA_E, dt=dt, J=J, spacing_nm=spacing, track_nx=track_nx, x0=0,
                    grain_map=gm, grain_ku=ku, grain_axis=axis, macro=macro, seed=seed, T=T,
                    Bx=z.copy(), By=z.copy(), Bz=np.full(N, bz, dtype=np.float32),
                    sx=z.copy(), sy=z.copy(), sz=mag.astype(np.float32), steps=steps,
                    shift_every=shift_every, bit_steps=bit_steps, notes=notes)


J_SC = (6.71e-21, 0.0, 0.0)
J_L10 = (5.0e-21, 2.0e-21, 0.8e-21)
A_SC = (0.3, 0.3, 0.3)
A_L10 = (0.2725, 0.2725, 0.371)


def make_config(i: int, uniform_T: Optional[float] = None) -> Workload:
    """BASELINE.json configs[i], i = 0..4, at full size."""
    if i == 0:
        n = 16
        N = n ** 3
        sx, sy, sz = tilted_spins(N, 5.0, seed=12)
        z = np.zeros(N, dtype=np.float32)
        return Workload(name="cfg0_sc16_pbc", lattice=SC, nx=n, ny=n, nz=n, pbc=(1, 1, 1),
                        mu_s=3.23 * MU_B, lam=0.1, gamma=GAMMA_E, dt=1e-16, J=J_SC, spacing_nm=A_SC,
                        track_nx=n, x0=0, grain_map=np.zeros((n, n), dtype=np.int32),
                        grain_ku=np.array([9.1e-23], dtype=np.float32),
                        grain_axis=np.array([[0.0, 0.0, 1.0]], dtype=np.float32), macro=(7, 7, 7), seed=1,
                        T=np.full(N, 300.0 if uniform_T is None else uniform_T, dtype=np.float32),
                        Bx=z.copy(), By=z.copy(), Bz=z.copy(), sx=sx, sy=sy, sz=sz, steps=1000)
    if i == 1:
        return _film("cfg1_sc_film_192x192x27", SC, 192, 192, 27, A_SC, J_SC, lam=1.0, dt=1e-15,
                     extra_track=0, macro=(7, 7, 7), pitch_nm=8.0, boundary_nm=1.0, grain_seed=2, seed=1,
                     uniform_T=uniform_T, steps=20000,
                     notes="uniform T swept 300..900 K in 50 K steps, 2e4 Heun steps per temperature")
    if i == 2:
        return _film("cfg2_l10_220x220x22", L10, 220, 220, 22, A_L10, J_L10, lam=0.1, dt=1e-15,
                     extra_track=0, macro=(7, 7, 5), pitch_nm=8.0, boundary_nm=1.0, grain_seed=2, seed=1,
                     spot=True, bz=-0.8, steps=10000)
    if i == 3:
        return _film("cfg3_sc_hamr_400x200x27", SC, 400, 200, 27, A_SC, J_SC, lam=0.1, dt=1e-15,
                     extra_track=80, macro=(7, 7, 7), pitch_nm=8.0, boundary_nm=1.0, grain_seed=2, seed=1,
                     spot=True, bz=0.8, steps=100000, shift_every=5000, bit_steps=100000)
    if i == 4:
        return _film("cfg4_l10_hamr_881x220x27", L10, 881, 220, 27, A_L10, J_L10, lam=0.1, dt=1e-15,
                     extra_track=80, macro=(7, 7, 5), pitch_nm=8.0, boundary_nm=1.0, grain_seed=2, seed=1,
                     spot=True, bz=0.8, steps=100000, shift_every=5000, bit_steps=100000)
    raise ValueError("config index must be 0..4")


def small_film(lattice: int, nx: int, ny: int, nz: int, extra_track: int = 0, pitch_nm: float = 3.0,
               boundary_nm: float = 0.6, lam: float = 0.1, dt: float = 1e-15, spot: bool = True,
               uniform_T: Optional[float] = None, bz: float = 0.8, grain_seed: int = 2, seed: int = 1,
               macro: Optional[Sequence[int]] = None, fwhm_nm: float = 6.0, tilt_deg: float = 0.0) -> Workload:
    """A shrunken film with the same structure as cfgs 1-4 (several grains, vacant boundaries,
    Gaussian spot, head field) that the oracle finishes in seconds: the parity-test work-horse."""
    spacing = A_SC if lattice == SC else A_L10
    J = J_SC if lattice == SC else J_L10
    if macro is None:
        macro = (3, 3, 3) if lattice == SC else (3, 3, 2)
    w = _film(f"small_{'sc' if lattice == SC else 'l10'}_{nx}x{ny}x{nz}", lattice, nx, ny, nz, spacing, J,
              lam=lam, dt=dt, extra_track=extra_track, macro=tuple(macro), pitch_nm=pitch_nm,
              boundary_nm=boundary_nm, grain_seed=grain_seed, seed=seed, uniform_T=uniform_T, spot=spot,
              fwhm_nm=fwhm_nm, bz=bz)
    if tilt_deg > 0.0:
        sx, sy, sz = tilted_spins(w.n_sites, tilt_deg, seed=seed + 100)
        mag = w.magnetic_mask().reshape(-1)
        w.sx, w.sy, w.sz = (sx * mag).astype(np.float32), (sy * mag).astype(np.float32), (sz * mag).astype(np.float32)
    return w


def shell_ell_table(w: "Workload"):
    """The built-in neighbour shells of `w` written out as a general ELL table (window-local site indices, -1 = no
    neighbour; exchange energy per pair in Joule): SC 6 nearest neighbours (J[0]); L1_0 4 in-plane nn (J[0]), 2
    out-of-plane (J[1]), 4 in-plane diagonals (J[2]).  Open boundaries; a bond exists only between magnetic sites of the
    SAME grain.  Pure indexing -- this is the data an external ELL user would hand to asd_create_lattice."""
    nx, ny, nz = w.nx, w.ny, w.nz
    if w.lattice == SC:
        offs = [(1, 0, 0, 0), (-1, 0, 0, 0), (0, 1, 0, 0), (0, -1, 0, 0), (0, 0, 1, 0), (0, 0, -1, 0)]
    else:
        offs = [(1, 0, 0, 0), (-1, 0, 0, 0), (0, 1, 0, 0), (0, -1, 0, 0), (0, 0, 1, 1), (0, 0, -1, 1),
                (1, 1, 0, 2), (1, -1, 0, 2), (-1, 1, 0, 2), (-1, -1, 0, 2)]
    gm = np.asarray(w.grain_map)[w.x0:w.x0 + nx]                         # [nx, ny]
    g3 = np.broadcast_to(gm[:, None, :], (nx, nz, ny))                   # site order (i, k, j)
    i, k, j = np.meshgrid(np.arange(nx), np.arange(nz), np.arange(ny), indexing="ij")
    idx = np.full((nx * ny * nz, len(offs)), -1, dtype=np.int32)
    J = np.zeros((nx * ny * nz, len(offs)), dtype=np.float32)
    for s, (dx, dy, dz, shell) in enumerate(offs):
        i2, j2, k2 = i + dx, j + dy, k + dz
        ok = (i2 >= 0) & (i2 < nx) & (j2 >= 0) & (j2 < ny) & (k2 >= 0) & (k2 < nz)
        i2c, j2c, k2c = np.clip(i2, 0, nx - 1), np.clip(j2, 0, ny - 1), np.clip(k2, 0, nz - 1)
        gn = gm[i2c, j2c]
        ok &= (g3 >= 0) & (gn == g3)
        n = (i2c * nz + k2c) * ny + j2c
        idx[:, s] = np.where(ok, n, -1).reshape(-1)
        J[:, s] = np.where(ok, w.J[shell], 0.0).reshape(-1)
    return idx, J


# ----------------------------------------------------------------------------------------------
# Drive schedule: integer planes per shift from a travel accumulator, a seeded
# NRZ bit pattern, and the head-field scale s(t) ramped linearly over one bit period.
# ----------------------------------------------------------------------------------------------
def planes_for_shift(q: int, ax_nm: float, step_nm: float = 1.0) -> int:
    """Planes to shift at the q-th shift (q = 1, 2, ...): floor(q*step/ax) - floor((q-1)*step/ax)."""
    eps = 1e-9
    return int(math.floor(q * step_nm / ax_nm + eps)) - int(math.floor((q - 1) * step_nm / ax_nm + eps))


def nrz_bits(n_bits: int, seed: int = 3) -> np.ndarray:
    """Seeded NRZ polarity pattern (+1/-1)."""
    return np.where(np.random.default_rng(seed).integers(0, 2, n_bits) > 0, 1.0, -1.0)


def field_scale_at(step: int, bits: np.ndarray, bit_steps: int, ramp_steps: Optional[int] = None) -> float:
    """s(t) in [-1, 1]: linear ramp from the previous bit's polarity to the current one."""
    if bit_steps <= 0:
        return 1.0
    ramp_steps = bit_steps if ramp_steps is None else ramp_steps
    b = min(step // bit_steps, len(bits) - 1)
    cur = float(bits[b])
    prev = float(bits[b - 1]) if b > 0 else cur
    f = min(1.0, (step - b * bit_steps) / float(ramp_steps))
    return prev + (cur - prev) * f


@dataclass
class ShiftSchedule:
    """Iterates (n_heun_steps, field_scale) batches and the p of the shift closing each period."""
    w: Workload
    batch: int = 100
    n_bits: int = 64

    def __post_init__(self):
        self.bits = nrz_bits(self.n_bits, self.w.bit_seed)

    def period(self, q: int):
        """Batches of the q-th shift period (q = 1, 2, ...) and the planes to shift at its end."""
        se = self.w.shift_every
        start = (q - 1) * se
        batches = []
        s = start
        while s < start + se:
            n = min(self.batch, start + se - s)
            batches.append((n, field_scale_at(s, self.bits, self.w.bit_steps)))
            s += n
        return batches, planes_for_shift(q, self.w.spacing_nm[0])
