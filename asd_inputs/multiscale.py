"""Inputs for the multiscale window (Fig. 1): a central
atomistic mesh with a micromagnetic LLG mesh either side, all moving along the granular track together.

Input generation only -- no method arithmetic.  The micromagnetic cells ARE the track macrocells (DESIGN.md sec. 14,
reading M1); their material parameters are the continuum limits of the atomistic ones (Eq. (9)-(10)):

    M_S^0 = mu_s / V_atom                         one moment per lattice cell of the (Fe sub)lattice
    K_0,g = k_u,g / V_atom                        per grain
    A_0,a = sum_j J_j r_j,a^2 / (4 V_atom)        per axis a; simple cubic: J / 2a along every axis (Eq. (9)); with one J on
                                                  all ten L1_0 neighbours: 3J / 2a in the plane (Eq. (10))
    T_C,g ~ Normal(T_C, 5 %)                      per grain ("a normal distribution with standard deviation about T_C ...
                                                  of 0.05 x T_C")

A cell column (cx, cy) of the track belongs to the grain that owns most of its magnetic columns, and is empty when fewer
than half of its columns are magnetic.
"""
from __future__ import annotations

import math
from dataclasses import dataclass
from typing import List, Optional, Sequence, Tuple

import numpy as np

from . import workloads as wl


@dataclass
class Multiscale:
    w: wl.Workload                 # the atomistic mesh (w.x0 = cells of the trailing mesh * mx)
    mcx: Tuple[int, int]           # cells along x of the trailing / leading micromagnetic mesh
    every: int                     # Heun steps per RK4 step (dt_mm = every * dt; 20 fs against 10 / 5 fs)
    Ms0: float                     # A/m
    A0: Tuple[float, float, float] # J/m along x, y, z
    K0: np.ndarray                 # [G] J/m^3
    Tc: np.ndarray                 # [G] K
    cell_grain: np.ndarray         # [ncx, ncy] int32, -1 = empty cell column
    T_mesh: List[np.ndarray]       # [2] per cell [mcx, ncy, ncz], K
    B_mesh: List[np.ndarray]       # [2] per cell [mcx, ncy, ncz, 3], Tesla
    spacing_m: Tuple[float, float, float]

    def track_cells(self) -> Tuple[int, int, int]:
        m = self.w.macro
        return (-(-self.w.track_nx // m[0]), -(-self.w.ny // m[1]), -(-self.w.nz // m[2]))


def cell_grain_map(grain_map: np.ndarray, macro: Sequence[int]) -> np.ndarray:
    """[ncx, ncy] majority grain of every track cell column; -1 when fewer than half of its columns are magnetic."""
    track_nx, ny = grain_map.shape
    mx, my = int(macro[0]), int(macro[1])
    ncx, ncy = -(-track_nx // mx), -(-ny // my)
    out = -np.ones((ncx, ncy), dtype=np.int32)
    for cx in range(ncx):
        for cy in range(ncy):
            blk = grain_map[cx * mx:(cx + 1) * mx, cy * my:(cy + 1) * my].reshape(-1)
            mag = blk[blk >= 0]
            if 2 * mag.size >= blk.size and mag.size > 0:
                ids, cnt = np.unique(mag, return_counts=True)
                out[cx, cy] = ids[np.argmax(cnt)]
    return out


def continuum_parameters(lattice: int, J: Sequence[float], spacing_nm: Sequence[float], mu_s: float, ku: np.ndarray):
    """(M_S^0, (A_x, A_y, A_z), K_0[G]) of the lattice's long-wavelength limit."""
    a = [s * 1e-9 for s in spacing_nm]
    V = a[0] * a[1] * a[2]
    if lattice == wl.SC:
        offs = [((1, 0, 0), 0), ((-1, 0, 0), 0), ((0, 1, 0), 0), ((0, -1, 0), 0), ((0, 0, 1), 0), ((0, 0, -1), 0)]
    else:
        offs = [((1, 0, 0), 0), ((-1, 0, 0), 0), ((0, 1, 0), 0), ((0, -1, 0), 0), ((0, 0, 1), 1), ((0, 0, -1), 1),
                ((1, 1, 0), 2), ((1, -1, 0), 2), ((-1, 1, 0), 2), ((-1, -1, 0), 2)]
    A = [sum(J[sh] * (d[ax] * a[ax]) ** 2 for d, sh in offs) / (4.0 * V) for ax in range(3)]
    return mu_s / V, tuple(A), np.asarray(ku, dtype=np.float64) / V


def multiscale_film(lattice: int = wl.SC, atom_cells: int = 48, mesh_cells: Tuple[int, int] = (48, 48),
                    width_nm: float = 60.0, nz: int = 27, extra_cells: int = 12, every: int = 20,
                    macro: Optional[Sequence[int]] = None, pitch_nm: float = 8.0, boundary_nm: float = 1.0,
                    fwhm_nm: float = 60.0, t_peak: float = 800.0, t_ambient: float = 300.0, bz: float = 0.8,
                    tc_mean: Optional[float] = None, tc_rel_sigma: float = 0.05, lam: float = 0.1, dt: float = 1e-15,
                    grain_seed: int = 2, seed: int = 1, tilt_deg: float = 0.0) -> Multiscale:
    """[trailing mesh | atomistic mesh | leading mesh] over a granular track.  Defaults follow the paper's split of a
    window into three equal parts ("a 100 nm long atomistic simulation region and two 100 nm long micromagnetic
    simulation regions") on the cfg3 lattice; the parity tests shrink every length."""
    spacing = wl.A_SC if lattice == wl.SC else wl.A_L10
    J = wl.J_SC if lattice == wl.SC else wl.J_L10
    if macro is None:
        macro = (7, 7, 7) if lattice == wl.SC else (7, 7, 5)
    mx, my, mz = (int(v) for v in macro)
    nx = atom_cells * mx
    ny = int(round(width_nm / spacing[1] / 4.0)) * 4
    x0 = mesh_cells[0] * mx
    track_nx = x0 + nx + (mesh_cells[1] + extra_cells) * mx
    gm, ku, axis = wl.voronoi_grain_map(track_nx, ny, spacing[0], spacing[1], pitch_nm=pitch_nm,
                                        boundary_nm=boundary_nm, seed=grain_seed)
    G = ku.shape[0]
    mu_s = 3.23 * wl.MU_B
    Ms0, A0, K0 = continuum_parameters(lattice, J, spacing, mu_s, ku)
    if tc_mean is None:
        # Eq. (8) with the paper's mean-field correction factors: T_C = eps z J / 3 k_B for a single J;
        # per-shell J: z J -> sum_j J_j
        eps = 0.72 if lattice == wl.SC else 0.78
        zJ = 6 * J[0] if lattice == wl.SC else 4 * J[0] + 2 * J[1] + 4 * J[2]
        tc_mean = eps * zJ / (3.0 * wl.K_B)
    rng = np.random.default_rng(grain_seed + 1000)
    Tc = tc_mean * (1.0 + tc_rel_sigma * rng.standard_normal(G))
    # profiles centred on the window [trailing mesh | atoms | leading mesh]; the spot sits on the atomistic mesh
    xc_nm = (x0 + 0.5 * nx) * spacing[0]
    yc_nm = 0.5 * ny * spacing[1]

    def temperature(x_nm, y_nm):
        r2 = (x_nm - xc_nm) ** 2 + (y_nm - yc_nm) ** 2
        return t_ambient + (t_peak - t_ambient) * np.exp(-4.0 * math.log(2.0) * r2 / fwhm_nm ** 2)
    xs = (x0 + np.arange(nx) + 0.5) * spacing[0]
    ys = (np.arange(ny) + 0.5) * spacing[1]
    T2 = temperature(xs[:, None], ys[None, :])
    N = nx * ny * nz
    T = np.broadcast_to(T2[:, None, :], (nx, nz, ny)).astype(np.float32).reshape(-1).copy()
    mag = np.broadcast_to((gm[x0:x0 + nx, :] >= 0)[:, None, :], (nx, nz, ny)).reshape(-1)
    z = np.zeros(N, dtype=np.float32)
    w = wl.Workload(name=f"multiscale_{'sc' if lattice == wl.SC else 'l10'}_{mesh_cells[0]}c+{nx}x{ny}x{nz}+{mesh_cells[1]}c",
                    lattice=lattice, nx=nx, ny=ny, nz=nz, pbc=(0, 0, 0), mu_s=mu_s, lam=lam, gamma=wl.GAMMA_E, dt=dt,
                    J=J, spacing_nm=spacing, track_nx=track_nx, x0=x0, grain_map=gm, grain_ku=ku, grain_axis=axis,
                    macro=(mx, my, mz), seed=seed, T=T, Bx=z.copy(), By=z.copy(), Bz=np.full(N, bz, dtype=np.float32),
                    sx=z.copy(), sy=z.copy(), sz=mag.astype(np.float32), steps=0, shift_every=0, bit_steps=0,
                    notes="multiscale window: micromagnetic | atomistic | micromagnetic (Fig. 1)")
    if tilt_deg > 0.0:
        sx, sy, sz = wl.tilted_spins(N, tilt_deg, seed=seed + 100)
        w.sx, w.sy, w.sz = (sx * mag).astype(np.float32), (sy * mag).astype(np.float32), (sz * mag).astype(np.float32)
    ncy, ncz = -(-ny // my), -(-nz // mz)
    cyc = (np.arange(ncy) + 0.5) * my * spacing[1]
    T_mesh, B_mesh = [], []
    for side, c0 in ((0, 0), (1, (x0 + nx) // mx)):
        cxc = (c0 + np.arange(mesh_cells[side]) + 0.5) * mx * spacing[0]
        Tm = temperature(cxc[:, None], cyc[None, :])
        T_mesh.append(np.broadcast_to(Tm[:, :, None], (mesh_cells[side], ncy, ncz)).copy())
        Bm = np.zeros((mesh_cells[side], ncy, ncz, 3))
        Bm[..., 2] = bz
        B_mesh.append(Bm)
    return Multiscale(w=w, mcx=(int(mesh_cells[0]), int(mesh_cells[1])), every=every, Ms0=Ms0, A0=A0, K0=K0, Tc=Tc,
                      cell_grain=cell_grain_map(gm, (mx, my, mz)), T_mesh=T_mesh, B_mesh=B_mesh,
                      spacing_m=tuple(s * 1e-9 for s in spacing))


def apply_multiscale(sim, ms: Multiscale):
    """Switches the micromagnetic meshes on in `sim` (the oracle or the CUDA context: same method names) and hands them
    their temperature and field profiles."""
    st = sim.mm_enable(ms.mcx, ms.every, ms.Ms0, ms.A0, ms.K0, ms.Tc, ms.cell_grain, ms.spacing_m)
    if st not in (None, 0):
        raise ValueError(f"mm_enable rejected the description (status {st})")
    for side in (0, 1):
        B = ms.B_mesh[side]
        sim.mm_set_fields(side, ms.T_mesh[side], B[..., 0], B[..., 1], B[..., 2])


# ----------------------------------------------------------------------------------------------------------------------
# Writing a bit sequence with a multiscale window (the paper's Fig. 3 experiment in miniature): the window
# [mesh | atoms | mesh] moves along the track one cell at a time while the head polarity follows a seeded bit pattern.
# ----------------------------------------------------------------------------------------------------------------------
@dataclass
class MultiscaleWrite:
    ms: Multiscale
    bits: np.ndarray               # NRZ polarity (+1 / -1) per bit
    bit_cells: int                 # cells per written bit
    steps_per_cell: int            # Heun steps between shifts of one cell (same velocity as 5000 steps per nm)
    batch: int
    spot_plane: float              # global plane under the spot centre when the pass starts
    write_offset: float            # planes from the spot centre back to where the grains freeze (edge of T > T_C)
    reader_sigma: Tuple[float, float]
    track_y: float

    @property
    def bit_origin(self) -> float:
        """Global plane where bit 0 starts: where the freezing point stands when the pass starts."""
        return self.spot_plane - self.write_offset

    def bit_at(self, gx: float) -> float:
        """Polarity the head writes while the spot centre is over global plane gx."""
        bp = self.bit_cells * self.ms.w.macro[0]
        b = min(max(int((gx - self.write_offset - self.bit_origin) // bp), 0), len(self.bits) - 1)
        return float(self.bits[b])

    def cells_per_pass(self) -> int:
        m = self.ms
        return m.track_cells()[0] - (m.w.x0 + m.w.nx) // m.w.macro[0] - m.mcx[1]

    def swept_bits(self, cells: Optional[int] = None) -> np.ndarray:
        cells = self.cells_per_pass() if cells is None else cells
        bp = self.bit_cells * self.ms.w.macro[0]
        b = np.arange(len(self.bits))
        return b[(b + 1) * bp <= cells * self.ms.w.macro[0]]

    def bit_centres(self) -> np.ndarray:
        return self.bit_origin + (np.arange(len(self.bits)) + 0.5) * self.bit_cells * self.ms.w.macro[0]


def multiscale_write(lattice: int = wl.SC, atom_cells: int = 57, mesh_cells: Tuple[int, int] = (24, 24), n_bits: int = 8,
                     bit_cells: int = 10, width_nm: float = 60.0, nz: int = 27, every: int = 20, fwhm_nm: float = 60.0,
                     steps_per_nm: int = 5000, batch: int = 100, bit_seed: int = 3, meshes: bool = True,
                     **kw) -> MultiscaleWrite:
    """meshes = False: the same atomistic mesh, track, schedule and bit pattern without the micromagnetic meshes (the
    fully atomistic window the paper compares with); the recipe still carries the mesh description, unused."""
    macro = kw.pop("macro", None) or ((7, 7, 7) if lattice == wl.SC else (7, 7, 5))
    total_bits_cells = n_bits * bit_cells
    ms = multiscale_film(lattice, atom_cells=atom_cells, mesh_cells=mesh_cells, width_nm=width_nm, nz=nz,
                         extra_cells=total_bits_cells, every=every, macro=macro, fwhm_nm=fwhm_nm, **kw)
    sp = ms.w.spacing_nm
    # the grains freeze where the trailing flank of the spot crosses T_C: T = T_amb + dT exp(-4 ln2 r^2 / FWHM^2) = T_C,
    # with the recipe's mean T_C (Eq. (8): 700 K for the SC exchange, 512 K for the L1_0 shells) and its 300 / 800 K spot
    t_amb, t_peak = float(kw.get("t_ambient", 300.0)), float(kw.get("t_peak", 800.0))
    t_c = min(float(np.mean(ms.Tc)), t_peak - 1.0)
    r_hot_nm = fwhm_nm * math.sqrt(math.log((t_peak - t_amb) / (t_c - t_amb)) / (4.0 * math.log(2.0)))
    return MultiscaleWrite(ms=ms, bits=wl.nrz_bits(n_bits, bit_seed), bit_cells=bit_cells,
                           steps_per_cell=int(round(steps_per_nm * macro[0] * sp[0])), batch=batch,
                           spot_plane=ms.w.x0 + 0.5 * ms.w.nx, write_offset=r_hot_nm / sp[0],
                           reader_sigma=(0.25 * bit_cells * macro[0], 0.25 * width_nm / sp[1]),
                           track_y=0.5 * ms.w.ny)


def drive_multiscale_write(sim, mw: MultiscaleWrite, cells: Optional[int] = None, with_meshes: bool = True) -> int:
    """One pass: per shift period the head polarity of the bit under the freezing point, steps_per_cell Heun steps, a
    shift by one cell; then asd_track_end_pass.  `sim`: the oracle or the CUDA context.  Returns the Heun steps taken."""
    if with_meshes:
        apply_multiscale(sim, mw.ms)
    cells = mw.cells_per_pass() if cells is None else cells
    mx = mw.ms.w.macro[0]
    gx, steps = mw.spot_plane, 0
    for _ in range(cells):
        sim.set_field_scale(mw.bit_at(gx))
        left = mw.steps_per_cell
        while left > 0:
            n = min(mw.batch, left)
            sim.step_heun(n)
            left -= n
            steps += n
        sim.shift_window(mx)
        gx += mx
    sim.track_end_pass()
    return steps
