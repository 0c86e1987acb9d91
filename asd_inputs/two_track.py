"""Second workload (sec. III / Fig. 4): two parallel tracks written one
after the other in an 80 nm wide window, 15 nm between the ~25 nm wide bit rows.

Input generation and call sequencing only -- no method arithmetic.  The same `TwoTrack` drives the oracle and the
CUDA library through `drive_pass`, which issues the identical sequence of library calls to either.

Geometry: the film is `width_nm` wide; the two track centres sit at (width - pitch)/2 and
(width + pitch)/2 with pitch = bit width + separation = 25 + 15 = 40 nm ("the bits are approximately 25 nm wide
as before, with the separation between tracks being 15 nm, for a total simulation window with 80 nm width").  Pass p
centres the laser spot on track p ("achieved by positioning the laser spot in the centre of the bottom track").
The spot FWHM is chosen so that its diameter above T_C is the 25 nm of P:86; for the paper's 710 K (simple cubic):
T = 300 + 500 exp(-4 ln2 r^2 / FWHM^2) > 710 K  <=>  r < 0.2675 FWHM  =>  FWHM = 46.7 nm; for the L1_0 shells of
BASELINE.json (mean-field T_C = 512 K) the same rule gives 22.5 nm.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field
from typing import Callable, List, Optional, Sequence, Tuple

import numpy as np

from . import workloads as wl


@dataclass
class TwoTrack:
    w: wl.Workload                     # lattice, grains, initial spins (+z); w.T = pass 0's temperature profile
    T_pass: List[np.ndarray]           # [2] per-site temperature [K], spot centred on track p
    bits: List[np.ndarray]             # [2] NRZ polarity (+1 / -1) per bit, one pattern per track
    track_y: Tuple[float, float]       # track centres across the film, in sites
    bit_planes: int                    # planes per written bit (20 nm)
    shift_every: int                   # Heun steps between window shifts
    batch: int                         # Heun steps per asd_step_heun call (field scale constant inside a batch)
    reader_sigma: Tuple[float, float]  # Gaussian reader footprint (along, across the track), in sites
    spot_plane: float                  # window plane under the centre of the laser spot
    write_offset: float = 0.0          # planes between the spot centre and the trailing edge of the region above T_C,
                                       # where the grains freeze: the head polarity follows the bit under THAT point

    @property
    def n_periods(self) -> int:
        """Shift periods of one full pass: the window travels from x0 = 0 to the end of the track."""
        planes = self.w.track_nx - self.w.nx
        q, done = 0, 0
        while done + wl.planes_for_shift(q + 1, self.w.spacing_nm[0]) <= planes:
            q += 1
            done += wl.planes_for_shift(q, self.w.spacing_nm[0])
        return q

    def bit_at_plane(self, p: int, gx: float) -> float:
        """Polarity the head writes while the spot centre is over global plane gx."""
        b = min(max(int((gx - self.write_offset) // self.bit_planes), 0), len(self.bits[p]) - 1)
        return float(self.bits[p][b])

    def bit_centres(self) -> np.ndarray:
        """Global plane coordinate of every bit centre."""
        return (np.arange(len(self.bits[0])) + 0.5) * self.bit_planes

    def written_bits(self, periods: Optional[int] = None) -> np.ndarray:
        """Indices of the bits whose whole length the freezing point has swept in a pass of `periods` shift periods."""
        periods = self.n_periods if periods is None else periods
        travel = sum(wl.planes_for_shift(q, self.w.spacing_nm[0]) for q in range(1, periods + 1))
        lo, hi = self.spot_plane - self.write_offset, self.spot_plane - self.write_offset + travel
        b = np.arange(len(self.bits[0]))
        return b[(b * self.bit_planes >= lo) & ((b + 1) * self.bit_planes <= hi)]


def two_track_film(lattice: int = wl.SC, length_nm: float = 120.0, width_nm: float = 80.0, nz: int = 27,
                   n_bits: int = 8, bit_nm: float = 20.0, separation_nm: float = 15.0, bit_width_nm: float = 25.0,
                   pitch_nm: float = 8.0, boundary_nm: float = 1.0, fwhm_nm: Optional[float] = None,
                   t_peak: float = 800.0, bz: float = 0.8, lam: float = 0.1, dt: float = 1e-15,
                   shift_every: int = 5000, batch: int = 100, macro: Optional[Sequence[int]] = None,
                   grain_seed: int = 2, seed: int = 1, bit_seeds: Tuple[int, int] = (3, 4),
                   t_c: Optional[float] = None) -> TwoTrack:
    """The two-track window at any size: defaults are the paper's geometry on the cfg3 / cfg4 lattices; the parity tests
    shrink every length."""
    spacing = wl.A_SC if lattice == wl.SC else wl.A_L10
    J = wl.J_SC if lattice == wl.SC else wl.J_L10
    if macro is None:
        macro = (7, 7, 7) if lattice == wl.SC else (7, 7, 5)
    nx = int(round(length_nm / spacing[0]))
    ny = int(round(width_nm / spacing[1] / 4.0)) * 4
    bit_planes = int(round(bit_nm / spacing[0]))
    track_nx = nx + n_bits * bit_planes
    if t_c is None:
        # the temperature the bits are written at: the paper's 710 K for its simple-cubic exchange; for the L1_0 shells
        # of BASELINE.json the mean-field estimate of Eq. (8), eps (4 J1 + 2 J2 + 4 J3) / 3 k_B = 512 K
        t_c = 710.0 if lattice == wl.SC else 0.78 * (4 * J[0] + 2 * J[1] + 4 * J[2]) / (3.0 * wl.K_B)
    if fwhm_nm is None:
        # spot width such that its diameter above t_c is the bit width: T = 300 + (t_peak - 300) exp(-4 ln2 r^2 / FWHM^2)
        frac = (t_c - 300.0) / (t_peak - 300.0)
        if not 0.0 < frac < 1.0:                 # a spot that never reaches t_c (the cool parity tests): the paper's proportions
            frac = 410.0 / 500.0
        fwhm_nm = bit_width_nm / (2.0 * math.sqrt(math.log(1.0 / frac) / (4.0 * math.log(2.0))))
    gm, ku, axis = wl.voronoi_grain_map(track_nx, ny, spacing[0], spacing[1], pitch_nm=pitch_nm,
                                        boundary_nm=boundary_nm, seed=grain_seed)
    N = nx * ny * nz
    pitch = bit_width_nm + separation_nm
    yc_nm = (0.5 * (width_nm - pitch), 0.5 * (width_nm + pitch))
    xc_nm = 0.5 * nx * spacing[0]
    T_pass = [wl.laser_temperature(nx, ny, nz, spacing[0], spacing[1], fwhm_nm=fwhm_nm, t_peak=t_peak,
                                   centre=(xc_nm, y)) for y in yc_nm]
    mag = np.broadcast_to((gm[:nx, :] >= 0)[:, None, :], (nx, nz, ny)).reshape(-1)
    z = np.zeros(N, dtype=np.float32)
    w = wl.Workload(name=f"two_track_{'sc' if lattice == wl.SC else 'l10'}_{nx}x{ny}x{nz}", lattice=lattice, nx=nx,
                    ny=ny, nz=nz, pbc=(0, 0, 0), mu_s=3.23 * wl.MU_B, lam=lam, gamma=wl.GAMMA_E, dt=dt, J=J,
                    spacing_nm=spacing, track_nx=track_nx, x0=0, grain_map=gm, grain_ku=ku, grain_axis=axis,
                    macro=tuple(macro), seed=seed, T=T_pass[0].copy(), Bx=z.copy(), By=z.copy(),
                    Bz=np.full(N, bz, dtype=np.float32), sx=z.copy(), sy=z.copy(), sz=mag.astype(np.float32),
                    steps=0, shift_every=shift_every, bit_steps=0,
                    notes="two parallel tracks, two passes (P:122-124)")
    bits = [wl.nrz_bits(n_bits, s) for s in bit_seeds]
    # reader: a footprint about half a bit long and one bit row wide (FWHM = 2.355 sigma)
    sigma = (0.5 * bit_nm / 2.355 / spacing[0], bit_width_nm / 2.355 / spacing[1])
    return TwoTrack(w=w, T_pass=T_pass, bits=bits, track_y=(yc_nm[0] / spacing[1], yc_nm[1] / spacing[1]),
                    bit_planes=bit_planes, shift_every=shift_every, batch=batch, reader_sigma=sigma,
                    spot_plane=0.5 * nx, write_offset=0.5 * bit_width_nm / spacing[0])


def drive_pass(sim, tt: TwoTrack, p: int, set_temperature: Callable, periods: Optional[int] = None,
               on_period: Optional[Callable] = None) -> int:
    """Pass p (0 or 1) of the track-shifting algorithm on `sim` (the oracle or the CUDA context: both expose
    set_field_scale / step_heun / shift_window / track_begin_pass / track_end_pass).  `set_temperature(sim, T)` uploads a
    per-site temperature array.  Returns the number of Heun steps taken."""
    if p > 0:
        sim.track_begin_pass(0)
    set_temperature(sim, tt.T_pass[p])
    periods = tt.n_periods if periods is None else periods
    ax = tt.w.spacing_nm[0]
    x0, steps = 0, 0
    for q in range(1, periods + 1):
        # the head polarity follows the bit the spot centre is over (piecewise constant per shift period)
        sim.set_field_scale(tt.bit_at_plane(p, x0 + tt.spot_plane))
        left = tt.shift_every
        while left > 0:
            n = min(tt.batch, left)
            sim.step_heun(n)
            left -= n
            steps += n
        pl = wl.planes_for_shift(q, ax)
        sim.shift_window(pl)
        x0 += pl
        if on_period is not None:
            on_period(q, x0)
    sim.track_end_pass()
    return steps


def read_tracks(sim, tt: TwoTrack) -> np.ndarray:
    """[2, n_bits]: the read-back figure of merit at every bit centre of both tracks."""
    c = tt.bit_centres()
    step = float(c[1] - c[0]) if len(c) > 1 else 1.0
    return np.stack([np.asarray(sim.track_read_scan(tt.track_y[t], tt.reader_sigma[0], tt.reader_sigma[1],
                                                    float(c[0]), step, len(c))) for t in (0, 1)])
