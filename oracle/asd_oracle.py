"""ctypes wrapper around oracle/asd_oracle.cpp -- the fp64 CPU oracle.

TEST INFRASTRUCTURE ONLY.  May be imported by tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs.  It never imports the CUDA package and the CUDA package
never imports it.  All arithmetic lives in asd_oracle.cpp; this file only marshals arguments.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from dataclasses import dataclass, field
from typing import Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "asd_oracle.cpp")
_LIB = os.path.join(_HERE, "libasd_oracle.so")

GAMMA_E = 1.76085963023e11   # rad s^-1 T^-1
MU_B = 9.2740100783e-24      # J/T
K_B = 1.380649e-23           # J/K


def build(force: bool = False) -> str:
    """Compile the oracle with g++ (-O2, OpenMP).  Returns the path of the shared library."""
    if (not force and os.path.exists(_LIB)
            and os.path.getmtime(_LIB) >= os.path.getmtime(_SRC)):
        return _LIB
    cmd = ["g++", "-O2", "-std=c++17", "-fPIC", "-shared", "-fopenmp", "-ffp-contract=off",
           "-o", _LIB, _SRC]
    subprocess.run(cmd, check=True)
    return _LIB


class _Desc(C.Structure):
    _fields_ = [
        ("lattice", C.c_int32), ("nx", C.c_int32), ("ny", C.c_int32), ("nz", C.c_int32),
        ("pbc", C.c_int32 * 3),
        ("n_grains", C.c_int32),
        ("mu_s", C.c_double), ("lam", C.c_double), ("gamma", C.c_double), ("dt", C.c_double),
        ("J", C.c_double * 3),
        ("track_nx", C.c_int64), ("x0", C.c_int64),
        ("grain_map", C.POINTER(C.c_int32)),
        ("grain_ku", C.POINTER(C.c_double)),
        ("grain_axis", C.POINTER(C.c_double)),
        ("macro", C.c_int32 * 3),
        ("ell_width", C.c_int32),
        ("ell_idx", C.POINTER(C.c_int32)),
        ("ell_J", C.POINTER(C.c_double)),
        ("seed", C.c_uint64),
    ]


class _MmDesc(C.Structure):
    _fields_ = [
        ("mcx", C.c_int32 * 2), ("every", C.c_int32),
        ("Ms0", C.c_double), ("A0", C.c_double * 3),
        ("K0", C.POINTER(C.c_double)), ("Tc", C.POINTER(C.c_double)),
        ("cell_grain", C.POINTER(C.c_int32)),
        ("spacing", C.c_double * 3),
    ]


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        L.orc_create.restype = C.c_void_p
        L.orc_create.argtypes = [C.POINTER(_Desc)]
        L.orc_destroy.argtypes = [C.c_void_p]
        L.orc_set_threads.argtypes = [C.c_void_p, C.c_int]
        L.orc_max_threads.restype = C.c_int
        fp = C.POINTER(C.c_float)
        dp = C.POINTER(C.c_double)
        ip64 = C.POINTER(C.c_int64)
        L.orc_set_spins.argtypes = [C.c_void_p, fp, fp, fp]
        L.orc_get_spins.argtypes = [C.c_void_p, dp, dp, dp]
        L.orc_set_spins_f64.argtypes = [C.c_void_p, dp, dp, dp]
        L.orc_set_fields.argtypes = [C.c_void_p, fp, fp, fp, fp]
        L.orc_set_field_scale.argtypes = [C.c_void_p, C.c_float]
        L.orc_step_heun.argtypes = [C.c_void_p, C.c_int64]
        L.orc_field.argtypes = [C.c_void_p, C.c_int, dp, dp, dp]
        L.orc_energy.restype = C.c_double
        L.orc_energy.argtypes = [C.c_void_p]
        L.orc_magnetisation.argtypes = [C.c_void_p, dp, dp]
        L.orc_grain_magnetisation.argtypes = [C.c_void_p, dp]
        L.orc_shift_window.restype = C.c_int
        L.orc_shift_window.argtypes = [C.c_void_p, C.c_int32]
        L.orc_track_set_init.argtypes = [C.c_void_p, fp, C.c_float]
        L.orc_track_ncell.restype = C.c_int64
        L.orc_track_ncell.argtypes = [C.c_void_p, ip64]
        L.orc_track_get.argtypes = [C.c_void_p, dp, ip64, dp]
        L.orc_track_end_pass.restype = C.c_int
        L.orc_track_end_pass.argtypes = [C.c_void_p]
        L.orc_track_begin_pass.restype = C.c_int
        L.orc_track_begin_pass.argtypes = [C.c_void_p, C.c_int64]
        L.orc_track_read_scan.argtypes = [C.c_void_p, C.c_double, C.c_double, C.c_double, C.c_double, C.c_double,
                                          C.c_int64, dp]
        L.orc_get_counters.argtypes = [C.c_void_p, ip64, ip64, ip64, ip64]
        L.orc_mm_enable.restype = C.c_int
        L.orc_mm_enable.argtypes = [C.c_void_p, C.POINTER(_MmDesc)]
        L.orc_mm_cells.restype = C.c_int64
        L.orc_mm_cells.argtypes = [C.c_void_p, C.c_int]
        L.orc_mm_set_fields.argtypes = [C.c_void_p, C.c_int, dp, dp, dp, dp]
        L.orc_mm_set_m.argtypes = [C.c_void_p, C.c_int, dp]
        L.orc_mm_get_m.argtypes = [C.c_void_p, C.c_int, dp]
        L.orc_mm_get_params.argtypes = [C.c_void_p, C.c_int, dp, dp]
        L.orc_mm_field.argtypes = [C.c_void_p, C.c_int, dp]
        L.orc_mm_step.argtypes = [C.c_void_p, C.c_int64, C.c_double]
        L.orc_mm_me.restype = C.c_double
        L.orc_mm_me.argtypes = [C.c_double, C.c_double, C.c_double]
        L.orc_langevin.restype = C.c_double
        L.orc_langevin.argtypes = [C.c_double]
        L.orc_set_counters.argtypes = [C.c_void_p, C.c_int64, C.c_int64, C.c_int64]
        u32p = C.POINTER(C.c_uint32)
        L.orc_philox4x32_10.argtypes = [u32p, u32p, u32p]
        L.orc_philox_block.argtypes = [C.c_uint64, C.c_uint64, C.c_uint64, C.c_uint32, u32p]
        L.orc_uniform.restype = C.c_double
        L.orc_uniform.argtypes = [C.c_uint32]
        L.orc_normals3.argtypes = [C.c_uint64, C.c_uint64, C.c_uint64, dp]
        L.orc_normals3_bulk.argtypes = [C.c_uint64, C.c_uint64, C.c_uint64, C.c_int64, dp]
        L.orc_theta_max.restype = C.c_double
        L.orc_theta_max.argtypes = [C.c_double]
        L.orc_sigma.restype = C.c_double
        L.orc_sigma.argtypes = [C.c_void_p, C.c_double]
        L.orc_enable_demag.argtypes = [C.c_void_p, dp]
        L.orc_set_demag_every.argtypes = [C.c_void_p, C.c_int]
        L.orc_newell_tensor.argtypes = [dp, dp, dp]
        L.orc_demag_cells.argtypes = [C.c_void_p, dp, ip64]
        L.orc_enable_track_stray.restype = C.c_int
        L.orc_enable_track_stray.argtypes = [C.c_void_p, C.c_int, C.c_int]
        L.orc_stray_cells.argtypes = [C.c_void_p, dp]
        L.orc_enable_track_exchange.argtypes = [C.c_void_p, C.c_int]
        _lib = L
    return _lib


def _f32(a):
    return None if a is None else np.ascontiguousarray(a, dtype=np.float32)


def _ptr(a, ct):
    return None if a is None else a.ctypes.data_as(C.POINTER(ct))


# ---- free functions (building blocks used by the pins) ----
def philox4x32_10(key: Sequence[int], ctr: Sequence[int]) -> np.ndarray:
    k = (C.c_uint32 * 2)(*[int(x) & 0xFFFFFFFF for x in key])
    c = (C.c_uint32 * 4)(*[int(x) & 0xFFFFFFFF for x in ctr])
    o = (C.c_uint32 * 4)()
    lib().orc_philox4x32_10(k, c, o)
    return np.array(list(o), dtype=np.uint32)


def philox_block(seed: int, n: int, g: int, stream: int) -> np.ndarray:
    o = (C.c_uint32 * 4)()
    lib().orc_philox_block(C.c_uint64(seed), C.c_uint64(n), C.c_uint64(g), C.c_uint32(stream), o)
    return np.array(list(o), dtype=np.uint32)


def uniform(r: int) -> float:
    return float(lib().orc_uniform(C.c_uint32(r)))


def normals3(seed: int, step: int, g: int) -> np.ndarray:
    o = np.zeros(3)
    lib().orc_normals3(C.c_uint64(seed), C.c_uint64(step), C.c_uint64(g), _ptr(o, C.c_double))
    return o


def normals3_bulk(seed: int, step: int, g0: int, count: int) -> np.ndarray:
    o = np.zeros((count, 3))
    lib().orc_normals3_bulk(C.c_uint64(seed), C.c_uint64(step), C.c_uint64(g0), C.c_int64(count),
                            _ptr(o, C.c_double))
    return o


def newell_tensor(cell, R) -> np.ndarray:
    """(Nxx, Nyy, Nzz, Nxy, Nxz, Nyz) of two equal cuboids `cell` (edge lengths) at centre offset R."""
    c = np.ascontiguousarray(cell, dtype=np.float64); r = np.ascontiguousarray(R, dtype=np.float64)
    out = np.zeros(6)
    lib().orc_newell_tensor(_ptr(c, C.c_double), _ptr(r, C.c_double), _ptr(out, C.c_double))
    return out


def theta_max(m: float) -> float:
    return float(lib().orc_theta_max(C.c_double(m)))


def mm_me(T: float, Tc: float, mu_s_Bext: float = 0.0) -> float:
    """m_e(T): largest root of m = B(3 T_C m / T + mu_s B_ext / k_B T)."""
    return float(lib().orc_mm_me(C.c_double(T), C.c_double(Tc), C.c_double(mu_s_Bext)))


def langevin(x: float) -> float:
    return float(lib().orc_langevin(C.c_double(x)))


def max_threads() -> int:
    return int(lib().orc_max_threads())


@dataclass
class LatticeSpec:
    """Plain description of a lattice; mirrors the quantities of SURVEY 8(b) but is the oracle's own."""
    lattice: int                       # 0 = SC, 1 = L1_0 Fe sublattice
    nx: int
    ny: int
    nz: int
    pbc: Sequence[int] = (0, 0, 0)
    mu_s: float = 3.23 * MU_B
    lam: float = 0.1
    gamma: float = GAMMA_E
    dt: float = 1e-15
    J: Sequence[float] = (6.71e-21, 0.0, 0.0)
    track_nx: Optional[int] = None
    x0: int = 0
    grain_map: Optional[np.ndarray] = None     # [track_nx, ny] int32, -1 vacant
    grain_ku: Optional[np.ndarray] = None      # [n_grains]
    grain_axis: Optional[np.ndarray] = None    # [n_grains, 3]
    macro: Sequence[int] = (7, 7, 7)
    ell_idx: Optional[np.ndarray] = None       # [N, W] int32
    ell_J: Optional[np.ndarray] = None         # [N, W] float
    seed: int = 1


class Oracle:
    def __init__(self, spec: LatticeSpec):
        L = lib()
        self.spec = spec
        track_nx = spec.track_nx if spec.track_nx is not None else spec.nx
        gm = spec.grain_map
        if gm is None:
            gm = np.zeros((track_nx, spec.ny), dtype=np.int32)
        self._gm = np.ascontiguousarray(gm, dtype=np.int32).reshape(track_nx, spec.ny)
        ku = spec.grain_ku if spec.grain_ku is not None else np.zeros(1)
        ax = spec.grain_axis if spec.grain_axis is not None else np.array([[0.0, 0.0, 1.0]])
        self._ku = np.ascontiguousarray(ku, dtype=np.float64).reshape(-1)
        self._ax = np.ascontiguousarray(ax, dtype=np.float64).reshape(-1, 3)
        assert self._ax.shape[0] == self._ku.shape[0]
        assert self._gm.max(initial=-1) < self._ku.shape[0]
        d = _Desc()
        d.lattice, d.nx, d.ny, d.nz = spec.lattice, spec.nx, spec.ny, spec.nz
        d.pbc = (C.c_int32 * 3)(*[int(x) for x in spec.pbc])
        d.n_grains = self._ku.shape[0]
        d.mu_s, d.lam, d.gamma, d.dt = spec.mu_s, spec.lam, spec.gamma, spec.dt
        d.J = (C.c_double * 3)(*[float(x) for x in spec.J])
        d.track_nx, d.x0 = track_nx, spec.x0
        d.grain_map = _ptr(self._gm, C.c_int32)
        d.grain_ku = _ptr(self._ku, C.c_double)
        d.grain_axis = _ptr(self._ax, C.c_double)
        d.macro = (C.c_int32 * 3)(*[int(x) for x in spec.macro])
        self.N = spec.nx * spec.ny * spec.nz
        if spec.ell_idx is not None:
            self._ei = np.ascontiguousarray(spec.ell_idx, dtype=np.int32).reshape(self.N, -1)
            self._ej = np.ascontiguousarray(spec.ell_J, dtype=np.float64).reshape(self.N, -1)
            d.ell_width = self._ei.shape[1]
            d.ell_idx = _ptr(self._ei, C.c_int32)
            d.ell_J = _ptr(self._ej, C.c_double)
        else:
            d.ell_width = 0
        d.seed = spec.seed
        self._h = L.orc_create(C.byref(d))
        if not self._h:
            raise ValueError("orc_create rejected the description")
        self.n_grains = int(d.n_grains)

    def __del__(self):
        try:
            if getattr(self, "_h", None):
                lib().orc_destroy(self._h)
                self._h = None
        except Exception:
            pass

    def set_threads(self, n: int):
        lib().orc_set_threads(self._h, int(n))

    def set_spins(self, sx, sy, sz):
        sx, sy, sz = _f32(sx).reshape(-1), _f32(sy).reshape(-1), _f32(sz).reshape(-1)
        assert sx.size == self.N and sy.size == self.N and sz.size == self.N
        lib().orc_set_spins(self._h, _ptr(sx, C.c_float), _ptr(sy, C.c_float), _ptr(sz, C.c_float))

    def set_spins_f64(self, S):
        """S: [3, N] float64, stored as given (vacant sites 0)."""
        S = np.ascontiguousarray(S, dtype=np.float64).reshape(3, self.N)
        lib().orc_set_spins_f64(self._h, _ptr(S[0], C.c_double), _ptr(S[1], C.c_double), _ptr(S[2], C.c_double))

    def get_spins(self) -> np.ndarray:
        """Returns [3, N] float64."""
        o = np.zeros((3, self.N))
        lib().orc_get_spins(self._h, _ptr(o[0], C.c_double), _ptr(o[1], C.c_double), _ptr(o[2], C.c_double))
        return o

    def set_fields(self, T=None, Bx=None, By=None, Bz=None):
        arrs = [None if a is None else _f32(a).reshape(-1) for a in (T, Bx, By, Bz)]
        for a in arrs:
            assert a is None or a.size == self.N
        lib().orc_set_fields(self._h, *[_ptr(a, C.c_float) for a in arrs])

    def enable_demag(self, spacing_m):
        """Demagnetising field on (Eq. (6)-(7)); spacing_m = lattice constants (ax, ay, az) in metres."""
        a = np.ascontiguousarray(spacing_m, dtype=np.float64)
        lib().orc_enable_demag(self._h, _ptr(a, C.c_double))

    def set_demag_every(self, every: int):
        """0: the field is recomputed in every Heun stage; P >= 1: from S at every P-th step, held in between."""
        lib().orc_set_demag_every(self._h, C.c_int(every))

    def demag_cells(self) -> np.ndarray:
        """Demagnetising field per window macrocell, Tesla: [dcx, dcy, dcz, 3]."""
        dims = np.zeros(3, dtype=np.int64)
        lib().orc_demag_cells(self._h, None, _ptr(dims, C.c_int64))
        out = np.zeros((int(dims[0]), int(dims[1]), int(dims[2]), 3))
        lib().orc_demag_cells(self._h, _ptr(out, C.c_double), _ptr(dims, C.c_int64))
        return out

    def enable_track_stray(self, on: bool = True, range_cells: int = 0) -> int:
        """Stray field of the frozen track on the window's macrocells (needs enable_demag); 0 = every track cell."""
        return int(lib().orc_enable_track_stray(self._h, int(bool(on)), int(range_cells)))

    def enable_track_exchange(self, on: bool = True):
        """The window's first / last plane exchange coupled to the frozen track's direction (reading E1)."""
        lib().orc_enable_track_exchange(self._h, int(bool(on)))

    def stray_cells(self) -> np.ndarray:
        """The track's stray field per window macrocell, Tesla: [dcx, dcy, dcz, 3]."""
        dims = np.zeros(3, dtype=np.int64)
        lib().orc_demag_cells(self._h, None, _ptr(dims, C.c_int64))
        out = np.zeros((int(dims[0]), int(dims[1]), int(dims[2]), 3))
        lib().orc_stray_cells(self._h, _ptr(out, C.c_double))
        return out

    def set_field_scale(self, s: float):
        lib().orc_set_field_scale(self._h, C.c_float(s))

    def step_heun(self, n: int = 1):
        lib().orc_step_heun(self._h, C.c_int64(n))

    def field(self, with_noise: bool = False) -> np.ndarray:
        o = np.zeros((3, self.N))
        lib().orc_field(self._h, int(with_noise), _ptr(o[0], C.c_double), _ptr(o[1], C.c_double),
                        _ptr(o[2], C.c_double))
        return o

    def energy(self) -> float:
        return float(lib().orc_energy(self._h))

    def magnetisation(self):
        m = np.zeros(3)
        n = C.c_double(0)
        lib().orc_magnetisation(self._h, _ptr(m, C.c_double), C.byref(n))
        return m, n.value

    def grain_magnetisation(self) -> np.ndarray:
        m = np.zeros((self.n_grains, 3))
        lib().orc_grain_magnetisation(self._h, _ptr(m, C.c_double))
        return m

    def shift_window(self, p: int) -> int:
        return int(lib().orc_shift_window(self._h, C.c_int32(p)))

    def track_dims(self):
        d = (C.c_int64 * 3)()
        lib().orc_track_ncell(self._h, d)
        return tuple(int(x) for x in d)

    def track_set_init(self, mean_spin=None, m0: float = 1.0):
        a = None if mean_spin is None else _f32(mean_spin).reshape(-1)
        lib().orc_track_set_init(self._h, _ptr(a, C.c_float), C.c_float(m0))

    def track_get(self):
        nc = int(np.prod(self.track_dims()))
        mean = np.zeros((nc, 3))
        cnt = np.zeros(nc, dtype=np.int64)
        sm = np.zeros((nc, 3))
        lib().orc_track_get(self._h, _ptr(mean, C.c_double), _ptr(cnt, C.c_int64), _ptr(sm, C.c_double))
        return mean, cnt, sm

    def track_end_pass(self) -> int:
        """Window -> track by Eq. (6); what the pass wrote becomes what lies ahead of the next one (reading T1)."""
        return int(lib().orc_track_end_pass(self._h))

    def track_begin_pass(self, x0_new: int = 0) -> int:
        """Written store cleared, pass += 1, window back at plane x0_new and regenerated from the track (reading T2)."""
        return int(lib().orc_track_begin_pass(self._h, C.c_int64(x0_new)))

    def track_read_scan(self, y_r: float, sigma_x: float, sigma_y: float, x_first: float, x_step: float,
                        count: int) -> np.ndarray:
        """Mean S_z per written magnetic site under a Gaussian reader footprint, at `count` positions (reading T3)."""
        out = np.zeros(int(count))
        lib().orc_track_read_scan(self._h, C.c_double(y_r), C.c_double(sigma_x), C.c_double(sigma_y),
                                  C.c_double(x_first), C.c_double(x_step), C.c_int64(count), _ptr(out, C.c_double))
        return out

    # ---- multiscale window: micromagnetic meshes either side of the atomistic mesh ----
    def mm_enable(self, mcx, every, Ms0, A0, K0, Tc, cell_grain, spacing_m) -> int:
        d = _MmDesc()
        d.mcx = (C.c_int32 * 2)(int(mcx[0]), int(mcx[1]))
        d.every = int(every)
        d.Ms0 = float(Ms0)
        A0 = np.broadcast_to(np.asarray(A0, dtype=np.float64), (3,))
        d.A0 = (C.c_double * 3)(*[float(x) for x in A0])
        self._mmK = np.ascontiguousarray(K0, dtype=np.float64).reshape(-1)
        self._mmT = np.ascontiguousarray(Tc, dtype=np.float64).reshape(-1)
        self._mmG = np.ascontiguousarray(cell_grain, dtype=np.int32).reshape(-1)
        assert self._mmK.size == self.n_grains and self._mmT.size == self.n_grains
        ncx, ncy, _ = self.track_dims()
        assert self._mmG.size == ncx * ncy
        d.K0, d.Tc, d.cell_grain = _ptr(self._mmK, C.c_double), _ptr(self._mmT, C.c_double), _ptr(self._mmG, C.c_int32)
        d.spacing = (C.c_double * 3)(*[float(x) for x in spacing_m])
        st = int(lib().orc_mm_enable(self._h, C.byref(d)))
        if st == 0:
            self.mm_mcx = (int(mcx[0]), int(mcx[1]))
        return st

    def mm_shape(self, side: int):
        _, ncy, ncz = self.track_dims()
        return (self.mm_mcx[side], ncy, ncz)

    def mm_set_fields(self, side: int, T=None, Bx=None, By=None, Bz=None):
        n = int(np.prod(self.mm_shape(side)))
        arrs = [None if a is None else np.ascontiguousarray(a, dtype=np.float64).reshape(-1) for a in (T, Bx, By, Bz)]
        for a in arrs:
            assert a is None or a.size == n
        lib().orc_mm_set_fields(self._h, int(side), *[_ptr(a, C.c_double) for a in arrs])

    def mm_set_m(self, side: int, m):
        a = np.ascontiguousarray(m, dtype=np.float64).reshape(-1)
        assert a.size == 3 * int(np.prod(self.mm_shape(side)))
        lib().orc_mm_set_m(self._h, int(side), _ptr(a, C.c_double))

    def mm_get_m(self, side: int) -> np.ndarray:
        """[mcx, ncy, ncz, 3]"""
        out = np.zeros(self.mm_shape(side) + (3,))
        lib().orc_mm_get_m(self._h, int(side), _ptr(out, C.c_double))
        return out

    def mm_params(self, side: int):
        """(m_e, alpha), each [mcx, ncy, ncz]"""
        me, al = np.zeros(self.mm_shape(side)), np.zeros(self.mm_shape(side))
        lib().orc_mm_get_params(self._h, int(side), _ptr(me, C.c_double), _ptr(al, C.c_double))
        return me, al

    def mm_field(self, side: int) -> np.ndarray:
        """Effective field per cell, Tesla, [mcx, ncy, ncz, 3] (boundary data exchanged now)."""
        out = np.zeros(self.mm_shape(side) + (3,))
        lib().orc_mm_field(self._h, int(side), _ptr(out, C.c_double))
        return out

    def mm_step(self, n: int, h: float):
        """n RK4 steps of length h [s] on the meshes alone."""
        lib().orc_mm_step(self._h, C.c_int64(n), C.c_double(h))

    def counters(self):
        a, b, c, d = C.c_int64(0), C.c_int64(0), C.c_int64(0), C.c_int64(0)
        lib().orc_get_counters(self._h, C.byref(a), C.byref(b), C.byref(c), C.byref(d))
        return {"step": a.value, "shift": b.value, "x0": c.value, "pass": d.value}

    def set_counters(self, step: int, shift: int = 0, pass_: int = 0):
        lib().orc_set_counters(self._h, C.c_int64(step), C.c_int64(shift), C.c_int64(pass_))

    def sigma(self, T: float) -> float:
        return float(lib().orc_sigma(self._h, C.c_double(T)))


def spec_from_workload(w, **over) -> "LatticeSpec":
    """asd_inputs.Workload -> LatticeSpec (argument marshalling only)."""
    d = dict(lattice=w.lattice, nx=w.nx, ny=w.ny, nz=w.nz, pbc=w.pbc, mu_s=w.mu_s, lam=w.lam, gamma=w.gamma,
             dt=w.dt, J=w.J, track_nx=w.track_nx, x0=w.x0, grain_map=w.grain_map,
             grain_ku=np.asarray(w.grain_ku, dtype=np.float64), grain_axis=np.asarray(w.grain_axis, dtype=np.float64),
             macro=w.macro, seed=w.seed)
    d.update(over)
    return LatticeSpec(**d)


def from_workload(w, **over) -> "Oracle":
    """An Oracle holding the workload's lattice, spins and fields."""
    o = Oracle(spec_from_workload(w, **over))
    o.set_spins(w.sx, w.sy, w.sz)
    o.set_fields(w.T, w.Bx, w.By, w.Bz)
    return o
