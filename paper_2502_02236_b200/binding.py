"""ctypes binding over libasd.so -- argument marshalling only (include/asd.h is the contract).

Every method of `Context` has the name of the C call it wraps (minus the asd_ prefix) and does nothing but
convert arguments: torch tensors -> device pointers, numpy arrays -> host pointers.
"""
from __future__ import annotations

import ctypes as C
import os
from dataclasses import dataclass
from typing import Optional, Sequence

import numpy as np

ASD_SC, ASD_L10_FE = 0, 1
KERNEL_AUTO, KERNEL_GENERAL, KERNEL_FAST, KERNEL_TMA, KERNEL_FUSED, KERNEL_PERSISTENT = 0, 1, 2, 3, 4, 5
GRAPH_AUTO, GRAPH_OFF, GRAPH_ON = 0, 1, 2
_STATUS = {0: "ASD_OK", 1: "ASD_EINVAL", 2: "ASD_ENOMEM", 3: "ASD_ECUDA", 4: "ASD_ESTATE", 5: "ASD_EUNSUPPORTED"}

EXPORTED_SYMBOLS = [
    "asd_workspace_bytes", "asd_create_lattice", "asd_destroy", "asd_set_spins", "asd_get_spins",
    "asd_set_spins_host", "asd_get_spins_host", "asd_set_fields", "asd_set_fields_host", "asd_set_field_scale",
    "asd_step_heun", "asd_set_kernel", "asd_set_graph_mode", "asd_demag_workspace_bytes", "asd_enable_demag",
    "asd_demag_field", "asd_demag_held_field", "asd_set_demag_every", "asd_staging_bytes", "asd_set_staging", "asd_stage_fields_host",
    "asd_commit_fields", "asd_shift_window", "asd_magnetisation", "asd_grain_magnetisation",
    "asd_track_dims", "asd_track_set_init", "asd_track_get",
    "asd_track_end_pass", "asd_track_begin_pass", "asd_track_read_scan",
    "asd_mm_workspace_bytes", "asd_mm_enable", "asd_mm_dims", "asd_mm_set_fields_host", "asd_mm_set_m_host",
    "asd_mm_get_m_host", "asd_planes_view", "asd_magnetisation_planes",
    "asd_track_stray_workspace_bytes", "asd_enable_track_stray", "asd_track_stray_field",
    "asd_track_exchange_workspace_bytes", "asd_enable_track_exchange", "asd_get_counters", "asd_set_counters",
    "asd_spin_sum_noalloc", "asd_launch_count", "asd_last_error", "asd_version",
]


class AsdError(RuntimeError):
    def __init__(self, status: int, msg: str):
        super().__init__(f"{_STATUS.get(status, status)}: {msg}")
        self.status = status


class _Desc(C.Structure):
    _fields_ = [
        ("lattice", C.c_int32), ("nx", C.c_int32), ("ny", C.c_int32), ("nz", C.c_int32),
        ("pbc", C.c_int32 * 3),
        ("mu_s", C.c_double), ("lam", C.c_double), ("gamma", C.c_double), ("dt", C.c_double),
        ("J", C.c_double * 3),
        ("track_nx", C.c_int64), ("x0", C.c_int64),
        ("grain_map", C.POINTER(C.c_int32)),
        ("n_grains", C.c_int32),
        ("grain_ku", C.POINTER(C.c_float)),
        ("grain_axis", C.POINTER(C.c_float)),
        ("macro", C.c_int32 * 3),
        ("ell_idx", C.POINTER(C.c_int32)),
        ("ell_J", C.POINTER(C.c_float)),
        ("ell_width", C.c_int32),
        ("seed", C.c_uint64),
    ]


class _MmDesc(C.Structure):
    _fields_ = [
        ("mcx", C.c_int32 * 2), ("every", C.c_int32),
        ("Ms0", C.c_double), ("A0", C.c_double * 3),
        ("K0", C.POINTER(C.c_double)), ("Tc", C.POINTER(C.c_double)),
        ("cell_grain", C.POINTER(C.c_int32)),
        ("spacing_m", C.c_double * 3),
    ]


_HERE = os.path.dirname(os.path.abspath(__file__))
_lib = None


def lib_path() -> str:
    return os.path.join(_HERE, "libasd.so")


def load_library(build_if_missing: bool = True):
    """Loads libasd.so (building it with nvcc if it is missing or stale).  Fails loudly: there is no fallback."""
    global _lib
    if _lib is not None:
        return _lib
    if build_if_missing:
        from . import build as _build
        try:
            _build.build()
        except Exception as e:  # stale sources without nvcc: use the existing library if there is one
            if not os.path.exists(lib_path()):
                raise RuntimeError(f"libasd.so is missing and cannot be built: {e}") from e
    if not os.path.exists(lib_path()):
        raise RuntimeError("libasd.so is missing: run `python -m paper_2502_02236_b200.build`")
    L = C.CDLL(lib_path())
    fp, dp, ip64 = C.c_void_p, C.POINTER(C.c_double), C.POINTER(C.c_int64)
    L.asd_workspace_bytes.restype = C.c_size_t
    L.asd_workspace_bytes.argtypes = [C.POINTER(_Desc)]
    L.asd_create_lattice.argtypes = [C.POINTER(_Desc), C.c_void_p, C.c_size_t, C.c_void_p, C.POINTER(C.c_void_p)]
    L.asd_destroy.argtypes = [C.c_void_p]
    for name in ("asd_set_spins", "asd_get_spins", "asd_set_spins_host", "asd_get_spins_host"):
        getattr(L, name).argtypes = [C.c_void_p, fp, fp, fp]
    for name in ("asd_set_fields", "asd_set_fields_host"):
        getattr(L, name).argtypes = [C.c_void_p, fp, fp, fp, fp]
    L.asd_set_field_scale.argtypes = [C.c_void_p, C.c_float]
    L.asd_staging_bytes.restype = C.c_size_t
    L.asd_staging_bytes.argtypes = [C.c_void_p]
    L.asd_set_staging.argtypes = [C.c_void_p, C.c_void_p, C.c_size_t]
    L.asd_stage_fields_host.argtypes = [C.c_void_p, fp, fp, fp, fp]
    L.asd_commit_fields.argtypes = [C.c_void_p]
    L.asd_step_heun.argtypes = [C.c_void_p, C.c_int64]
    L.asd_set_kernel.argtypes = [C.c_void_p, C.c_int32]
    L.asd_set_graph_mode.argtypes = [C.c_void_p, C.c_int32]
    L.asd_demag_workspace_bytes.restype = C.c_size_t
    L.asd_demag_workspace_bytes.argtypes = [C.c_void_p]
    L.asd_enable_demag.argtypes = [C.c_void_p, dp, C.c_void_p, C.c_size_t]
    L.asd_demag_field.argtypes = [C.c_void_p, fp, C.POINTER(C.c_int64)]
    L.asd_demag_held_field.argtypes = [C.c_void_p, fp, C.POINTER(C.c_int64)]
    L.asd_set_demag_every.argtypes = [C.c_void_p, C.c_int32]
    L.asd_track_stray_workspace_bytes.restype = C.c_size_t
    L.asd_track_stray_workspace_bytes.argtypes = [C.c_void_p, C.c_int32]
    L.asd_enable_track_stray.argtypes = [C.c_void_p, C.c_int32, C.c_int32, C.c_void_p, C.c_size_t]
    L.asd_track_stray_field.argtypes = [C.c_void_p, fp]
    L.asd_track_exchange_workspace_bytes.restype = C.c_size_t
    L.asd_track_exchange_workspace_bytes.argtypes = [C.c_void_p]
    L.asd_enable_track_exchange.argtypes = [C.c_void_p, C.c_int32, C.c_void_p, C.c_size_t]
    L.asd_shift_window.argtypes = [C.c_void_p, C.c_int32]
    L.asd_magnetisation.argtypes = [C.c_void_p, dp, dp]
    L.asd_spin_sum_noalloc.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_size_t, C.c_void_p, C.c_void_p]
    L.asd_grain_magnetisation.argtypes = [C.c_void_p, dp]
    L.asd_track_dims.argtypes = [C.c_void_p, ip64]
    L.asd_track_set_init.argtypes = [C.c_void_p, C.c_void_p, C.c_float]
    L.asd_track_get.argtypes = [C.c_void_p, dp, ip64]
    L.asd_track_end_pass.argtypes = [C.c_void_p]
    L.asd_track_begin_pass.argtypes = [C.c_void_p, C.c_int64]
    L.asd_track_read_scan.argtypes = [C.c_void_p, C.c_double, C.c_double, C.c_double, C.c_double, C.c_double,
                                      C.c_int64, dp]
    L.asd_mm_workspace_bytes.restype = C.c_size_t
    L.asd_mm_workspace_bytes.argtypes = [C.c_void_p, C.POINTER(_MmDesc)]
    L.asd_mm_enable.argtypes = [C.c_void_p, C.POINTER(_MmDesc), C.c_void_p, C.c_size_t]
    L.asd_mm_dims.argtypes = [C.c_void_p, C.c_int32, ip64]
    L.asd_mm_set_fields_host.argtypes = [C.c_void_p, C.c_int32, fp, fp, fp, fp]
    L.asd_mm_set_m_host.argtypes = [C.c_void_p, C.c_int32, fp]
    L.asd_mm_get_m_host.argtypes = [C.c_void_p, C.c_int32, fp]
    L.asd_planes_view.argtypes = [C.c_void_p, C.c_int32, C.c_int32, C.c_int32, C.POINTER(C.c_void_p), C.POINTER(C.c_size_t)]
    L.asd_magnetisation_planes.argtypes = [C.c_void_p, C.c_int32, C.c_int32, dp, dp]
    L.asd_get_counters.argtypes = [C.c_void_p, ip64, ip64, ip64, ip64]
    L.asd_set_counters.argtypes = [C.c_void_p, C.c_int64, C.c_int64, C.c_int64]
    L.asd_launch_count.restype = C.c_int64
    L.asd_launch_count.argtypes = [C.c_void_p]
    L.asd_last_error.restype = C.c_char_p
    L.asd_last_error.argtypes = [C.c_void_p]
    L.asd_version.restype = C.c_char_p
    _lib = L
    return L


def version() -> str:
    return load_library().asd_version().decode()


@dataclass
class LatticeDesc:
    """Python mirror of asd_lattice_desc (include/asd.h)."""
    lattice: int
    nx: int
    ny: int
    nz: int
    pbc: Sequence[int] = (0, 0, 0)
    mu_s: float = 3.23 * 9.2740100783e-24
    lam: float = 0.1
    gamma: float = 0.0
    dt: float = 1e-15
    J: Sequence[float] = (6.71e-21, 0.0, 0.0)
    track_nx: Optional[int] = None
    x0: int = 0
    grain_map: Optional[np.ndarray] = None
    n_grains: int = 1
    grain_ku: Optional[np.ndarray] = None
    grain_axis: Optional[np.ndarray] = None
    macro: Sequence[int] = (7, 7, 7)
    ell_idx: Optional[np.ndarray] = None
    ell_J: Optional[np.ndarray] = None
    seed: int = 1

    def to_c(self):
        """Returns (struct, keepalive list)."""
        d = _Desc()
        keep = []
        d.lattice, d.nx, d.ny, d.nz = int(self.lattice), int(self.nx), int(self.ny), int(self.nz)
        d.pbc = (C.c_int32 * 3)(*[int(x) for x in self.pbc])
        d.mu_s, d.lam, d.gamma, d.dt = float(self.mu_s), float(self.lam), float(self.gamma), float(self.dt)
        d.J = (C.c_double * 3)(*[float(x) for x in self.J])
        d.track_nx = int(self.track_nx if self.track_nx is not None else self.nx)
        d.x0 = int(self.x0)

        def host(a, dt, ct):
            if a is None:
                return None
            arr = np.ascontiguousarray(a, dtype=dt)
            keep.append(arr)
            return arr.ctypes.data_as(C.POINTER(ct))
        d.grain_map = host(self.grain_map, np.int32, C.c_int32)
        d.n_grains = int(self.n_grains)
        d.grain_ku = host(self.grain_ku, np.float32, C.c_float)
        d.grain_axis = host(self.grain_axis, np.float32, C.c_float)
        d.macro = (C.c_int32 * 3)(*[int(x) for x in self.macro])
        d.ell_idx = host(self.ell_idx, np.int32, C.c_int32)
        d.ell_J = host(self.ell_J, np.float32, C.c_float)
        d.ell_width = 0 if self.ell_idx is None else int(np.asarray(self.ell_idx).reshape(self.nx * self.ny * self.nz, -1).shape[1])
        d.seed = int(self.seed)
        return d, keep


NOALLOC_MAX_COUNT = 8388608     # ASD_NOALLOC_MAX_COUNT (include/asd.h)


def spin_sum_noalloc(sx, sy, sz, out4, stream=None) -> None:
    """asd_spin_sum_noalloc: (sum S_x, sum S_y, sum S_z, number of spins) of three fp32 CUDA tensors into the fp64 CUDA
    tensor out4[4], on `stream` (default: torch's current stream); allocates nothing, does not synchronise."""
    import torch
    L = load_library()
    for t in (sx, sy, sz):
        if not (t.is_cuda and t.dtype == torch.float32 and t.is_contiguous() and t.numel() == sx.numel()):
            raise ValueError("sx, sy, sz: contiguous fp32 CUDA tensors of equal length")
    if not (out4.is_cuda and out4.dtype == torch.float64 and out4.is_contiguous() and out4.numel() == 4):
        raise ValueError("out4: contiguous fp64 CUDA tensor of 4 elements")
    st = stream if stream is not None else torch.cuda.current_stream(sx.device)
    with torch.cuda.device(sx.device):
        rc = L.asd_spin_sum_noalloc(C.c_void_p(sx.data_ptr()), C.c_void_p(sy.data_ptr()), C.c_void_p(sz.data_ptr()),
                                    C.c_size_t(sx.numel()), C.c_void_p(out4.data_ptr()), C.c_void_p(st.cuda_stream))
    if rc != 0:
        raise AsdError(rc, L.asd_last_error(None).decode())


def workspace_bytes(desc: LatticeDesc) -> int:
    d, _keep = desc.to_c()
    return int(load_library().asd_workspace_bytes(C.byref(d)))


def _dev_ptr(t):
    if t is None:
        return None
    import torch
    assert isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float32 and t.is_contiguous()
    return C.c_void_p(t.data_ptr())


def _host_ptr(a, keep):
    if a is None:
        return None
    import torch
    if isinstance(a, torch.Tensor):
        assert not a.is_cuda and a.dtype == torch.float32 and a.is_contiguous()
        keep.append(a)
        return C.c_void_p(a.data_ptr())
    arr = np.ascontiguousarray(a, dtype=np.float32)
    keep.append(arr)
    return C.c_void_p(arr.ctypes.data)


class Context:
    """One asd_ctx plus its torch-allocated workspace.  Methods = the C calls."""

    def __init__(self, desc: LatticeDesc, device: str = "cuda:0", stream=None):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("libasd needs a CUDA device: there is no CPU fallback")
        self._L = load_library()
        self.desc = desc
        self.device = torch.device(device)
        torch.cuda.set_device(self.device)
        d, keep = desc.to_c()
        nbytes = int(self._L.asd_workspace_bytes(C.byref(d)))
        if nbytes == 0:
            raise AsdError(1, self._L.asd_last_error(None).decode())
        self.workspace = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
        base = (self.workspace.data_ptr() + 255) // 256 * 256
        self._stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        h = C.c_void_p()
        st = self._L.asd_create_lattice(C.byref(d), C.c_void_p(base), C.c_size_t(nbytes),
                                        C.c_void_p(self._stream.cuda_stream), C.byref(h))
        if st != 0:
            raise AsdError(st, self._L.asd_last_error(None).decode())
        self._h = h
        self.N = desc.nx * desc.ny * desc.nz
        self.n_grains = desc.n_grains

    def _ck(self, st):
        if st != 0:
            raise AsdError(st, self._L.asd_last_error(self._h).decode())

    def destroy(self):
        if getattr(self, "_h", None):
            self._L.asd_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass

    # ---- spins / fields ----
    def set_spins(self, sx, sy, sz):
        self._ck(self._L.asd_set_spins(self._h, _dev_ptr(sx), _dev_ptr(sy), _dev_ptr(sz)))

    def get_spins(self, sx, sy, sz):
        self._ck(self._L.asd_get_spins(self._h, _dev_ptr(sx), _dev_ptr(sy), _dev_ptr(sz)))

    def set_spins_host(self, sx, sy, sz):
        keep = []
        self._ck(self._L.asd_set_spins_host(self._h, _host_ptr(sx, keep), _host_ptr(sy, keep), _host_ptr(sz, keep)))
        self._sync_if_unpinned(keep)

    def get_spins_host(self) -> np.ndarray:
        out = np.empty((3, self.N), dtype=np.float32)
        self._ck(self._L.asd_get_spins_host(self._h, C.c_void_p(out[0].ctypes.data), C.c_void_p(out[1].ctypes.data),
                                            C.c_void_p(out[2].ctypes.data)))
        return out

    def set_fields(self, T=None, Bx=None, By=None, Bz=None):
        self._ck(self._L.asd_set_fields(self._h, _dev_ptr(T), _dev_ptr(Bx), _dev_ptr(By), _dev_ptr(Bz)))

    def set_fields_host(self, T=None, Bx=None, By=None, Bz=None):
        keep = []
        self._ck(self._L.asd_set_fields_host(self._h, _host_ptr(T, keep), _host_ptr(Bx, keep), _host_ptr(By, keep),
                                             _host_ptr(Bz, keep)))
        self._sync_if_unpinned(keep)

    def stage_fields_host(self, T=None, Bx=None, By=None, Bz=None):
        """asd_stage_fields_host (allocates the staging buffer on first use).  Pass PINNED torch tensors and keep them
        alive and unchanged until commit_fields() has been called and the stream has passed it."""
        import torch
        if getattr(self, "_staging", None) is None:
            nbytes = int(self._L.asd_staging_bytes(self._h))
            self._staging = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
            ptr = (self._staging.data_ptr() + 255) & ~255
            self._ck(self._L.asd_set_staging(self._h, C.c_void_p(ptr), C.c_size_t(nbytes)))
        keep = []
        self._ck(self._L.asd_stage_fields_host(self._h, _host_ptr(T, keep), _host_ptr(Bx, keep), _host_ptr(By, keep),
                                               _host_ptr(Bz, keep)))
        self._staged_keep = keep

    def commit_fields(self):
        self._ck(self._L.asd_commit_fields(self._h))

    def _sync_if_unpinned(self, keep):
        import torch
        if any(not (isinstance(a, torch.Tensor) and a.is_pinned()) for a in keep):
            self._stream.synchronize()      # temporaries must outlive the asynchronous copy

    def set_field_scale(self, s: float):
        self._ck(self._L.asd_set_field_scale(self._h, C.c_float(s)))

    # ---- dynamics ----
    def step_heun(self, n: int = 1):
        self._ck(self._L.asd_step_heun(self._h, C.c_int64(n)))

    def set_kernel(self, variant: int):
        self._ck(self._L.asd_set_kernel(self._h, C.c_int32(variant)))

    def enable_demag(self, spacing_m):
        """asd_enable_demag: spacing_m = lattice constants (ax, ay, az) in metres; allocates the demag workspace."""
        import torch
        nbytes = int(self._L.asd_demag_workspace_bytes(self._h))
        if nbytes == 0:
            raise AsdError(5, "asd_demag_workspace_bytes failed")
        self._demag_ws = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
        ptr = (self._demag_ws.data_ptr() + 255) & ~255
        a = (C.c_double * 3)(*[float(x) for x in spacing_m])
        self._ck(self._L.asd_enable_demag(self._h, a, C.c_void_p(ptr), C.c_size_t(nbytes)))

    def enable_track_stray(self, on: bool = True, range_cells: int = 0):
        """asd_enable_track_stray (allocates its workspace): the frozen track's stray field on the window's macrocells."""
        import torch
        if not on:
            self._ck(self._L.asd_enable_track_stray(self._h, C.c_int32(0), C.c_int32(0), None, C.c_size_t(0)))
            return
        nbytes = int(self._L.asd_track_stray_workspace_bytes(self._h, C.c_int32(range_cells)))
        if nbytes == 0:
            raise AsdError(4, "asd_track_stray_workspace_bytes: asd_enable_demag has not been called")
        self._stray_ws = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
        ptr = (self._stray_ws.data_ptr() + 255) & ~255
        self._ck(self._L.asd_enable_track_stray(self._h, C.c_int32(1), C.c_int32(range_cells), C.c_void_p(ptr), C.c_size_t(nbytes)))

    def enable_track_exchange(self, on: bool = True):
        """asd_enable_track_exchange (allocates its workspace): the window's ends exchange coupled to the frozen track."""
        import torch
        if not on:
            self._ck(self._L.asd_enable_track_exchange(self._h, C.c_int32(0), None, C.c_size_t(0)))
            return
        nbytes = int(self._L.asd_track_exchange_workspace_bytes(self._h))
        self._tex_ws = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
        ptr = (self._tex_ws.data_ptr() + 255) & ~255
        self._ck(self._L.asd_enable_track_exchange(self._h, C.c_int32(1), C.c_void_p(ptr), C.c_size_t(nbytes)))

    def stray_cells(self) -> np.ndarray:
        """asd_track_stray_field: [dcx, dcy, dcz, 3] Tesla."""
        dims = (C.c_int64 * 3)()
        self._ck(self._L.asd_demag_field(self._h, None, dims))
        out = np.zeros((dims[0], dims[1], dims[2], 3), dtype=np.float32)
        self._ck(self._L.asd_track_stray_field(self._h, C.c_void_p(out.ctypes.data)))
        return out

    def set_demag_every(self, every: int):
        self._ck(self._L.asd_set_demag_every(self._h, C.c_int32(every)))

    def demag_field(self) -> np.ndarray:
        """asd_demag_field: demagnetising field of the current spins per macrocell, Tesla, [dcx, dcy, dcz, 3]."""
        dims = (C.c_int64 * 3)()
        self._ck(self._L.asd_demag_field(self._h, None, dims))
        out = np.zeros((dims[0], dims[1], dims[2], 3), dtype=np.float32)
        self._ck(self._L.asd_demag_field(self._h, out.ctypes.data_as(C.POINTER(C.c_float)), dims))
        return out

    def demag_held_field(self) -> np.ndarray:
        """asd_demag_held_field: the cell field as the last Heun stage used it (nothing recomputed), [dcx, dcy, dcz, 3]."""
        dims = (C.c_int64 * 3)()
        self._ck(self._L.asd_demag_held_field(self._h, None, dims))
        out = np.zeros((dims[0], dims[1], dims[2], 3), dtype=np.float32)
        self._ck(self._L.asd_demag_held_field(self._h, out.ctypes.data_as(C.POINTER(C.c_float)), dims))
        return out

    def set_graph_mode(self, mode: int):
        self._ck(self._L.asd_set_graph_mode(self._h, C.c_int32(mode)))

    def shift_window(self, p: int):
        self._ck(self._L.asd_shift_window(self._h, C.c_int32(p)))

    # ---- observables ----
    def magnetisation(self):
        m = np.zeros(3)
        n = C.c_double(0)
        self._ck(self._L.asd_magnetisation(self._h, m.ctypes.data_as(C.POINTER(C.c_double)), C.byref(n)))
        return m, n.value

    def grain_magnetisation(self) -> np.ndarray:
        m = np.zeros((self.n_grains, 3))
        self._ck(self._L.asd_grain_magnetisation(self._h, m.ctypes.data_as(C.POINTER(C.c_double))))
        return m

    # ---- track store ----
    def track_dims(self):
        d = (C.c_int64 * 3)()
        self._ck(self._L.asd_track_dims(self._h, d))
        return tuple(int(x) for x in d)

    def track_set_init(self, mean_spin=None, m0: float = 1.0):
        keep = []
        self._ck(self._L.asd_track_set_init(self._h, _host_ptr(mean_spin, keep), C.c_float(m0)))

    def track_get(self):
        nc = int(np.prod(self.track_dims()))
        s = np.zeros((nc, 3))
        cnt = np.zeros(nc, dtype=np.int64)
        self._ck(self._L.asd_track_get(self._h, s.ctypes.data_as(C.POINTER(C.c_double)),
                                       cnt.ctypes.data_as(C.POINTER(C.c_int64))))
        return s, cnt

    def track_end_pass(self):
        self._ck(self._L.asd_track_end_pass(self._h))

    def track_begin_pass(self, x0_new: int = 0):
        self._ck(self._L.asd_track_begin_pass(self._h, C.c_int64(x0_new)))

    def track_read_scan(self, y_r: float, sigma_x: float, sigma_y: float, x_first: float, x_step: float,
                        count: int) -> np.ndarray:
        out = np.zeros(int(count))
        self._ck(self._L.asd_track_read_scan(self._h, C.c_double(y_r), C.c_double(sigma_x), C.c_double(sigma_y),
                                             C.c_double(x_first), C.c_double(x_step), C.c_int64(count),
                                             out.ctypes.data_as(C.POINTER(C.c_double))))
        return out

    # ---- slab decomposition ----
    def planes_view(self, comp: int, i0: int, n: int):
        """asd_planes_view as a torch tensor over the context's own workspace (no copy): [n * nz * row_stride] fp32."""
        import torch
        ptr, cnt = C.c_void_p(), C.c_size_t()
        self._ck(self._L.asd_planes_view(self._h, C.c_int32(comp), C.c_int32(i0), C.c_int32(n), C.byref(ptr), C.byref(cnt)))
        off = ptr.value - self.workspace.data_ptr()
        return self.workspace[off:off + 4 * cnt.value].view(torch.float32)

    def magnetisation_planes(self, i0: int, n: int):
        s = np.zeros(3)
        cnt = C.c_double(0)
        self._ck(self._L.asd_magnetisation_planes(self._h, C.c_int32(i0), C.c_int32(n),
                                                  s.ctypes.data_as(C.POINTER(C.c_double)), C.byref(cnt)))
        return s, cnt.value

    # ---- multiscale window ----
    def mm_enable(self, mcx, every, Ms0, A0, K0, Tc, cell_grain, spacing_m):
        """asd_mm_enable (allocates the mesh workspace)."""
        import torch
        d = _MmDesc()
        d.mcx = (C.c_int32 * 2)(int(mcx[0]), int(mcx[1]))
        d.every = int(every)
        d.Ms0 = float(Ms0)
        d.A0 = (C.c_double * 3)(*[float(x) for x in np.broadcast_to(np.asarray(A0, dtype=np.float64), (3,))])
        K0 = np.ascontiguousarray(K0, dtype=np.float64).reshape(-1)
        Tc = np.ascontiguousarray(Tc, dtype=np.float64).reshape(-1)
        cg = np.ascontiguousarray(cell_grain, dtype=np.int32).reshape(-1)
        ncx, ncy, _ = self.track_dims()
        if K0.size != self.n_grains or Tc.size != self.n_grains or cg.size != ncx * ncy:
            raise AsdError(1, "mm_enable: K0 / Tc need one entry per grain, cell_grain one per track cell column")
        d.K0 = K0.ctypes.data_as(C.POINTER(C.c_double))
        d.Tc = Tc.ctypes.data_as(C.POINTER(C.c_double))
        d.cell_grain = cg.ctypes.data_as(C.POINTER(C.c_int32))
        d.spacing_m = (C.c_double * 3)(*[float(x) for x in spacing_m])
        nbytes = int(self._L.asd_mm_workspace_bytes(self._h, C.byref(d)))
        if nbytes == 0:
            raise AsdError(1, "asd_mm_workspace_bytes rejected the description")
        self._mm_ws = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
        ptr = (self._mm_ws.data_ptr() + 255) & ~255
        self._ck(self._L.asd_mm_enable(self._h, C.byref(d), C.c_void_p(ptr), C.c_size_t(nbytes)))

    def mm_shape(self, side: int):
        d = (C.c_int64 * 3)()
        self._ck(self._L.asd_mm_dims(self._h, C.c_int32(side), d))
        return tuple(int(x) for x in d)

    def mm_set_fields(self, side: int, T=None, Bx=None, By=None, Bz=None):
        keep = []
        self._ck(self._L.asd_mm_set_fields_host(self._h, C.c_int32(side), _host_ptr(T, keep), _host_ptr(Bx, keep),
                                                _host_ptr(By, keep), _host_ptr(Bz, keep)))

    def mm_set_m(self, side: int, m):
        keep = []
        self._ck(self._L.asd_mm_set_m_host(self._h, C.c_int32(side), _host_ptr(m, keep)))

    def mm_get_m(self, side: int) -> np.ndarray:
        out = np.zeros(self.mm_shape(side) + (3,), dtype=np.float32)
        self._ck(self._L.asd_mm_get_m_host(self._h, C.c_int32(side), C.c_void_p(out.ctypes.data)))
        return out

    # ---- counters ----
    def counters(self):
        a, b, c, d = C.c_int64(0), C.c_int64(0), C.c_int64(0), C.c_int64(0)
        self._ck(self._L.asd_get_counters(self._h, C.byref(a), C.byref(b), C.byref(c), C.byref(d)))
        return {"step": a.value, "shift": b.value, "x0": c.value, "pass": d.value}

    def set_counters(self, step: int, shift: int = 0, pass_: int = 0):
        self._ck(self._L.asd_set_counters(self._h, C.c_int64(step), C.c_int64(shift), C.c_int64(pass_)))

    def launch_count(self) -> int:
        return int(self._L.asd_launch_count(self._h))


def desc_from_workload(w, **over) -> "LatticeDesc":
    """asd_inputs.Workload -> LatticeDesc (argument marshalling only)."""
    d = dict(lattice=w.lattice, nx=w.nx, ny=w.ny, nz=w.nz, pbc=w.pbc, mu_s=w.mu_s, lam=w.lam, gamma=w.gamma,
             dt=w.dt, J=w.J, track_nx=w.track_nx, x0=w.x0, grain_map=w.grain_map, n_grains=w.n_grains,
             grain_ku=w.grain_ku, grain_axis=w.grain_axis, macro=w.macro, seed=w.seed)
    d.update(over)
    return LatticeDesc(**d)


def context_from_workload(w, device: str = "cuda:0", **over) -> "Context":
    """A Context holding the workload's lattice, spins and fields (uploaded from host arrays)."""
    import torch
    ctx = Context(desc_from_workload(w, **over), device=device)
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).to(ctx.device)
    ctx.set_spins(t(w.sx), t(w.sy), t(w.sz))
    ctx.set_fields(t(w.T), t(w.Bx), t(w.By), t(w.Bz))
    torch.cuda.synchronize()
    return ctx
