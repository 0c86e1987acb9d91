"""CPU-side checks of the boundary: libasd.so builds, loads and exports every symbol include/asd.h declares;
host-side validation works without a GPU (no compute calls here)."""
import ctypes as C
import os
import re

import numpy as np

import paper_2502_02236_b200 as asd

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    src = open(os.path.join(ROOT, "include", "asd.h")).read()
    return sorted(set(re.findall(r"ASD_API[^;(]*?\b(asd_\w+)\s*\(", src)))


def test_library_exports_every_declared_symbol():
    L = asd.load_library()
    names = _declared()
    assert len(names) >= 20
    for n in names:
        assert hasattr(L, n), n
    assert sorted(asd.EXPORTED_SYMBOLS) == names


def test_version_and_workspace_bytes_without_gpu():
    assert "sm_100a" in asd.version()
    d = asd.LatticeDesc(asd.ASD_SC, 16, 16, 16, pbc=(1, 1, 1))
    b0 = asd.workspace_bytes(d)
    assert b0 >= 13 * 4096 * 4
    d2 = asd.LatticeDesc(asd.ASD_L10_FE, 881, 220, 27, track_nx=961, macro=(7, 7, 5))
    assert asd.workspace_bytes(d2) >= 13 * 881 * 220 * 27 * 4


def test_host_side_validation():
    bad = [
        asd.LatticeDesc(asd.ASD_SC, 16, 2, 16, pbc=(0, 1, 0)),             # periodic n < 3
        asd.LatticeDesc(7, 4, 4, 4),                                        # unknown lattice
        asd.LatticeDesc(asd.ASD_SC, 4, 4, 4, dt=0.0),
        asd.LatticeDesc(asd.ASD_SC, 4, 4, 4, lam=-0.1),
        asd.LatticeDesc(asd.ASD_SC, 4, 4, 4, track_nx=3),
        asd.LatticeDesc(asd.ASD_SC, 4, 4, 4, grain_map=np.full((4, 4), 5, np.int32), n_grains=2),
        asd.LatticeDesc(asd.ASD_SC, 4, 4, 4, grain_axis=np.array([[0, 0, 2.0]], np.float32)),
        asd.LatticeDesc(asd.ASD_SC, 4, 4, 4, macro=(0, 1, 1)),
        asd.LatticeDesc(asd.ASD_SC, 4, 4, 4, pbc=(1, 0, 0), track_nx=8),
    ]
    for d in bad:
        assert asd.workspace_bytes(d) == 0
    L = asd.load_library()
    assert L.asd_last_error(None)
    # NULL context handling
    assert L.asd_step_heun(None, 1) == 1
    assert L.asd_launch_count(None) == 0


def test_create_without_device_fails_loudly():
    import torch
    if torch.cuda.is_available():
        return
    try:
        asd.Context(asd.LatticeDesc(asd.ASD_SC, 4, 4, 4))
    except RuntimeError as e:
        assert "no CPU fallback" in str(e)
    else:
        raise AssertionError("Context() must fail without a CUDA device")
