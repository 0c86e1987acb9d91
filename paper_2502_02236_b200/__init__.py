"""paper_2502_02236_b200 -- B200-native atomistic spin dynamics (the ASD window of arXiv 2502.02236).

The product is libasd.so (include/asd.h): hand-written CUDA kernels for sm_100a behind a C ABI.
This package is only the thin Python binding over it (ctypes; torch for device memory and streams).
There is no CPU path: importing works anywhere, creating a context needs a CUDA device and the built library.
"""
from .binding import (  # noqa: F401
    ASD_SC, ASD_L10_FE, AsdError, Context, LatticeDesc, lib_path, load_library, version, workspace_bytes,
    EXPORTED_SYMBOLS, KERNEL_AUTO, KERNEL_GENERAL, KERNEL_FAST, KERNEL_TMA, KERNEL_FUSED, KERNEL_PERSISTENT, GRAPH_AUTO, GRAPH_OFF, GRAPH_ON,
    desc_from_workload, context_from_workload, spin_sum_noalloc, NOALLOC_MAX_COUNT,
)
