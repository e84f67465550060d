"""paper_2110_12749_b200 — B200-native two-stage subband incoherent dedispersion.

The product is ``libgsp.so`` (hand-written CUDA for sm_100a behind the C ABI of
``include/gsp.h``).  This package is the thin Python binding with the same names:
argument marshalling only; every step of the path runs in the library's kernels.
PyTorch is used by callers for device memory and streams, nothing else.

There is no CPU fallback.  Importing works without a GPU (so the ABI can be
checked), but creating a plan without a CUDA device raises ``GspError``.
"""
from .binding import (  # noqa: F401
    GSP_F32,
    GSP_IMPL_AUTO,
    GSP_IMPL_GENERIC,
    GSP_IMPL_TILED,
    GSP_IMPL_WINDOWED,
    GSP_U8,
    GspError,
    Plan,
    Search,
    declared_symbols,
    dedisperse_multi,
    dedisperse_multi_launches,
    dedisperse_static,
    static_workspace_bytes,
    delay_tables,
    lib,
    library_path,
)

__all__ = ["Plan", "Search", "GspError", "lib", "library_path", "declared_symbols", "delay_tables", "dedisperse_multi", "dedisperse_multi_launches", "dedisperse_static", "static_workspace_bytes", "GSP_U8", "GSP_F32",
           "GSP_IMPL_AUTO", "GSP_IMPL_GENERIC", "GSP_IMPL_TILED", "GSP_IMPL_WINDOWED"]
