"""B200-native octahedron-KPZ hot path (Kelling & Odor, arXiv:1110.6745): thin Python binding of libkpz_b200.so.

The product is the CUDA library behind include/kpz.h; this package only marshals arguments (ctypes) and uses
PyTorch for device memory and streams.  There is no CPU fallback: importing works anywhere, but creating a
lattice without the compiled extension or without a CUDA device raises.
"""
from .binding import (KPZ, KpzError, load_library, workspace_bytes, philox_selftest, measure_peaks, measure_layouts, overlap_plan, exported_symbols,
                      KPZ_OK, KPZ_EINVAL, KPZ_ENOMEM, KPZ_ECUDA, KPZ_EOVERFLOW, KPZ_ESTATE)

__all__ = ["KPZ", "KpzError", "load_library", "workspace_bytes", "philox_selftest", "measure_peaks", "measure_layouts", "overlap_plan", "exported_symbols",
           "KPZ_OK", "KPZ_EINVAL", "KPZ_ENOMEM", "KPZ_ECUDA", "KPZ_EOVERFLOW", "KPZ_ESTATE"]
