"""B200-native doubly-periodic Stokes mobility product (arXiv 2210.01837): thin Python binding of the C-ABI library.

Every step of the path runs in the CUDA library (``csrc/`` -> ``libdpstokes.so``, declared in ``include/dp.h``);
this package only marshals arguments.  PyTorch is used for device memory and streams, nothing else.
There is no CPU fallback: if the library is missing or no CUDA device is present, calls fail loudly.
"""
from .binding import (BOTTOM_WALL, SLIT, DPError, Plan, bin_particles_static, es_dphi_cut, es_norm, exported_symbols, library_path, load_library,
                      supported_nz)

__all__ = ["BOTTOM_WALL", "SLIT", "DPError", "Plan", "bin_particles_static", "es_dphi_cut", "es_norm", "exported_symbols", "library_path", "load_library",
           "supported_nz"]
