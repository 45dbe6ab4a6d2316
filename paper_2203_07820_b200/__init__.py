"""B200-native Chebyshev-filter hot path of DFT-FE (arxiv 2203.07820): thin Python binding of libchfsi.

Everything on the path runs in the CUDA kernels behind the C ABI of `include/chfsi.h`; this module only
marshals arguments (ctypes) and uses PyTorch for device memory and streams.  There is no CPU fallback: the
import works without a GPU (so the symbols can be checked), any compute call without one raises.
"""
from .binding import (ChfsiError, Operator, lib, load_library, measure_fp64_peak, mesh_mass, EXPORTED_SYMBOLS)  # noqa: F401

__all__ = ["ChfsiError", "Operator", "lib", "load_library", "measure_fp64_peak", "mesh_mass", "EXPORTED_SYMBOLS"]
