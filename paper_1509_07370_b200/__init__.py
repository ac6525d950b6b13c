"""bh-b200: Barnes-Hut potential of AMR cells as point masses on one B200 (arXiv 1509.07370's hot path).

Thin ctypes binding of the C ABI in include/bh.h -- argument marshalling only; every step of the path
(keys, sort, permute, topology, moments, walk, scatter, direct sum) runs in the CUDA kernels of
libbh.so.  PyTorch supplies device memory and the stream.  There is no CPU fallback: if libbh.so is
missing it is built with nvcc, and if that fails the import of `Context` users fails loudly.
"""
from .binding import (BH_MAC_BARNES94, BH_MAC_BH86, BHError, Context, Stats, lib, lib_path,  # noqa: F401
                      EXPORTED_SYMBOLS, NOALLOC_MAX_N, direct_noalloc)

__all__ = ["Context", "Stats", "BHError", "BH_MAC_BH86", "BH_MAC_BARNES94", "lib", "lib_path", "EXPORTED_SYMBOLS",
           "direct_noalloc", "NOALLOC_MAX_N"]
