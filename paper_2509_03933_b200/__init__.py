"""B200-native Pipelined-TDMA hot path (arxiv 2509.03933): batched divide-and-conquer tridiagonal
solve along y of an nx*ny*nz fp64 slab.  The product is ``libtdma.so`` (C ABI in
``include/tdma.h``, hand-written sm_100a kernels under ``csrc/``); this package is its thin
ctypes binding.  See DESIGN.md."""
from .binding import *  # noqa: F401,F403
from .binding import (Plan, TdmaError, load_library, library_path, EXPORTED_SYMBOLS,
                      tdma_options)

__all__ = [n for n in dir() if n.startswith(("tdma_", "TDMA_"))] + [
    "Plan", "TdmaError", "load_library", "library_path", "EXPORTED_SYMBOLS"]
