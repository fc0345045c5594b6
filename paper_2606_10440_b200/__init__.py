"""B200-native cycle-synchronous cache-line collective simulator (hot path of ASTRA-sim 3.0,
arxiv/paper_2606_10440).  The product is the CUDA engine in csrc/ behind the C-ABI of
include/astra.h; this package is the thin Python binding (argument marshalling only).

There is no CPU fallback: `Engine(...)` raises when the CUDA library or a device is missing.
"""
from .binding import (AstraError, Engine, Summary, load_library, simulate_workload,
                      EXPORTED_SYMBOLS)

__all__ = ["AstraError", "Engine", "Summary", "load_library", "simulate_workload", "EXPORTED_SYMBOLS"]
