"""B200-native synthesis hot path of the iterative Neumann-series Marchenko method (arXiv 2106.04649).

`configs` / `gen`  : the seeded synthetic workloads (no method arithmetic).
`binding`          : thin ctypes binding of the C-ABI library `libmk.so` (include/mk.h); argument
                     marshalling only — every step of the path runs in the CUDA kernels.
"""
from . import configs, gen  # noqa: F401

__all__ = ["configs", "gen"]
