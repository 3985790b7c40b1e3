"""B200-native hot path of arXiv 1104.2499: active-Brownian ensemble integration.

The product is the C-ABI library built from `csrc/` (declared in `include/abm.h`); `binding`
is the thin ctypes layer with the same names, `workloads` the seeded synthetic inputs.
"""
from . import workloads  # noqa: F401
