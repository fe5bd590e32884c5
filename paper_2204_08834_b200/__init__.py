"""B200-native projection step of the FluTAS two-fluid method (arxiv 2204.08834, sec. 3.3).

`Plan` wraps the C ABI of libflutas_b200.so (include/flutas.h).  Importing the package builds
(if needed) and loads the CUDA library and fails loudly if that is impossible: there is no CPU
fallback.  The seeded synthetic inputs live in the top-level module `workloads` (they also feed the
tests' CPU checker, so they are not part of this package).
"""
from .binding import (BC_Z_PERIODIC, BC_Z_WALL, FlutasError, Plan, lib,  # noqa: F401
                      vof_noalloc_max_cells, vof_step_noalloc)
