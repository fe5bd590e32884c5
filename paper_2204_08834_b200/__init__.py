"""B200-native projection step of the FluTAS two-fluid method (arxiv 2204.08834, sec. 3.3).

`Plan` wraps the C ABI of libflutas_b200.so (include/flutas.h); `workloads` holds the seeded
synthetic inputs.  Importing the package builds (if needed) and loads the CUDA library and
fails loudly if that is impossible: there is no CPU fallback.
"""
from . import workloads  # noqa: F401
from .binding import BC_Z_PERIODIC, BC_Z_WALL, FlutasError, Plan, lib  # noqa: F401
