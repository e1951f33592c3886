"""spegg-b200: the per-time-step update of sPEGG (arXiv 1603.09255) as hand-written sm_100a CUDA
behind a small C ABI (include/spegg.h).  `binding` is the ctypes layer, `workloads` the seeded
synthetic configurations, `build` compiles libspegg.so in-tree."""
from . import workloads  # noqa: F401
