"""CPU oracle for the sPEGG per-time-step update -- TEST INFRASTRUCTURE ONLY.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  It is a ctypes wrapper around
``oracle/spegg_oracle.cpp`` (plain single-threaded C++, see that file's header for the
PAPER.md citations and the pins).  It imports nothing from the CUDA package
``paper_1603_09255_b200`` and shares no code with it.
"""
from .binding import (  # noqa: F401
    Oracle,
    build,
    draw,
    exp_neg64,
    expf_spec,
    lib,
    normal_delta,
    normal_table,
    philox4x32_10,
    poisson_count,
    poisson_table,
)
