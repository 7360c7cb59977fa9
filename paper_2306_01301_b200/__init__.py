"""paper_2306_01301_b200 -- B200-native kernel-style N-turn nonholonomic planner (arXiv 2306.01301).

Thin ctypes binding over libnhplan.so (include/nhplan.h).  Argument marshalling only: every step of the
path (rendering, sweeps, back-tracking) runs in the CUDA kernels under csrc/.  PyTorch provides device
memory and the stream, nothing else.  There is no CPU fallback: importing `Planner` without the built
library, or constructing one without a CUDA device, raises.
"""
from .binding import (  # noqa: F401
    DEFAULT_CYCLES, FLAG_FIXED_WORK, FLAG_FORWARD_ONLY, FLAG_NO_SHORTCUTS, FLAG_SECTIONS, FLAG_NO_SECTIONS, FLAG_SIMPLE_KERNELS, FLAG_SOFT, INF, MANEUVER_NAMES, NhpError, NOALLOC_MAX_N, Planner, lib_path, load_library, soft_from_hard_noalloc,
)
