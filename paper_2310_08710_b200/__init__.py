"""B200-native Waymax closed-loop step (arXiv 2310.08710): CUDA C-ABI library + thin binding.

The package holds only what the hot path needs: `csrc/` (hand-written sm_100a kernels and
the C-ABI of include/wm.h), `_build.py` (in-tree nvcc build) and `binding.py` (ctypes,
argument marshalling only).  It never imports `oracle/`.
"""
from .binding import *  # noqa: F401,F403
from .binding import load, lib_path, EXPORTS
