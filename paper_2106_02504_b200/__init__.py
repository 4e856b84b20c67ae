"""B200-native RANLUX++ stream generation (arxiv 2106.02504): CUDA kernels + C ABI
(csrc/, include/rlxpp.h) and a thin ctypes binding with the same names (binding.py).
The shared library is loaded on first use; nothing here computes on the CPU."""
from .binding import *  # noqa: F401,F403
from .binding import EXPORTS, LIB_PATH, Handle, RlxppError, load  # noqa: F401
