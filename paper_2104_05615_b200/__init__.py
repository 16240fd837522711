"""paper_2104_05615_b200 -- B200-native (sm_100a) hot path of MSPCG for Moebius domain-wall fermions (arXiv 2104.05615).

The product is the CUDA library behind include/mspcg.h (csrc/ -> libmspcg.so); `binding` is a thin ctypes layer over
it and `synth` makes the seeded synthetic inputs shared with the CPU oracle (which lives in /oracle and is test
infrastructure only).
"""
from . import synth  # noqa: F401
from .binding import (F16, F32, F64, LAYOUT_ABI, LAYOUT_NATIVE, Mspcg, MspcgError, dot2_noalloc, load_library)  # noqa: F401
