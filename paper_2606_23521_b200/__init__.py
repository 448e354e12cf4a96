"""Concordia delta-checkpoint hot path for NVIDIA B200 (sm_100a).

CUDA kernels + C ABI: csrc/ and include/concordia.h.  This package is the thin Python binding.
It never imports oracle/ (the CPU oracle is test infrastructure) and has no CPU fallback.
"""
from .binding import *  # noqa: F401,F403
from .binding import Context, Result, load_library, lib_path, dirty_pages_static, EXPORTS  # noqa: F401
