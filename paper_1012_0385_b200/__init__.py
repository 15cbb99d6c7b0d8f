"""paper_1012_0385_b200 — B200-native (sm_100a) KPZ/ASEP lattice-gas sweep behind a C ABI (include/kpz_b200.h).

    from paper_1012_0385_b200 import KpzSim, LanesSim

The package holds only what the hot path needs: csrc/ (CUDA kernels + C ABI), build.py (nvcc, in-tree) and
binding.py (ctypes marshalling).  There is no CPU fallback.
"""
from .binding import (KPZ2D_PATH_CLUSTER, KPZ_PATH_AUTO, KPZ_PATH_ONCHIP, KPZ_PATH_STREAM, KPZ_PATH_BLOCKED, KpzError, KpzSim, Kpz2dSim, LanesSim, jit_check, kpz2d_jit_check, lanes_crossing_jit_check, lanes_jit_check,
                      kernel_launches, load_library, debug_config, debug_dump_cubins, words_from_numpy, words_to_numpy,
                      noalloc_height_sums, KPZ_NOALLOC_MAX_TILES)

__all__ = ["KpzSim", "Kpz2dSim", "LanesSim", "KpzError", "load_library", "kernel_launches", "debug_config", "debug_dump_cubins", "jit_check", "kpz2d_jit_check", "lanes_jit_check", "lanes_crossing_jit_check", "words_to_numpy", "words_from_numpy",
           "noalloc_height_sums", "KPZ_NOALLOC_MAX_TILES", "KPZ2D_PATH_CLUSTER", "KPZ_PATH_AUTO", "KPZ_PATH_ONCHIP", "KPZ_PATH_STREAM", "KPZ_PATH_BLOCKED"]
