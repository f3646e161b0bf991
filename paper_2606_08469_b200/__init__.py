"""paper_2606_08469_b200 — OctaOctree radiance-cache query for NVIDIA B200 (sm_100a).

A thin ctypes binding over ``liboo.so`` (the C ABI of ``include/oo.h``).  PyTorch is used for device memory and streams
only; every step of the path runs in the library's CUDA kernels.  There is no CPU fallback: without the built library
or without a B200 the calls raise.
"""
from .binding import (OOError, OctaOctree, lib_path, load_library, PATH_AUTO, PATH_GENERIC, PATH_UNFUSED,  # noqa: F401
                      PATH_FUSED_MMA, PATH_FUSED_TC, PATH_FUSED_TC_TMEM, PATH_FULL, EXPORTED_SYMBOLS,
                      oo_sort_queries_static, SORT_STATIC_MAX_QUERIES)
