"""B200-native fisheye plane-sweeping stereo (arXiv 1809.06132, section III-A) behind the C ABI of include/fsw.h.

The package holds the CUDA sources (csrc/), the in-tree build of libfsw.so (build.py) and the ctypes binding
(binding.py).  Nothing here imports oracle/: the oracle is test infrastructure only.
"""
from .binding import (  # noqa: F401
    DEPTH_RANGE, DEPTH_Z, F32, FILTER_COST, FILTER_RATIO, INDEX_FROM_CROP, INVERSE, LINEAR, REASON_COST_FILTER,
    REASON_MASKED, REASON_NO_PLANE, REASON_OK, REASON_RATIO_FILTER, U8, Context, FswError, PlaneSet, Rig,
    load_library, plan_schedule, version,
)
