"""Bench-only probe (libfsw_probe.so, csrc/probe_fp32_peak.cu): the FP32 FMA rate of the device, which bench.py uses
as the denominator of the "alu" roofline.  Not part of the library's ABI (include/fsw.h)."""
from __future__ import annotations

import ctypes
import os

_HERE = os.path.dirname(os.path.abspath(__file__))
PROBE_PATH = os.path.join(_HERE, "libfsw_probe.so")


def measure_fp32_peak(device=0):
    """(TFLOP/s, ms) of an FFMA-chain kernel timed with CUDA events on torch's current stream of `device`."""
    import torch
    if not os.path.exists(PROBE_PATH):
        from . import build as _build
        _build.build()
    L = ctypes.CDLL(PROBE_PATH)
    L.fsw_probe_fp32_peak.argtypes = [ctypes.c_int32, ctypes.c_void_p, ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_double)]
    L.fsw_probe_fp32_peak.restype = ctypes.c_int32
    t, ms = ctypes.c_double(), ctypes.c_double()
    rc = L.fsw_probe_fp32_peak(int(device), torch.cuda.current_stream(device).cuda_stream, ctypes.byref(t), ctypes.byref(ms))
    if rc != 0:
        raise RuntimeError("fsw_probe_fp32_peak failed with cudaError %d" % rc)
    return t.value, ms.value
