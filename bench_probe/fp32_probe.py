"""Bench-side helper: what the FP32 FMA pipe of the current device sustains (libfp32probe.so, built from
csrc/fp32_probe.cu).  Not part of the product ABI; bench.py reports it next to the derived FP32 peak."""
from __future__ import annotations

import ctypes

from . import build


def probe_fp32_peak(stream=None):
    """(FFMA TFLOP/s, FFMA2 TFLOP/s) with register-resident independent FMA chains, 8 CTAs x 256 threads per SM."""
    lib = ctypes.CDLL(build.build_probe())
    lib.fp32_probe_peak.argtypes = [ctypes.c_void_p, ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_double)]
    a, b = ctypes.c_double(), ctypes.c_double()
    rc = lib.fp32_probe_peak(None if stream is None else ctypes.c_void_p(stream), ctypes.byref(a), ctypes.byref(b))
    if rc != 0:
        raise RuntimeError(f"fp32_probe_peak failed with CUDA error {rc}")
    return a.value, b.value
