"""Bench-side helper, beside bench.py and outside the product package: what the FP32 FMA pipe of the current device
sustains (bench_probe/libfp32probe.so, built from fp32_probe.cu).  Not part of liblinmin.so or of include/linmin.h;
bench.py reports it next to the derived FP32 peak."""
from __future__ import annotations

import ctypes
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
PROBE_LIB = os.path.join(HERE, "libfp32probe.so")


def build_probe(force: bool = False) -> str:
    src = os.path.join(HERE, "fp32_probe.cu")
    if not force and os.path.exists(PROBE_LIB) and os.path.getmtime(PROBE_LIB) >= os.path.getmtime(src):
        return PROBE_LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    tmp = PROBE_LIB + f".tmp{os.getpid()}"
    subprocess.check_call([nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
                           "-Xcompiler", "-fPIC", "-shared", "-o", tmp, src, "-lcudart"])
    os.replace(tmp, PROBE_LIB)
    return PROBE_LIB


def probe_fp32_peak(stream=None):
    """(FFMA TFLOP/s, FFMA2 TFLOP/s) with register-resident independent FMA chains, 8 CTAs x 256 threads per SM."""
    lib = ctypes.CDLL(build_probe())
    lib.fp32_probe_peak.argtypes = [ctypes.c_void_p, ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_double)]
    a, b = ctypes.c_double(), ctypes.c_double()
    rc = lib.fp32_probe_peak(None if stream is None else ctypes.c_void_p(stream), ctypes.byref(a), ctypes.byref(b))
    if rc != 0:
        raise RuntimeError(f"fp32_probe_peak failed with CUDA error {rc}")
    return a.value, b.value
