"""ctypes wrapper around oracle/linmin_oracle.c (plain C, fp64, OpenMP over pixels).

TEST INFRASTRUCTURE: see oracle/__init__.py for who may call this.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from dataclasses import dataclass
from typing import Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "linmin_oracle.c")
_LIB = os.path.join(_HERE, "liblinmin_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (-O2, OpenMP).  Called by __graft_entry__.build() and lazily here."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".tmp{os.getpid()}"
        subprocess.check_call(["gcc", "-O2", "-std=c11", "-fPIC", "-shared", "-fopenmp",
                               "-Wall", "-Wextra", "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        f = lib.linmin_oracle_solve
        P = ctypes.c_void_p
        f.argtypes = [P, P, P, ctypes.c_int64, ctypes.c_int32, ctypes.c_int32, ctypes.c_int64,
                      ctypes.c_int64, P, P, P, P, P, P, P, P, P, ctypes.c_int32]
        f.restype = ctypes.c_int
        fx = lib.linmin_oracle_solve_ex
        fx.argtypes = [P, P, P, ctypes.c_int64, ctypes.c_int32, ctypes.c_int32, ctypes.c_int64,
                       ctypes.c_int64, ctypes.c_int32, P, ctypes.c_int32, P, P, P, P, P, P, P, P, P, ctypes.c_int32]
        fx.restype = ctypes.c_int
        lib.linmin_oracle_max_threads.restype = ctypes.c_int
        _lib = lib
    return _lib


def max_threads() -> int:
    return int(_load().linmin_oracle_max_threads())


@dataclass
class OracleResult:
    coeffs: np.ndarray        # (N, R) float64, minimiser of eq. 2 under eq. 3-4
    coeff_sigma: np.ndarray   # (N, R) float64, reading R3
    resid: np.ndarray         # (N,)  float64 RMS, reading R8
    lam: np.ndarray           # (N, R) multipliers of a >= 0 (scale of g = A'(Aa - y))
    nu: np.ndarray            # (N,)
    support_size: np.ndarray  # (N,) int32
    steps: np.ndarray         # (N,) int32 active-set steps
    rank_margin: np.ndarray   # (N,) smallest |R_jj| of the final QR of A_F Z
    status: np.ndarray        # (N,) int32: 1 rank-deficient index rejected, 2 step cap, 4 non-finite


def _ptr(a: Optional[np.ndarray]):
    return None if a is None else a.ctypes.data_as(ctypes.c_void_p)


CONSTRAINTS = {"sto": 0, "slo": 1, "pos": 2}


def solve(A: np.ndarray, Y: np.ndarray, sigma: Optional[np.ndarray] = None,
          nthreads: int = 0, constraint: str = "sto", cov: Optional[np.ndarray] = None) -> OracleResult:
    """A (L,R) float32, Y (N,L) float32, sigma None | (L,) | (N,L) float32.
    constraint: "sto" (eq. 3 + 4), "slo" (sum lower than one), "pos" (eq. 3 only) -- PAPER.md:35, 157, 221.
    cov: None (unweighted fit, eq. 2), (L,) per-channel noise std of a diagonal covariance, or (L,L) covariance
    matrix: the renormalised problem of PAPER.md:77-86 (eq. 5-6); sigma is then ignored."""
    A = np.ascontiguousarray(A, dtype=np.float32)
    Y = np.ascontiguousarray(Y, dtype=np.float32)
    L, R = A.shape
    N = Y.shape[0]
    assert Y.ndim == 2 and Y.shape[1] == L
    stride = 0
    if sigma is not None:
        sigma = np.ascontiguousarray(sigma, dtype=np.float32)
        if sigma.ndim == 2:
            assert sigma.shape == (N, L)
            stride = L
        else:
            assert sigma.shape == (L,)
    out = OracleResult(np.empty((N, R)), np.empty((N, R)), np.empty(N), np.empty((N, R)),
                       np.empty(N), np.empty(N, np.int32), np.empty(N, np.int32), np.empty(N),
                       np.empty(N, np.int32))
    cov_kind = 0
    if cov is not None:
        cov = np.ascontiguousarray(cov, dtype=np.float32)
        if cov.ndim == 1:
            assert cov.shape == (L,)
            cov_kind = 1
        else:
            assert cov.shape == (L, L)
            cov_kind = 2
    rc = _load().linmin_oracle_solve_ex(_ptr(A), _ptr(Y), _ptr(sigma), N, L, R, L, stride,
                                        CONSTRAINTS[constraint], _ptr(cov), cov_kind,
                                        _ptr(out.coeffs), _ptr(out.coeff_sigma), _ptr(out.resid),
                                        _ptr(out.lam), _ptr(out.nu), _ptr(out.support_size),
                                        _ptr(out.steps), _ptr(out.rank_margin), _ptr(out.status),
                                        int(nthreads))
    if rc == -2:
        raise ValueError("covariance is not positive definite")
    if rc != 0:
        raise RuntimeError(f"linmin_oracle_solve failed with code {rc}")
    if (out.status & 2).any():
        raise RuntimeError("oracle hit its step cap on %d pixels" % int((out.status & 2 != 0).sum()))
    return out
