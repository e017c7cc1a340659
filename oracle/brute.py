"""Brute-force pin for the oracle (tiny R only) -- TEST INFRASTRUCTURE.

PAPER.md:57 (sec. 2.1) describes the exhaustive alternative the constrained solvers replace:
"test all combination of reference spectra S in order to keep only positive case".  For a convex
quadratic over the simplex the minimiser restricted to its own support solves the
equality-constrained least squares on that support, so enumerating every non-empty support
(2^R - 1), solving min ||y - A_F a_F|| s.t. 1'a_F = 1 with a library routine (numpy lstsq on the
null-space parametrisation), discarding supports whose solution has a negative entry and keeping
the smallest objective yields the minimiser of eq. 2 under eq. 3-4 by definition.
"""
from __future__ import annotations

import itertools

import numpy as np


def eq_constrained_ls(AF: np.ndarray, y: np.ndarray) -> np.ndarray:
    """min ||y - AF a|| s.t. sum(a) = 1, by eliminating the last coefficient (a library lstsq)."""
    k = AF.shape[1]
    if k == 1:
        return np.ones(1)
    D = AF[:, :-1] - AF[:, -1:]
    c, *_ = np.linalg.lstsq(D, y - AF[:, -1], rcond=None)
    return np.concatenate([c, [1.0 - c.sum()]])


def brute_force_fcls(A: np.ndarray, y: np.ndarray):
    """Returns (a, objective) over all supports.  A (L,R), y (L,), float64.  R <= ~12."""
    A = np.asarray(A, dtype=np.float64)
    y = np.asarray(y, dtype=np.float64)
    R = A.shape[1]
    best, best_a = np.inf, None
    for k in range(1, R + 1):
        for F in itertools.combinations(range(R), k):
            aF = eq_constrained_ls(A[:, F], y)
            if (aF < 0).any():
                continue
            a = np.zeros(R)
            a[list(F)] = aF
            obj = float(np.sum((y - A @ a) ** 2))
            if obj < best:
                best, best_a = obj, a
    return best_a, best
