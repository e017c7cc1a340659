"""Plain numpy definitions of the detection layer, the library builder and the autofit test -- TEST INFRASTRUCTURE.

NEXT rows 3 and 4 of SURVEY.md 8(f).  Each function is the paper's definition written out (loops and numpy library
routines, fp64); nothing here is shared with the CUDA path (paper_1402_2518_b200/csrc/detect.cuh).

  additional_spectra   PAPER.md:112-114 (sec. 2.5) and :333-339 (appendix: "33 Flat 1, 34 Flat 0.0001, 35 Slope
                       Increasing, 36 Slope Decreasing, 37 cos 1/4, 38 sin 1/4, 39 -cos 1/4, 40 -sin 1/4, 41 cos 1/2,
                       42 sin 1/2, 43 -cos 1/2, 44 -sin 1/2"); "cosine function with periods x2 and x4 of the spectral
                       domain": reading R18 of DESIGN.md -- with x in [0, 1] the position in the spectral domain,
                       "1/4" is a quarter period over the domain (cos(pi x / 2), period = 4 domains) and "1/2" half a
                       period (cos(pi x), period = 2 domains); slopes are x and 1 - x.
  thresholds           PAPER.md:149-153 (eq. 8): C^i = 1/2 (mean(A+) - 2 std(A+) + mean(A-) + 6 std(A-)), A+ / A- the
                       ESTIMATED coefficients of endmember i that are detections (> 0) on the pixels where i is /
                       is not part of the true mixture (Fig. 4: green = positive, red = false detections); reading R19:
                       population std, an empty class contributes 0.
  detect               PAPER.md:239-246: coefficient above the threshold, error on the coefficient below the
                       coefficient, RMS below the noise level.
  second_pass          PAPER.md:294: "a second pass of the LinMin algorithm with the detected spectrum only".
  autofit              PAPER.md:94-100 (eq. 7): S_n = A'.S' + E with S' = S without S_n, unconstrained and under
                       positivity; returns the residues E.
"""
from __future__ import annotations

import numpy as np


def additional_spectra(L: int, n_extra: int, wavelength=None) -> np.ndarray:
    """(L, n_extra) float64, n_extra in {4, 12}, columns in the paper's order 33..44."""
    assert n_extra in (4, 12)
    if wavelength is None:
        x = np.arange(L, dtype=np.float64) / max(L - 1, 1)
    else:
        w = np.asarray(wavelength, dtype=np.float64)
        x = (w - w[0]) / (w[-1] - w[0])
    cols = [np.ones(L), np.full(L, 1e-4), x, 1.0 - x]
    if n_extra == 12:
        for frac in (0.25, 0.5):
            ph = 2.0 * np.pi * frac * x
            cols += [np.cos(ph), np.sin(ph), -np.cos(ph), -np.sin(ph)]
    return np.stack(cols, axis=1)


def thresholds(coeffs: np.ndarray, present: np.ndarray, whole_class: bool = False) -> np.ndarray:
    """eq. 8, one value per endmember.  coeffs (N, R) estimated, present (N, R) bool: i belongs to the true mixture.
    whole_class False (reading R19): A+ / A- are the DETECTIONS (estimate > 0) on present / absent pixels, the green
    and red points of Fig. 4 ("in the case of positive / false detection").  whole_class True (the alternative reading
    of PAPER.md:131, "~30 ... with non-null mixing coefficient (noted A^positive) and ~970 with null mixing coefficient
    (A^false)"): every pixel of each class enters, estimates of exactly 0 included -- what an interior-point iterate
    that never returns an exact 0 would feed eq. 8."""
    coeffs = np.asarray(coeffs, dtype=np.float64)
    present = np.asarray(present, dtype=bool)
    R = coeffs.shape[1]
    out = np.zeros(R)
    for i in range(R):
        counted = np.ones(coeffs.shape[0], dtype=bool) if whole_class else (coeffs[:, i] > 0)
        pos = coeffs[present[:, i] & counted, i]
        neg = coeffs[~present[:, i] & counted, i]
        mp, sp = (pos.mean(), pos.std()) if len(pos) else (0.0, 0.0)
        mf, sf = (neg.mean(), neg.std()) if len(neg) else (0.0, 0.0)
        out[i] = 0.5 * (mp - 2.0 * sp + mf + 6.0 * sf)
    return out


def detect(coeffs, coeff_sigma, resid, thr, rms_max):
    """(mask (N, R) bool, counts (R,)): the three conditions of PAPER.md:241-246, written as loops."""
    N, R = coeffs.shape
    mask = np.zeros((N, R), dtype=bool)
    for p in range(N):
        if not (resid[p] < rms_max):
            continue
        for i in range(R):
            mask[p, i] = (coeffs[p, i] > thr[i]) and (coeff_sigma[p, i] < coeffs[p, i])
    return mask, mask.sum(0)


def second_pass(A, Y, sigma, keep, solve):
    """Re-solve with the columns keep (bool (R,)) only; coefficients of the others are 0.  `solve` is the fp64 oracle."""
    keep = np.asarray(keep, dtype=bool)
    idx = np.nonzero(keep)[0]
    res = solve(np.ascontiguousarray(A[:, idx]), Y, sigma)
    N, R = Y.shape[0], A.shape[1]
    coeffs = np.zeros((N, R)); csig = np.zeros((N, R))
    coeffs[:, idx] = res.coeffs; csig[:, idx] = res.coeff_sigma
    return coeffs, csig, res.resid


def autofit(A, solve_pos):
    """eq. 7 for every endmember n: residues of the best unconstrained (numpy lstsq) and non-negative (`solve_pos`:
    the oracle's pos option, pinned against scipy NNLS) mixture of the OTHER endmembers.  Returns (E_ls, E_nn), (L, R)."""
    A64 = np.asarray(A, dtype=np.float64)
    L, R = A64.shape
    E_ls = np.zeros((L, R)); E_nn = np.zeros((L, R))
    for n in range(R):
        others = [j for j in range(R) if j != n]
        S = A64[:, others]
        c = np.linalg.lstsq(S, A64[:, n], rcond=None)[0]
        E_ls[:, n] = A64[:, n] - S @ c
        a = solve_pos(np.ascontiguousarray(A[:, others]), np.ascontiguousarray(A[:, n][None, :])).coeffs[0]
        E_nn[:, n] = A64[:, n] - S @ a
    return E_ls, E_nn
