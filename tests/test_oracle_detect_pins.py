"""Pins for oracle/detect.py (NEXT rows 3-4 of SURVEY.md 8(f)) against things other than itself.  No GPU."""
import os

import numpy as np

import oracle
from oracle import detect as D
from paper_1402_2518_b200.synth import make_workload

HERE = os.path.dirname(os.path.abspath(__file__))


def test_eq8_hand_worked_golden():
    rows = np.loadtxt(os.path.join(HERE, "golden", "eq8_hand_worked.txt"))
    data, expected = rows[rows[:, 1] >= 0], rows[rows[:, 1] < 0][0, 0]
    thr = D.thresholds(data[:, :1], data[:, 1:2] > 0.5)
    np.testing.assert_allclose(thr[0], expected, rtol=1e-14)


def test_eq8_whole_class_hand_worked_golden():
    """The alternative reading of PAPER.md:131 (every pixel of a class, exact zeros included): its own hand-worked
    value on the same eight pixels, and it differs from reading R19's."""
    rows = np.loadtxt(os.path.join(HERE, "golden", "eq8_whole_class_hand_worked.txt"))
    data, expected = rows[rows[:, 1] >= 0], rows[rows[:, 1] < 0][0, 0]
    thr = D.thresholds(data[:, :1], data[:, 1:2] > 0.5, whole_class=True)
    np.testing.assert_allclose(thr[0], expected, rtol=1e-14)
    assert abs(D.thresholds(data[:, :1], data[:, 1:2] > 0.5)[0] - expected) > 0.1
    # an estimator that never returns an exact zero (the paper's interior-point iterate): both readings coincide
    rng = np.random.default_rng(3)
    c = rng.uniform(1e-6, 0.5, (200, 3)); present = rng.uniform(size=(200, 3)) < 0.2
    np.testing.assert_allclose(D.thresholds(c, present, whole_class=True), D.thresholds(c, present), rtol=1e-14)


def test_detect_hand_worked_golden():
    """each of the three conditions alone flips the entries the file says (derivation in the file);
    a swapped comparison, a non-strict one, a shared threshold or a wrong broadcast of the RMS fails a row."""
    rows = np.loadtxt(os.path.join(HERE, "golden", "detect_hand_worked.txt"))
    par, data = rows[rows[:, 6] < 0][0], rows[rows[:, 6] >= 0]
    thr, rms_max = par[:2], par[2]
    mask, counts = D.detect(data[:, 0:2], data[:, 2:4], data[:, 4], thr, rms_max)
    expected = data[:, 5:7] > 0.5
    assert data.shape[0] == 11 and mask.shape == (11, 2)
    assert np.array_equal(mask, expected), np.nonzero(mask != expected)
    assert np.array_equal(counts, expected.sum(0)) and list(counts) == [6, 5]


def test_eq8_against_a_vectorised_restatement_and_edge_cases():
    rng = np.random.default_rng(0)
    N, R = 500, 6
    present = rng.uniform(size=(N, R)) < 0.3
    coeffs = np.where(present, rng.uniform(0.05, 0.6, (N, R)), rng.uniform(0, 0.05, (N, R)))
    coeffs[rng.uniform(size=(N, R)) < 0.4] = 0.0
    present[:, 4] = False                      # an endmember that is never present
    coeffs[:, 5] = 0.0                         # an endmember that is never detected
    thr = D.thresholds(coeffs, present)
    for i in range(R):
        det = coeffs[:, i] > 0
        a, b = coeffs[det & present[:, i], i], coeffs[det & ~present[:, i], i]
        ma, sa = (a.mean(), np.sqrt(((a - a.mean()) ** 2).mean())) if a.size else (0, 0)
        mb, sb = (b.mean(), np.sqrt(((b - b.mean()) ** 2).mean())) if b.size else (0, 0)
        np.testing.assert_allclose(thr[i], 0.5 * (ma - 2 * sa + mb + 6 * sb), rtol=1e-13, atol=1e-15)
    assert thr[5] == 0.0


def test_additional_spectra_properties():
    """PAPER.md:112-114, 333-339.  Flat 1 = 1; the two slopes add up to Flat 1 (the linear dependence the paper says the
    constraints remove); +/- pairs cancel; cos^2 + sin^2 = 1; "1/4" runs over a quarter period (cos: 1 -> 0, sin: 0 -> 1),
    "1/2" over half a period (cos: 1 -> -1, sin: 0 -> 1 -> 0); with a wavelength grid the position is the normalised
    wavelength; under positivity and sum-to-one the linearly DEPENDENT extended library still has a unique answer."""
    L = 41
    E = D.additional_spectra(L, 12)
    assert E.shape == (L, 12)
    assert (E[:, 0] == 1).all() and (E[:, 1] == 1e-4).all()
    np.testing.assert_allclose(E[:, 2] + E[:, 3], 1.0, atol=1e-15)
    assert E[0, 2] == 0 and E[-1, 2] == 1 and (np.diff(E[:, 2]) > 0).all()
    for c0 in (4, 8):
        np.testing.assert_allclose(E[:, c0] + E[:, c0 + 2], 0, atol=1e-15)
        np.testing.assert_allclose(E[:, c0 + 1] + E[:, c0 + 3], 0, atol=1e-15)
        np.testing.assert_allclose(E[:, c0] ** 2 + E[:, c0 + 1] ** 2, 1.0, atol=1e-14)
    np.testing.assert_allclose([E[0, 4], E[-1, 4], E[0, 5], E[-1, 5]], [1, 0, 0, 1], atol=1e-15)
    np.testing.assert_allclose([E[0, 8], E[-1, 8], E[L // 2, 9], E[-1, 9]], [1, -1, 1, 0], atol=1e-15)
    assert np.array_equal(D.additional_spectra(L, 4), E[:, :4])
    wl = np.linspace(0.95, 2.5, L) ** 1.3
    Ew = D.additional_spectra(L, 4, wl)
    np.testing.assert_allclose(Ew[:, 2], (wl - wl[0]) / (wl[-1] - wl[0]), atol=1e-15)
    w = make_workload("tiny", N=20)
    lib = np.concatenate([w.A[:, :6], D.additional_spectra(w.L, 4)], axis=1).astype(np.float32)
    # Flat 1 = Slope up + Slope down = 1e4 x Flat 0.0001: the four additional spectra span only two dimensions
    assert np.linalg.matrix_rank(lib.astype(np.float64), tol=1e-6) == lib.shape[1] - 2
    res = oracle.solve(lib, w.Y)
    sing = np.linalg.svd(lib.astype(np.float64), compute_uv=False)
    assert (res.rank_margin > 1e-6 * sing[0]).all()


def test_detect_conditions_and_second_pass_and_autofit():
    from scipy.optimize import nnls
    w = make_workload("tiny", N=300)
    res = oracle.solve(w.A, w.Y, w.sigma)
    thr = D.thresholds(res.coeffs, w.a0 > 0)
    mask, counts = D.detect(res.coeffs, res.coeff_sigma, res.resid, thr, rms_max=0.006)
    ref = (res.coeffs > thr[None]) & (res.coeff_sigma < res.coeffs) & (res.resid < 0.006)[:, None]      # vectorised restatement
    assert np.array_equal(mask, ref) and np.array_equal(counts, ref.sum(0))
    assert 0 < mask.sum() < mask.size
    # second pass: the same answer as solving with the sub-library directly, zeros elsewhere
    keep = counts >= 5
    keep[-2:] = True
    c2, s2, r2 = D.second_pass(w.A, w.Y, w.sigma, keep, oracle.solve)
    direct = oracle.solve(np.ascontiguousarray(w.A[:, keep]), w.Y, w.sigma)
    assert np.array_equal(c2[:, keep], direct.coeffs) and (c2[:, ~keep] == 0).all() and np.array_equal(r2, direct.resid)
    # autofit (eq. 7): residues orthogonal to the other endmembers (unconstrained), equal to scipy NNLS (positivity),
    # and never smaller under positivity ("The unconstrained problem shows smaller residues")
    E_ls, E_nn = D.autofit(w.A, lambda A, Y: oracle.solve(A, Y, constraint="pos"))
    A64 = w.A.astype(np.float64)
    for n in range(w.R):
        others = [j for j in range(w.R) if j != n]
        np.testing.assert_allclose(A64[:, others].T @ E_ls[:, n], 0, atol=1e-10)
        x, rn = nnls(A64[:, others], A64[:, n], maxiter=10000)
        np.testing.assert_allclose(np.linalg.norm(E_nn[:, n]), rn, rtol=1e-9)
        assert np.linalg.norm(E_nn[:, n]) >= np.linalg.norm(E_ls[:, n]) - 1e-12
