"""Pins for the oracle's NEXT-row options against things OTHER than itself: the constraint variants
slo / pos and the renormalised problem with a shared noise covariance
(eq. 5-6).  No GPU, no CUDA code."""
import itertools

import numpy as np
import pytest

import oracle
from paper_1402_2518_b200.synth import make_workload


def rand_library(rng, L, R, corr=0.0):
    base = rng.uniform(0.2, 0.6, size=(L, 1))
    return ((1 - corr) * rng.uniform(0.05, 0.9, size=(L, R)) + corr * base).astype(np.float32)


def objective(A, y, a, Ci=None):
    r = y.astype(np.float64) - A.astype(np.float64) @ a
    return float(r @ r) if Ci is None else float(r @ Ci @ r)


def ls_on_support(AF, y, sum_to_one):
    """numpy library routines only: unconstrained lstsq, or lstsq after eliminating the last coefficient."""
    k = AF.shape[1]
    if not sum_to_one:
        return np.linalg.lstsq(AF, y, rcond=None)[0]
    if k == 1:
        return np.ones(1)
    D = AF[:, :-1] - AF[:, -1:]
    c = np.linalg.lstsq(D, y - AF[:, -1], rcond=None)[0]
    return np.concatenate([c, [1.0 - c.sum()]])


def brute_force(A, y, constraint):
    """Every face of the feasible set: a support F with all members > 0, and (slo) the sum constraint either active
    or not; the smallest objective among the feasible face minimisers is the minimiser (convex QP on a polytope)."""
    A = np.asarray(A, np.float64); y = np.asarray(y, np.float64)
    R = A.shape[1]
    best, best_a = float(y @ y) if constraint != "sto" else np.inf, np.zeros(R)
    for k in range(1, R + 1):
        for F in itertools.combinations(range(R), k):
            cands = []
            if constraint in ("sto", "slo"):
                cands.append(ls_on_support(A[:, F], y, True))
            if constraint in ("pos", "slo"):
                aF = ls_on_support(A[:, F], y, False)
                if constraint == "pos" or aF.sum() <= 1.0:
                    cands.append(aF)
            for aF in cands:
                if (aF < 0).any():
                    continue
                a = np.zeros(R); a[list(F)] = aF
                obj = float(np.sum((y - A @ a) ** 2))
                if obj < best:
                    best, best_a = obj, a
    return best_a, best


def kkt_general(A, y, a, constraint, Ci=None, tol=1e-9):
    """Scaled optimality conditions recomputed in numpy for any constraint option and metric C^-1."""
    A = A.astype(np.float64); y = y.astype(np.float64)
    Ci = np.eye(len(y)) if Ci is None else Ci
    g = A.T @ (Ci @ (A @ a - y))
    F = a > 0
    # scale of g plus its rounding floor (g = 0 exactly when every endmember is active and none constrained)
    gs = np.abs(g).max() + 1e-4 * (np.abs(A).T @ np.abs(Ci @ y)).max()
    assert a.min() >= 0
    if constraint == "sto":
        assert abs(a.sum() - 1) <= 1e-12
        nu = -float(g[F] @ a[F])
    elif constraint == "slo":
        assert a.sum() <= 1 + 1e-12
        nu = -float(g[F] @ a[F]) / a.sum() if (F.any() and a.sum() >= 1 - 1e-12) else 0.0
        assert nu >= -tol * gs                              # multiplier of sum a <= 1
    else:
        nu = 0.0
    assert np.abs((g + nu)[F]).max(initial=0.0) <= tol * gs  # stationarity on the support
    assert (g + nu)[~F].min(initial=0.0) >= -tol * gs        # multipliers of a >= 0
    return nu


# ------------------------------------------------------------------ pos (NNLS)
def test_pos_equals_scipy_nnls_and_brute_force():
    from scipy.optimize import nnls
    rng = np.random.default_rng(1)
    for (L, R, corr) in [(12, 4, 0.0), (20, 7, 0.6), (30, 9, 0.9), (6, 8, 0.3)]:
        A = rand_library(rng, L, R, corr)
        a0 = rng.dirichlet(0.3 * np.ones(R), size=25) * rng.uniform(0.3, 1.7, size=(25, 1))
        Y = (a0 @ A.astype(np.float64).T + 0.02 * rng.standard_normal((25, L))).astype(np.float32)
        Y[3] = -np.abs(Y[3])                                  # a pixel whose answer is a = 0
        res = oracle.solve(A, Y, constraint="pos")
        assert (res.status & 2 == 0).all()
        for p in range(25):
            x, _ = nnls(A.astype(np.float64), Y[p].astype(np.float64), maxiter=10000)
            assert abs(objective(A, Y[p], res.coeffs[p]) - objective(A, Y[p], x)) <= 1e-10 * max(objective(A, Y[p], x), 1e-9)
            if R <= L:
                np.testing.assert_allclose(res.coeffs[p], x, atol=1e-8)
            kkt_general(A, Y[p], res.coeffs[p], "pos")
            assert res.nu[p] == 0.0
            if R <= 8:
                _, obj = brute_force(A, Y[p], "pos")
                assert abs(objective(A, Y[p], res.coeffs[p]) - obj) <= 1e-10 * max(obj, 1e-9)
        assert (res.coeffs[3] == 0).all() and res.support_size[3] == 0


def test_pos_sigma_and_resid():
    """Reading R3 without the sum constraint: J = A_F^+, so homoscedastic sigma gives s sqrt(diag (A_F'A_F)^-1);
    heteroscedastic: sqrt(sum_l J_il^2 s_l^2); finite differences of the solution map agree."""
    rng = np.random.default_rng(2)
    L, R = 24, 6
    A = rand_library(rng, L, R, 0.4)
    a0 = np.array([0.5, 0.0, 0.3, 0.0, 0.2, 0.0])
    y = (A.astype(np.float64) @ a0 + 0.004 * rng.standard_normal(L)).astype(np.float32)
    s = rng.uniform(0.002, 0.01, L).astype(np.float32)
    res = oracle.solve(A, y[None], s[None], constraint="pos")
    F = np.nonzero(res.coeffs[0] > 0)[0]
    assert 2 <= len(F) < R
    AF = A.astype(np.float64)[:, F]
    J = np.linalg.pinv(AF)
    ref = np.zeros(R); ref[F] = np.sqrt((J ** 2) @ (s.astype(np.float64) ** 2))
    np.testing.assert_allclose(res.coeff_sigma[0], ref, rtol=1e-9, atol=1e-14)
    resh = oracle.solve(A, y[None], np.full((1, L), 0.005, np.float32), constraint="pos")
    refh = np.zeros(R); refh[F] = np.float64(np.float32(0.005)) * np.sqrt(np.diag(np.linalg.inv(AF.T @ AF)))
    np.testing.assert_allclose(resh.coeff_sigma[0], refh, rtol=1e-9, atol=1e-14)
    r = y.astype(np.float64) - A.astype(np.float64) @ res.coeffs[0]
    np.testing.assert_allclose(res.resid[0], np.sqrt((r ** 2).mean()), rtol=1e-12)
    h = 2.0 ** -12
    Yp = np.repeat(y[None], L, 0); Ym = Yp.copy()
    for l in range(L):
        Yp[l, l] += np.float32(h); Ym[l, l] -= np.float32(h)
    rp = oracle.solve(A, Yp, constraint="pos"); rm = oracle.solve(A, Ym, constraint="pos")
    step = (Yp.astype(np.float64) - Ym.astype(np.float64))[np.arange(L), np.arange(L)]
    Jfd = ((rp.coeffs - rm.coeffs) / step[:, None]).T
    np.testing.assert_allclose(np.sqrt((Jfd ** 2) @ (s.astype(np.float64) ** 2)), res.coeff_sigma[0], rtol=1e-6, atol=1e-12)


# ------------------------------------------------------------------ slo
def test_slo_brute_force_kkt_and_its_two_regimes():
    from scipy.optimize import nnls
    rng = np.random.default_rng(3)
    n_inactive = n_active = 0
    for (L, R, corr) in [(10, 3, 0.0), (16, 5, 0.5), (24, 8, 0.9), (5, 7, 0.3)]:
        A = rand_library(rng, L, R, corr)
        a0 = rng.dirichlet(0.3 * np.ones(R), size=30) * rng.uniform(0.3, 1.6, size=(30, 1))    # sums below AND above one
        Y = (a0 @ A.astype(np.float64).T + 0.02 * rng.standard_normal((30, L))).astype(np.float32)
        res = oracle.solve(A, Y, constraint="slo")
        sto = oracle.solve(A, Y)
        for p in range(30):
            a = res.coeffs[p]
            _, obj = brute_force(A, Y[p], "slo")
            assert abs(objective(A, Y[p], a) - obj) <= 1e-10 * max(obj, 1e-9)
            nu = kkt_general(A, Y[p], a, "slo")
            x, _ = nnls(A.astype(np.float64), Y[p].astype(np.float64), maxiter=10000)
            if x.sum() < 1 - 1e-9:            # the bound is inactive: slo == NNLS
                n_inactive += 1
                assert abs(objective(A, Y[p], a) - objective(A, Y[p], x)) <= 1e-10 * max(obj, 1e-9)
                assert a.sum() < 1 and abs(res.nu[p]) <= 1e-9 * max(np.abs(res.lam[p]).max(), 1e-30) + 1e-12
            elif a.sum() > 1 - 1e-12:         # the bound is active: slo == sto, with a non-negative multiplier
                n_active += 1
                assert abs(objective(A, Y[p], a) - objective(A, Y[p], sto.coeffs[p])) <= 1e-10 * max(obj, 1e-9)
                assert res.nu[p] >= -1e-9 and abs(res.nu[p] - nu) <= 1e-8 * max(abs(nu), 1e-6)
            assert res.support_size[p] == int((a > 0).sum())
    assert n_inactive > 10 and n_active > 10


# ------------------------------------------------------------------ renormalised problem (eq. 5-6)
def banded_cov(rng, L, smin=0.002, smax=0.01, rho=0.6):
    s = rng.uniform(smin, smax, L)
    idx = np.arange(L)
    C = (rho ** np.abs(idx[:, None] - idx[None, :])) * np.outer(s, s)
    C[np.abs(idx[:, None] - idx[None, :]) > 3] = 0.0            # banded (still positive definite: diagonally dominant enough)
    C += 0.05 * np.diag(s ** 2)
    return C.astype(np.float32)


def paper_whitening(C, A, Y):
    """PAPER.md:79-86 literally, in numpy: C^-1 = L.L^T (lower Cholesky of the inverse), X' = X.L, S' = S.L."""
    Lc = np.linalg.cholesky(np.linalg.inv(C.astype(np.float64)))
    return Lc.T @ A.astype(np.float64), Y.astype(np.float64) @ Lc


@pytest.mark.parametrize("constraint", ["sto", "slo", "pos"])
def test_weighted_equals_brute_force_on_paper_whitened_data(constraint):
    rng = np.random.default_rng(4)
    L, R, N = 14, 5, 20
    A = rand_library(rng, L, R, 0.5)
    C = banded_cov(rng, L)
    a0 = rng.dirichlet(0.4 * np.ones(R), size=N) * (1.0 if constraint == "sto" else rng.uniform(0.4, 1.5, size=(N, 1)))
    Y = (a0 @ A.astype(np.float64).T + rng.multivariate_normal(np.zeros(L), C.astype(np.float64), size=N)).astype(np.float32)
    res = oracle.solve(A, Y, constraint=constraint, cov=C)
    Aw, Yw = paper_whitening(C, A, Y)
    Ci = np.linalg.inv(C.astype(np.float64))
    for p in range(N):
        a, obj = brute_force(Aw, Yw[p], constraint)
        assert abs(objective(A, Y[p], res.coeffs[p], Ci) - obj) <= 1e-9 * max(obj, 1e-9)
        np.testing.assert_allclose(res.coeffs[p], a, atol=1e-8)
        kkt_general(A, Y[p], res.coeffs[p], constraint, Ci)
        r = Y[p].astype(np.float64) - A.astype(np.float64) @ res.coeffs[p]
        np.testing.assert_allclose(res.resid[p], np.sqrt(r @ Ci @ r / L), rtol=1e-9)       # whitened RMS (R17)


def test_weighted_r2_closed_form_and_sigma():
    """R = 2: a_1 = clip(d'C^-1(y - A_2) / d'C^-1 d, 0, 1), sigma_1 = 1/sqrt(d'C^-1 d) inside (0, 1)."""
    rng = np.random.default_rng(5)
    L, N = 12, 100
    A = rand_library(rng, L, 2, 0.3)
    C = banded_cov(rng, L)
    Y = rng.uniform(-0.1, 1.1, size=(N, L)).astype(np.float32)
    res = oracle.solve(A, Y, cov=C)
    A64 = A.astype(np.float64); Ci = np.linalg.inv(C.astype(np.float64))
    d = A64[:, 0] - A64[:, 1]
    t = (Y.astype(np.float64) - A64[:, 1]) @ Ci @ d / (d @ Ci @ d)
    np.testing.assert_allclose(res.coeffs[:, 0], np.clip(t, 0, 1), atol=1e-10)
    inside = (t > 0) & (t < 1)
    assert inside.sum() > 5 and (~inside).sum() > 5
    np.testing.assert_allclose(res.coeff_sigma[inside], 1.0 / np.sqrt(d @ Ci @ d), rtol=1e-9)
    assert (res.coeff_sigma[~inside] == 0).all()


def test_weighted_diagonal_forms_agree_and_reduce_to_row_scaling():
    rng = np.random.default_rng(6)
    w = make_workload("tiny", N=64)
    s = (2.0 ** rng.integers(-9, -6, size=w.L)).astype(np.float32)         # powers of two: y / s is exact in fp32
    r1 = oracle.solve(w.A, w.Y, cov=s)
    r2 = oracle.solve(w.A, w.Y, cov=np.diag(s.astype(np.float64) ** 2).astype(np.float32))
    np.testing.assert_allclose(r1.coeffs, r2.coeffs, atol=1e-12)
    np.testing.assert_allclose(r1.coeff_sigma, r2.coeff_sigma, rtol=1e-10, atol=1e-15)
    r3 = oracle.solve((w.A / s[:, None]).astype(np.float32), (w.Y / s[None, :]).astype(np.float32))      # unweighted, pre-whitened
    np.testing.assert_allclose(r1.coeffs, r3.coeffs, atol=1e-12)
    np.testing.assert_allclose(r1.resid, r3.resid, rtol=1e-12)
    np.testing.assert_allclose(r1.coeff_sigma, r3.coeff_sigma, rtol=1e-10, atol=1e-15)
    # identity covariance == the unweighted problem with sigma == 1
    r4 = oracle.solve(w.A, w.Y, cov=np.ones(w.L, np.float32)); r5 = oracle.solve(w.A, w.Y)
    assert np.array_equal(r4.coeffs, r5.coeffs) and np.array_equal(r4.coeff_sigma, r5.coeff_sigma)


def test_weighted_sigma_is_projected_inverse_hessian_and_monte_carlo():
    """coeff_sigma = sqrt(diag H_w), H_w = K - K11'K/(1'K1), K = (A_F'C^-1 A_F)^-1 (PAPER.md:88 with eq. 6); and the
    std of the coefficients under resampling of CORRELATED noise on an interior construction (support stable)."""
    rng = np.random.default_rng(7)
    w = make_workload("tiny")
    L, R = w.L, w.R
    A64 = w.A.astype(np.float64)
    C = (banded_cov(rng, L, 2e-6, 1e-5)).astype(np.float32)
    Ci = np.linalg.inv(C.astype(np.float64))
    y = A64 @ np.full(R, 1.0 / R)
    lin = oracle.solve(w.A, y.astype(np.float32)[None], cov=C)
    assert lin.support_size[0] == R
    K = np.linalg.inv(A64.T @ Ci @ A64); one = np.ones(R)
    H = K - np.outer(K @ one, one @ K) / (one @ K @ one)
    np.testing.assert_allclose(lin.coeff_sigma[0], np.sqrt(np.diag(H)), rtol=1e-7)
    Yn = (y[None] + rng.multivariate_normal(np.zeros(L), C.astype(np.float64), size=20000)).astype(np.float32)
    mc = oracle.solve(w.A, Yn, cov=C)
    assert (mc.support_size == R).all()
    np.testing.assert_allclose(mc.coeffs.std(0), lin.coeff_sigma[0], rtol=0.02)


def test_weighted_rejects_indefinite_covariance():
    w = make_workload("tiny", N=4)
    C = -np.eye(w.L, dtype=np.float32)
    with pytest.raises(ValueError):
        oracle.solve(w.A, w.Y, cov=C)


@pytest.mark.parametrize("constraint,weighted", [("sto", False), ("pos", False), ("slo", False), ("sto", True), ("slo", True)])
def test_tie_sigma_helper_of_the_parity_checks_agrees_with_the_oracle(constraint, weighted):
    """tests/parity.py::sigma_reference_next is what the GPU's uncertainties are held to on tie pixels (R10).  It is
    written from R3 / R17 with numpy's inverse in coefficient space; the oracle goes through a QR in data space.
    Two routes, one quantity: they must agree on the oracle's own support, for every option."""
    import sys, os
    sys.path.insert(0, os.path.dirname(os.path.abspath(__file__)))
    from parity import sigma_reference_next
    w = make_workload("tiny", N=60)
    rng = np.random.default_rng(5)
    Y = (w.Y * rng.uniform(0.6, 1.1, size=(w.N, 1))).astype(np.float32)          # sums below and at one
    cov = None
    if weighted:
        s = rng.uniform(0.002, 0.01, w.L)
        idx = np.arange(w.L)
        cov = ((0.5 ** np.abs(idx[:, None] - idx[None, :])) * np.outer(s, s)).astype(np.float32)
    ora = oracle.solve(w.A, Y, None if weighted else w.sigma, constraint=constraint, cov=cov)
    Ci = np.linalg.inv(cov.astype(np.float64)) if weighted else None
    A64 = w.A.astype(np.float64)
    seen = set()
    for p in range(w.N):
        a = ora.coeffs[p]
        eq = constraint == "sto" or (constraint == "slo" and a.sum() >= 1 - 1e-9)
        seen.add(eq)
        ref = sigma_reference_next(A64, np.nonzero(a > 0)[0], eq, Ci, None if weighted else w.sigma[p])
        np.testing.assert_allclose(ora.coeff_sigma[p], ref, rtol=1e-6, atol=1e-12)
    if constraint == "slo":
        assert seen == {True, False}
