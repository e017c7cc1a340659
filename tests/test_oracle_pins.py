"""Pins for the CPU oracle (oracle/linmin_oracle.c) against things OTHER than itself.

Each test names the passage of /root/reference/PAPER.md that fixes the expected value:
eq. 2 (line 54), eq. 3 (line 63), eq. 4 (line 68), the closed forms of sec. 2.1-2.2 (lines 57, 71),
and readings R3/R4/R8 of DESIGN.md for PAPER.md:88 and :143.  No GPU, no CUDA code.
"""
import os

import numpy as np
import pytest

import oracle
from oracle.brute import brute_force_fcls
from paper_1402_2518_b200.synth import make_workload

HERE = os.path.dirname(os.path.abspath(__file__))


def rand_library(rng, L, R, corr=0.0):
    """Positive random library; corr in [0,1) mixes a common smooth component in (correlated spectra)."""
    base = rng.uniform(0.2, 0.6, size=(L, 1))
    A = (1 - corr) * rng.uniform(0.05, 0.9, size=(L, R)) + corr * base
    return A.astype(np.float32)


def simplex_points(rng, n, R, alpha=0.5):
    return rng.dirichlet(alpha * np.ones(R), size=n)


def objective(A, y, a):
    r = y.astype(np.float64) - A.astype(np.float64) @ a
    return float(r @ r)


def kkt(A, y, a):
    """Scaled KKT residuals (R11) recomputed in numpy from the coefficients alone."""
    A = A.astype(np.float64); y = y.astype(np.float64)
    g = A.T @ (A @ a - y)
    F = a > 0
    nu = -float(g[F] @ a[F])
    lam = np.where(F, 0.0, g + nu)
    gs = max(np.abs(g).max(), 1e-300)
    return dict(sum=abs(a.sum() - 1.0), neg=float(max(0.0, -a.min())),
                lam_neg=float(max(0.0, -lam.min())) / gs,
                comp=float(np.max(a * np.abs(np.where(F, g + nu, 0.0)))) / gs,
                stat=float(np.abs((g + nu)[F]).max()) / gs)


def assert_kkt(A, Y, coeffs, tol=1e-9):
    for p in range(Y.shape[0]):
        k = kkt(A, Y[p], coeffs[p])
        assert k["sum"] <= 1e-12, (p, k)
        assert k["neg"] == 0.0, (p, k)
        assert k["lam_neg"] <= tol, (p, k)
        assert k["comp"] <= tol, (p, k)
        assert k["stat"] <= tol, (p, k)


# ---------------------------------------------------------------- golden, hand-worked
def test_hand_worked_golden():
    rows = np.loadtxt(os.path.join(HERE, "golden", "hand_worked.txt"))
    A = np.eye(2, dtype=np.float32)
    for row in rows:
        y = row[0:2].astype(np.float32)[None, :]
        s = row[2:4].astype(np.float32)[None, :]
        r = oracle.solve(A, y, s)
        np.testing.assert_allclose(r.coeffs[0], row[4:6], atol=1e-7)
        np.testing.assert_allclose(r.coeff_sigma[0], row[6:8], atol=1e-7)
        np.testing.assert_allclose(r.resid[0], row[8], atol=1e-7)


# ---------------------------------------------------------------- brute force
@pytest.mark.parametrize("R,L,corr", [(2, 5, 0.0), (3, 7, 0.5), (5, 12, 0.9), (8, 20, 0.97), (7, 6, 0.5)])
def test_brute_force_random(R, L, corr):
    rng = np.random.default_rng(100 + R)
    A = rand_library(rng, L, R, corr)
    a0 = simplex_points(rng, 30, R, 0.3)
    Y = (a0 @ A.astype(np.float64).T + 0.02 * rng.standard_normal((30, L))).astype(np.float32)
    res = oracle.solve(A, Y)
    for p in range(Y.shape[0]):
        a, obj = brute_force_fcls(A, Y[p])
        assert abs(objective(A, Y[p], res.coeffs[p]) - obj) <= 1e-12 * max(obj, 1e-12)
        if R <= L:     # unique minimiser
            np.testing.assert_allclose(res.coeffs[p], a, atol=1e-9)


def test_brute_force_tiny_config(tiny):
    res = oracle.solve(tiny.A, tiny.Y[:60], tiny.sigma[:60])
    for p in range(60):
        a, obj = brute_force_fcls(tiny.A, tiny.Y[p])
        np.testing.assert_allclose(res.coeffs[p], a, atol=1e-11)
        assert res.support_size[p] == int((a > 0).sum())


# ---------------------------------------------------------------- KKT (R11)
@pytest.mark.parametrize("name,n", [("tiny", 1000), ("omega", 1500), ("crism", 400), ("stress", 100)])
def test_kkt_on_configs(name, n):
    w = make_workload(name, N=n)
    res = oracle.solve(w.A, w.Y, w.sigma)
    assert (res.status == 0).all()
    assert_kkt(w.A, w.Y, res.coeffs)
    # the oracle's own multipliers agree with the recomputed ones
    p = 0
    A = w.A.astype(np.float64)
    g = A.T @ (A @ res.coeffs[p] - w.Y[p])
    np.testing.assert_allclose(res.lam[p], np.where(res.coeffs[p] > 0, 0, g + res.nu[p]), atol=1e-9)


# ---------------------------------------------------------------- noiseless recovery
def test_noiseless_recovery_exact_inputs():
    """y = A a0 exactly representable in fp32 -> a* = a0 and F* = 0 (full column rank)."""
    rng = np.random.default_rng(7)
    L, R, N = 24, 10, 50
    A = (rng.integers(1, 1024, size=(L, R)) / 1024.0).astype(np.float32)
    a0 = np.zeros((N, R))
    for p in range(N):
        k = rng.integers(1, 5)
        idx = rng.choice(R, size=k, replace=False)
        cuts = np.sort(rng.choice(np.arange(1, 256), size=k - 1, replace=False)) if k > 1 else np.array([], int)
        parts = np.diff(np.concatenate([[0], cuts, [256]])) / 256.0
        a0[p, idx] = parts
    Y64 = a0 @ A.astype(np.float64).T
    Y = Y64.astype(np.float32)
    assert (Y.astype(np.float64) == Y64).all()
    res = oracle.solve(A, Y)
    np.testing.assert_allclose(res.coeffs, a0, atol=1e-11)
    assert res.resid.max() < 1e-12


# ---------------------------------------------------------------- R = 2 closed form
def test_r2_closed_form():
    rng = np.random.default_rng(3)
    L, N = 16, 200
    A = rand_library(rng, L, 2, 0.3)
    Y = rng.uniform(-0.2, 1.2, size=(N, L)).astype(np.float32)
    s = rng.uniform(0.01, 0.1, size=(N, L)).astype(np.float32)
    res = oracle.solve(A, Y, s)
    A64 = A.astype(np.float64)
    d = A64[:, 0] - A64[:, 1]
    t = (Y.astype(np.float64) - A64[:, 1]) @ d / (d @ d)
    a1 = np.clip(t, 0, 1)
    np.testing.assert_allclose(res.coeffs[:, 0], a1, atol=1e-13)
    np.testing.assert_allclose(res.coeffs[:, 1], 1 - a1, atol=1e-13)
    interior = (t > 0) & (t < 1)
    assert interior.sum() > 5 and (~interior).sum() > 5
    sig = np.sqrt((s.astype(np.float64) ** 2) @ (d ** 2)) / (d @ d)
    np.testing.assert_allclose(res.coeff_sigma[interior, 0], sig[interior], rtol=1e-12)
    np.testing.assert_allclose(res.coeff_sigma[interior, 1], sig[interior], rtol=1e-12)
    assert (res.coeff_sigma[~interior] == 0).all()


# ---------------------------------------------------------------- orthonormal library
def simplex_projection(v):
    """Textbook sort-and-threshold Euclidean projection onto the probability simplex."""
    u = np.sort(v)[::-1]
    css = np.cumsum(u) - 1.0
    rho = np.nonzero(u - css / np.arange(1, len(v) + 1) > 0)[0][-1]
    return np.maximum(v - css[rho] / (rho + 1.0), 0.0)


@pytest.mark.parametrize("R", [5, 24, 64])
def test_orthonormal_library_is_simplex_projection(R):
    L = 64
    H = np.array([[1.0]])
    while H.shape[0] < L:
        H = np.block([[H, H], [H, -H]])
    rng = np.random.default_rng(R)
    cols = rng.choice(L, size=R, replace=False)
    A = (H[:, cols] / 8.0).astype(np.float32)          # exactly orthonormal in fp32
    assert np.array_equal(A.astype(np.float64).T @ A.astype(np.float64), np.eye(R))
    Y = (rng.standard_normal((40, L)) * 0.3).astype(np.float32)
    res = oracle.solve(A, Y)
    for p in range(40):
        ref = simplex_projection(A.astype(np.float64).T @ Y[p].astype(np.float64))
        np.testing.assert_allclose(res.coeffs[p], ref, atol=1e-13)


# ---------------------------------------------------------------- interior closed forms
def test_interior_equals_scls_and_unconstrained():
    rng = np.random.default_rng(11)
    L, R, N = 30, 6, 40
    A = rand_library(rng, L, R, 0.2)
    A64 = A.astype(np.float64)
    a0 = simplex_points(rng, N, R, 5.0) * 0.7 + 0.3 / R        # well inside the simplex
    Y = (a0 @ A64.T + 1e-3 * rng.standard_normal((N, L))).astype(np.float32)
    res = oracle.solve(A, Y)
    K = np.linalg.inv(A64.T @ A64)
    one = np.ones(R)
    for p in range(N):
        b = A64.T @ Y[p].astype(np.float64)
        scls = K @ b - K @ one * ((one @ K @ b - 1.0) / (one @ K @ one))      # Settle-Drake
        assert scls.min() > 0
        np.testing.assert_allclose(res.coeffs[p], scls, atol=1e-11)
    # unconstrained LS is the answer when it is itself on the simplex
    Q, _ = np.linalg.qr(np.concatenate([A64, rng.standard_normal((L, L - R))], axis=1))
    perp = Q[:, R:]
    A_exact = (np.round(A64 * 1024) / 1024)
    a_exact = np.round(a0 * 256) / 256
    a_exact[:, -1] = 1.0 - a_exact[:, :-1].sum(1)
    Y2 = a_exact @ A_exact.T
    res2 = oracle.solve(A_exact.astype(np.float32), Y2.astype(np.float32))
    ls = np.linalg.lstsq(A_exact, Y2.T, rcond=None)[0].T
    np.testing.assert_allclose(res2.coeffs, ls, atol=1e-10)
    del perp


# ---------------------------------------------------------------- invariances and orderings
def test_invariances_and_orderings():
    rng = np.random.default_rng(5)
    L, R, N = 32, 8, 30
    # few mantissa bits so that scaling by 2 and offsets of 0.25 are exact in fp32
    A = (rng.integers(64, 1024, size=(L, R)) / 1024.0).astype(np.float32)
    a0 = simplex_points(rng, N, R, 0.3)
    Y = np.round((a0 @ A.astype(np.float64).T + 0.01 * rng.standard_normal((N, L))) * 4096) / 4096
    Y = Y.astype(np.float32)
    base = oracle.solve(A, Y)
    perm = rng.permutation(R)
    rp = oracle.solve(np.ascontiguousarray(A[:, perm]), Y)
    np.testing.assert_allclose(rp.coeffs, base.coeffs[:, perm], atol=1e-11)
    rs = oracle.solve(2 * A, 2 * Y)
    np.testing.assert_allclose(rs.coeffs, base.coeffs, atol=1e-11)
    np.testing.assert_allclose(rs.resid, 2 * base.resid, rtol=1e-10)
    ro = oracle.solve(A + np.float32(0.25), Y + np.float32(0.25))        # sum-to-one => offset invariance
    np.testing.assert_allclose(ro.coeffs, base.coeffs, atol=1e-10)
    A64 = A.astype(np.float64)
    K = np.linalg.inv(A64.T @ A64); one = np.ones(R)
    for p in range(N):
        y = Y[p].astype(np.float64)
        Fs = objective(A, Y[p], base.coeffs[p])
        for j in range(R):
            assert Fs <= objective(A, Y[p], np.eye(R)[j]) + 1e-14
        for a in simplex_points(rng, 20, R, 1.0):
            assert Fs <= objective(A, Y[p], a) + 1e-14
        b = A64.T @ y
        ls = K @ b
        scls = ls - K @ one * ((one @ ls - 1.0) / (one @ K @ one))
        assert Fs >= objective(A, Y[p], scls) - 1e-12 >= objective(A, Y[p], ls) - 2e-12


def test_nnls_cross_check():
    """Approximate: FCLS == NNLS on the system augmented with a heavily weighted sum-to-one row."""
    from scipy.optimize import nnls
    w = make_workload("tiny")
    res = oracle.solve(w.A, w.Y[:40])
    delta = 1e3
    A64 = w.A.astype(np.float64)
    Aa = np.vstack([A64, delta * np.ones((1, w.R))])
    for p in range(40):
        x, _ = nnls(Aa, np.concatenate([w.Y[p].astype(np.float64), [delta]]), maxiter=1000)
        np.testing.assert_allclose(res.coeffs[p], x, atol=2e-5)


# ---------------------------------------------------------------- uncertainties (R3, R4)
def test_sigma_homoscedastic_projected_inverse_hessian():
    """sigma constant => coeff_sigma_i = sigma * sqrt(H_ii), H = K - K11'K/(1'K1), K = (A_F'A_F)^-1."""
    w = make_workload("tiny")
    res = oracle.solve(w.A, w.Y[:100], w.sigma[:100])
    A64 = w.A.astype(np.float64)
    for p in range(100):
        F = np.nonzero(res.coeffs[p] > 0)[0]
        ref = np.zeros(w.R)
        if len(F) > 1:
            K = np.linalg.inv(A64[:, F].T @ A64[:, F]); one = np.ones(len(F))
            H = K - np.outer(K @ one, one @ K) / (one @ K @ one)
            ref[F] = 0.005 * np.sqrt(np.diag(H))
        np.testing.assert_allclose(res.coeff_sigma[p], ref, rtol=1e-7, atol=1e-12)


def test_sigma_is_propagation_through_solution_map():
    """Finite differences of the (brute-force pinned) minimiser give J; sigma^2 = sum_l J_il^2 s_l^2."""
    rng = np.random.default_rng(21)
    L, R = 12, 5
    A = rand_library(rng, L, R, 0.5)
    a0 = np.array([0.5, 0.3, 0.2, 0.0, 0.0])
    y = (A.astype(np.float64) @ a0 + 0.01 * rng.standard_normal(L)).astype(np.float32)
    s = rng.uniform(0.002, 0.01, size=L).astype(np.float32)
    base = oracle.solve(A, y[None], s[None])
    F = base.coeffs[0] > 0
    assert 2 <= F.sum() < R and base.coeffs[0][F].min() > 0.02
    h = 2.0 ** -12
    Yp = np.repeat(y[None], L, 0); Ym = Yp.copy()
    for l in range(L):
        Yp[l, l] += np.float32(h); Ym[l, l] -= np.float32(h)
    rp = oracle.solve(A, Yp); rm = oracle.solve(A, Ym)
    assert ((rp.coeffs > 0) == F).all() and ((rm.coeffs > 0) == F).all()
    step = (Yp.astype(np.float64) - Ym.astype(np.float64))[np.arange(L), np.arange(L)]
    J = ((rp.coeffs - rm.coeffs) / step[:, None]).T            # (R, L)
    ref = np.sqrt((J ** 2) @ (s.astype(np.float64) ** 2))
    np.testing.assert_allclose(base.coeff_sigma[0], ref, rtol=1e-7, atol=1e-12)
    np.testing.assert_allclose(J.sum(0), 0.0, atol=1e-9)       # rows of Cov sum to zero (1'H = 0)


def _mc(A, y_clean, s, n, rng):
    Y = (y_clean[None] + s[None] * rng.standard_normal((n, len(y_clean)))).astype(np.float32)
    return oracle.solve(A, Y)


def test_sigma_monte_carlo_interior():
    """R4(i): all endmembers strongly present; resampled std of a == linearised sigma within 2 %."""
    rng = np.random.default_rng(31)
    w = make_workload("tiny")
    A64 = w.A.astype(np.float64)
    a0 = np.full(w.R, 1.0 / w.R)
    y = A64 @ a0
    s = rng.uniform(2e-6, 1e-5, size=w.L).astype(np.float32)
    lin = oracle.solve(w.A, y.astype(np.float32)[None], s[None])
    assert lin.support_size[0] == w.R and (lin.coeffs[0] / lin.coeff_sigma[0]).min() > 100
    mc = _mc(w.A, y, s.astype(np.float64), 20000, rng)
    assert (mc.support_size == w.R).all()
    np.testing.assert_allclose(mc.coeffs.std(0), lin.coeff_sigma[0], rtol=0.02)


def test_sigma_monte_carlo_strongly_active():
    """R4(ii): two endmembers pushed hard against a >= 0 (pseudo-abundance -0.25), heteroscedastic noise."""
    rng = np.random.default_rng(32)
    w = make_workload("tiny")
    A64 = w.A.astype(np.float64)
    a0 = np.array([0.5, 0.4, 0.3, 0.3, -0.25, -0.25, 0.0, 0.0])
    a0[6] = 1.0 - a0.sum() - 0.0
    a0[7] = 1.0 - a0.sum()
    y = A64 @ a0
    s = rng.uniform(5e-6, 4e-5, size=w.L).astype(np.float32)
    lin = oracle.solve(w.A, y.astype(np.float32)[None], s[None])
    F = lin.coeffs[0] > 0
    assert not F[4] and not F[5] and F.sum() >= 3
    mc = _mc(w.A, y, s.astype(np.float64), 20000, rng)
    assert ((mc.coeffs > 0) == F).all()          # same support in every resample
    np.testing.assert_allclose(mc.coeffs.std(0)[F], lin.coeff_sigma[0][F], rtol=0.02)
    assert (lin.coeff_sigma[0][~F] == 0).all()


# ---------------------------------------------------------------- residual (R8)
def test_resid_definition_and_noise_level():
    w = make_workload("omega", N=3000)
    res = oracle.solve(w.A, w.Y, w.sigma)
    r = w.Y.astype(np.float64) - res.coeffs @ w.A.astype(np.float64).T
    np.testing.assert_allclose(res.resid, np.sqrt((r ** 2).mean(1)), rtol=1e-12)
    # "RMS compatible with the level of noise": E[L RMS^2] ~ sum_l s_l^2 (1 - (k-1)/L) on average
    s2 = (w.sigma.astype(np.float64) ** 2)
    expect = (s2.sum(1) * (1.0 - (res.support_size - 1) / w.L)).mean()
    got = (w.L * res.resid ** 2).mean()
    assert abs(got / expect - 1.0) < 0.03


# ---------------------------------------------------------------- degenerate inputs
def test_degenerate_cases():
    rng = np.random.default_rng(9)
    L = 10
    # R = 1: a = 1 whatever y
    A1 = rand_library(rng, L, 1)
    y = rng.uniform(0, 1, size=(3, L)).astype(np.float32)
    r = oracle.solve(A1, y, np.full((3, L), 0.01, np.float32))
    assert (r.coeffs == 1.0).all() and (r.coeff_sigma == 0).all()
    # duplicate column: objective still minimal, sum of the twins equals the unique answer
    A = rand_library(rng, L, 4, 0.3)
    Ad = np.concatenate([A, A[:, :1]], axis=1)
    a0 = np.array([0.5, 0.2, 0.3, 0.0])
    Y = (A.astype(np.float64) @ a0 + 0.01 * rng.standard_normal((20, L))).astype(np.float32)
    ru = oracle.solve(A, Y); rd = oracle.solve(Ad, Y)
    np.testing.assert_allclose(rd.coeffs[:, 0] + rd.coeffs[:, 4], ru.coeffs[:, 0], atol=1e-10)
    np.testing.assert_allclose(rd.resid, ru.resid, rtol=1e-10)
    # non-finite pixel -> NaN outputs, flagged; neighbours untouched
    Yn = Y.copy(); Yn[3, 2] = np.nan
    rn = oracle.solve(A, Yn)
    assert np.isnan(rn.coeffs[3]).all() and rn.status[3] == 4
    np.testing.assert_array_equal(rn.coeffs[4], ru.coeffs[4])
    # R > L (PAPER.md:92 says R <= L; configs[3] violates it): objective equals brute force
    Aw = rand_library(rng, 4, 6, 0.2)
    Yw = rng.uniform(0.1, 0.9, size=(10, 4)).astype(np.float32)
    rw = oracle.solve(Aw, Yw)
    for p in range(10):
        _, obj = brute_force_fcls(Aw, Yw[p])
        assert abs(objective(Aw, Yw[p], rw.coeffs[p]) - obj) <= 1e-12 * max(obj, 1e-9)
    # empty batch
    r0 = oracle.solve(A, np.zeros((0, L), np.float32))
    assert r0.coeffs.shape == (0, 4)


# ---------------------------------------------------------------- rank margin (R9): the uniqueness mask of tests/parity.py
def _sigma_min_AFZ(A64, F):
    """sigma_min(A_F Z) from numpy's SVD, Z = ANY orthonormal basis of {z : 1'z = 0} (here from numpy's QR of
    [1 | I]; the singular values do not depend on the choice)."""
    k = len(F)
    Q, _ = np.linalg.qr(np.concatenate([np.ones((k, 1)), np.eye(k)[:, : k - 1]], axis=1))
    Z = Q[:, 1:]
    assert np.abs(Z.sum(0)).max() < 1e-12
    return np.linalg.svd(A64[:, F] @ Z, compute_uv=False)[-1]


@pytest.mark.parametrize("name,n", [("tiny", 400), ("omega", 400), ("crism", 150), ("stress", 120)])
def test_rank_margin_brackets_sigma_min(name, n):
    """rank_margin (smallest |R_jj| of the column-pivoted QR of A_F Z on the final support) decides which pixels
    get element-wise coefficient / sigma assertions (tests/parity.py).  For a column-pivoted QR
    sigma_min <= min |R_jj| <= sqrt(m) 2^(m-1) sigma_min in theory and a small multiple in practice: pin
    it inside [1, 6] x numpy's sigma_min(A_F Z), so a bookkeeping slip (wrong column, stale value of an earlier
    support, wrong reduction) cannot silently switch the assertions off."""
    w = make_workload(name, N=n)
    res = oracle.solve(w.A, w.Y, w.sigma)
    A64 = w.A.astype(np.float64)
    ratios = []
    for p in range(n):
        F = np.nonzero(res.coeffs[p] > 0)[0]
        assert len(F) == res.support_size[p]
        if len(F) == 1:
            assert np.isinf(res.rank_margin[p])
            continue
        ratios.append(res.rank_margin[p] / _sigma_min_AFZ(A64, F))
    ratios = np.array(ratios)
    assert len(ratios) > n // 2
    assert ratios.min() >= 1.0 - 1e-9 and ratios.max() <= 6.0, (ratios.min(), ratios.max())


def test_rank_margin_of_near_duplicate_columns():
    """Two members that differ by delta: the margin must come out at the size of delta (here ~1e-7 of
    sigma_max, below the 1e-6 mask of tests/parity.py), and scale with delta."""
    rng = np.random.default_rng(41)
    L = 16
    base = rand_library(rng, L, 3, 0.2).astype(np.float64)
    v = rng.standard_normal(L)
    margins = []
    for delta in (2.0 ** -20, 2.0 ** -17):
        A = np.concatenate([base, base[:, :1] + delta * v[:, None]], axis=1).astype(np.float32)
        a0 = np.array([0.3, 0.25, 0.15, 0.3])
        y = (A.astype(np.float64) @ a0).astype(np.float32)
        res = oracle.solve(A, y[None])
        F = np.nonzero(res.coeffs[0] > 0)[0]
        if len(F) == 4:            # both twins active: the margin is that of the near-dependent pair
            smin = _sigma_min_AFZ(A.astype(np.float64), F)
            assert 1.0 - 1e-9 <= res.rank_margin[0] / smin <= 6.0
            smax = np.linalg.svd(A.astype(np.float64), compute_uv=False)[0]
            assert res.rank_margin[0] < 1e-5 * smax
            margins.append(res.rank_margin[0])
    assert len(margins) == 2 and 6.0 < margins[1] / margins[0] < 10.0      # delta ratio is 8
    # exact duplicate: the second twin is rejected as rank-deficient and the pixel is flagged
    Ad = np.concatenate([base, base[:, :1]], axis=1).astype(np.float32)
    y = (Ad.astype(np.float64) @ np.array([0.3, 0.25, 0.15, 0.3]) + 1e-3 * rng.standard_normal(L)).astype(np.float32)
    rd = oracle.solve(Ad, y[None])
    assert rd.coeffs[0, 0] == 0.0 or rd.coeffs[0, 3] == 0.0


# ---------------------------------------------------------------- the certificate tests/parity.py runs on every compared pixel
@pytest.mark.parametrize("name,n", [("tiny", 1000), ("omega", 20000), ("crism", 3000), ("stress", 300)])
def test_parity_certificate_on_oracle_outputs(name, n):
    """tests/parity.py::check_oracle_kkt (numpy, independent of oracle/) accepts the oracle's answers, multipliers
    included, on every pixel; and it rejects a perturbed answer (so it is not vacuous)."""
    import sys
    sys.path.insert(0, HERE)
    from parity import check_oracle_kkt
    w = make_workload(name, N=n)
    res = oracle.solve(w.A, w.Y, w.sigma)
    worst = check_oracle_kkt(w.A, w.Y, res, label=name)
    assert worst["lam_neg"] <= 1e-9
    # move 1e-6 of mass between two active members of one pixel, or drop a weakly active member: must be caught
    p = int(np.argmax(res.support_size))
    F = np.nonzero(res.coeffs[p] > 0)[0]
    bad = oracle.OracleResult(*[np.array(getattr(res, f), copy=True) for f in
                                ("coeffs", "coeff_sigma", "resid", "lam", "nu", "support_size", "steps", "rank_margin", "status")])
    bad.coeffs[p, F[0]] += 1e-6; bad.coeffs[p, F[1]] -= 1e-6
    with pytest.raises(AssertionError):
        check_oracle_kkt(w.A, w.Y, bad, label="perturbed")
