"""Shared parity checks: CUDA path (through the C ABI) vs the fp64 oracle, on identical inputs.

Tolerances are north_star's (BASELINE.json), read as in DESIGN.md R10/R12:
  max |a_gpu - a*| <= 1e-4, |sum a - 1| <= 1e-5, a >= -1e-6,
  |F(a_gpu) - F*| <= 1e-5 max(F*, 1e-12 ||y||^2) with F re-evaluated here in fp64,
  resid within 1e-5 relative (same floor), coeff_sigma within 1 % relative (+1e-7 absolute) where the
  supports agree; where they differ (ties, R10) the GPU value is compared with reading R3 evaluated
  in numpy ON THE GPU's support, and the number of such pixels must stay below 0.5 %.

Before the oracle's answer is used as the reference for a pixel it is itself certified HERE, in numpy,
independently of oracle/ (check_oracle_kkt): the scaled optimality conditions of the problem (R11) on its
coefficients, and its multipliers against the recomputed ones, for EVERY compared pixel.
"""
import numpy as np


def sigma_reference_on_support(A64, F, sig):
    """Reading R3 written out with numpy for a given support (independent of oracle/ and of csrc/)."""
    out = np.zeros(A64.shape[1])
    F = np.asarray(F)
    if len(F) <= 1:
        return out
    AF = A64[:, F]
    K = np.linalg.inv(AF.T @ AF)
    one = np.ones(len(F))
    H = K - np.outer(K @ one, one @ K) / (one @ K @ one)
    J = H @ AF.T
    out[F] = np.sqrt((J ** 2) @ (sig.astype(np.float64) ** 2))
    return out


def sigma_reference_next(A64, F, equality, Ci=None, sig=None):
    """Reading R3 (and R17 for the renormalised problem) written out with numpy for a given support and option:
    a = H A_F' M y + const with M = C^-1 (identity when unweighted), K = (A_F' M A_F)^-1, H = K under positivity only
    and K - K 1 1' K / (1' K 1) under the sum constraint; cov(a) = J Sigma J', J = H A_F' M.  Weighted: Sigma = C, so
    cov(a) = H K^-1 H = H; unweighted: Sigma = diag(sig^2)."""
    out = np.zeros(A64.shape[1])
    F = np.asarray(F)
    if len(F) == 0 or (equality and len(F) <= 1):
        return out
    AF = A64[:, F]
    M = np.eye(A64.shape[0]) if Ci is None else Ci
    K = np.linalg.inv(AF.T @ M @ AF)
    one = np.ones(len(F))
    H = K - np.outer(K @ one, one @ K) / (one @ K @ one) if equality else K
    if Ci is not None:
        out[F] = np.sqrt(np.maximum(np.diag(H), 0.0))
    else:
        s2 = np.ones(A64.shape[0]) if sig is None else sig.astype(np.float64) ** 2
        out[F] = np.sqrt(((H @ AF.T) ** 2) @ s2)
    return out


def check_oracle_kkt(A, Y, ora, label="", tol=1e-9, chunk=65536):
    """Optimality conditions of eq. 2 under eq. 3-4 for the ORACLE's coefficients, recomputed
    in numpy from the coefficients alone, on every pixel handed in (scaled as reading R11): sum a = 1, a >= 0,
    multipliers >= -tol, complementarity and stationarity on the support <= tol, all relative to ||g||_inf plus the
    rounding scale of g (1e-13 max_i sum_l |A_li||y_l|: g = 0 exactly on a noiseless pixel).  Also compares the
    oracle's own lambda / nu outputs with the recomputed ones.  A pixel on which the oracle blocked an index
    (rank loss or degenerate tie) is certified like any other: a wrongly blocked index shows up as a negative
    multiplier here."""
    A64 = A.astype(np.float64)
    absA = np.abs(A64)
    worst = dict(sum=0.0, neg=0.0, lam_neg=0.0, stat=0.0, lam_out=0.0, nu_out=0.0)
    N = Y.shape[0]
    for p0 in range(0, N, chunk):
        sl = slice(p0, min(N, p0 + chunk))
        a = ora.coeffs[sl]
        y = Y[sl].astype(np.float64)
        ok = np.isfinite(y).all(1)
        a, y = a[ok], y[ok]
        if a.shape[0] == 0:
            continue
        g = (a @ A64.T - y) @ A64                      # gradient of F/2
        F = a > 0
        nu = -(g * a).sum(1)
        scale = np.abs(g).max(1) + 1e-4 * (np.abs(y) @ absA).max(1)   # 1e-4 * tol = the 1e-13 rounding floor
        lam = np.where(F, 0.0, g + nu[:, None])
        worst["sum"] = max(worst["sum"], float(np.abs(a.sum(1) - 1.0).max()))
        worst["neg"] = max(worst["neg"], float(max(0.0, -a.min())))
        worst["lam_neg"] = max(worst["lam_neg"], float((np.maximum(0.0, -lam.min(1)) / scale).max()))
        worst["stat"] = max(worst["stat"], float((np.abs(np.where(F, g + nu[:, None], 0.0)).max(1) / scale).max()))
        worst["lam_out"] = max(worst["lam_out"], float((np.abs(ora.lam[sl][ok] - lam).max(1) / scale).max()))
        worst["nu_out"] = max(worst["nu_out"], float((np.abs(ora.nu[sl][ok] - nu) / scale).max()))
    assert worst["sum"] <= 1e-12, (label, "oracle KKT", worst)
    assert worst["neg"] == 0.0, (label, "oracle KKT", worst)
    assert worst["lam_neg"] <= tol, (label, "oracle KKT", worst)
    assert worst["stat"] <= tol, (label, "oracle KKT", worst)
    assert worst["lam_out"] <= tol and worst["nu_out"] <= tol, (label, "oracle multipliers", worst)
    return worst


def check_parity(A, Y, sigma, gpu, ora, label="", min_unique=0.99, max_tie_frac=0.005):
    """gpu: dict(coeffs, coeff_sigma, resid) numpy float32 arrays for the SAME pixels as ora.
    min_unique: asserted lower bound on the fraction of pixels whose minimiser is unique (R9) and on which the
    coefficients and uncertainties are therefore compared element by element."""
    A64 = A.astype(np.float64)
    Y64 = Y.astype(np.float64)
    a = gpu["coeffs"].astype(np.float64)
    N, R = a.shape
    L = A.shape[0]
    assert np.isfinite(a).all(), label
    kkt = check_oracle_kkt(A, Y, ora, label)
    # feasibility
    assert np.abs(a.sum(1) - 1.0).max() <= 1e-5, (label, np.abs(a.sum(1) - 1.0).max())
    assert a.min() >= -1e-6, (label, a.min())
    # objective (R12)
    Fg = ((Y64 - a @ A64.T) ** 2).sum(1)
    Fo = ((Y64 - ora.coeffs @ A64.T) ** 2).sum(1)
    floor = 1e-12 * (Y64 ** 2).sum(1)
    rel = np.abs(Fg - Fo) / np.maximum(Fo, floor)
    assert rel.max() <= 1e-5, (label, "objective", rel.max(), int(rel.argmax()))
    # coefficients: where the minimiser is unique (R9); the mask is pinned by tests/test_oracle_pins.py::
    # test_rank_margin_* and its size is asserted, never just printed
    sing = np.linalg.svd(A64, compute_uv=False)
    unique = ora.rank_margin > 1e-6 * sing[0]
    assert unique.mean() >= min_unique, (label, "unique fraction", unique.mean(), min_unique)
    assert unique.any(), (label, "no pixel with a unique minimiser")
    da = np.abs(a - ora.coeffs).max(1)
    assert da[unique].max() <= 1e-4, (label, "coeffs", da[unique].max(), int(np.argmax(np.where(unique, da, 0))))
    stats = dict(pixels=int(N), max_da=float(da[unique].max()), max_rel_obj=float(rel.max()),
                 n_nonunique=int((~unique).sum()), oracle_kkt=max(kkt["lam_neg"], kkt["stat"]))
    # residual
    if gpu.get("resid") is not None:
        rg = gpu["resid"].astype(np.float64)
        rr = np.abs(rg - ora.resid) / np.maximum(ora.resid, np.sqrt(floor / L))
        assert rr.max() <= 1e-5, (label, "resid", rr.max())
        stats["max_rel_resid"] = float(rr.max())
    # uncertainties
    if gpu.get("coeff_sigma") is not None:
        sg = gpu["coeff_sigma"].astype(np.float64)
        Fg_sup = a > 0
        Fo_sup = ora.coeffs > 0
        same = (Fg_sup == Fo_sup).all(1)
        err = np.abs(sg - ora.coeff_sigma) - (0.01 * ora.coeff_sigma + 1e-7)
        if (same & unique).any():
            assert err[same & unique].max() <= 0, (label, "sigma", err[same & unique].max())
        ties = np.nonzero(~same & unique)[0]
        assert len(ties) <= max(2, max_tie_frac * N), (label, "support mismatches", len(ties))
        for p in ties:
            # the differing members must be marginal (tiny coefficient on either side)
            diff = Fg_sup[p] ^ Fo_sup[p]
            assert max(a[p][diff].max(), ora.coeffs[p][diff].max()) < 1e-4, (label, p)
            sp = sigma[p] if sigma.ndim == 2 else sigma
            ref = sigma_reference_on_support(A64, np.nonzero(Fg_sup[p])[0], sp)
            assert (np.abs(sg[p] - ref) <= 0.01 * ref + 1e-7).all(), (label, "tie sigma", p)
        stats["n_support_ties"] = int(len(ties))
        m = same & unique
        pos = ora.coeff_sigma[m] > 1e-6
        stats["max_rel_sigma"] = float((np.abs(sg[m] - ora.coeff_sigma[m])[pos] / ora.coeff_sigma[m][pos]).max()) if pos.any() else 0.0
    return stats


def check_parity_next(A, Y, gpu, ora, constraint="sto", cov=None, label="", max_tie_frac=0.005, sigma=None,
                      coeff_outliers=(0, 1e-4)):
    """Same tolerances for the NEXT-row options: constraint "sto" | "slo" | "pos", and the renormalised
    problem (cov = (L,) noise std or (L, L) covariance; objective and residual in the C^-1 metric, unit noise for the
    uncertainties).  The oracle's answer is first certified in numpy (optimality conditions in that metric).
    sigma: the per-channel noise std both sides were given (unweighted problem; None = ones), used on tie pixels (R10),
    where the GPU's uncertainties must equal R3 evaluated in numpy on the GPU's own support.
    coeff_outliers = (k, bound): at most k pixels may miss the 1e-4 coefficient tolerance and none may miss `bound`;
    their indices come back in stats["coeff_outliers"] and the CALLER has to account for each of them (the default
    allows none).  Used by one test only, reading R20."""
    A64 = A.astype(np.float64); Y64 = Y.astype(np.float64)
    N, L = Y.shape
    R = A.shape[1]
    if cov is None:
        Ci = np.eye(L)
    elif cov.ndim == 1:
        Ci = np.diag(1.0 / cov.astype(np.float64) ** 2)
    else:
        Ci = np.linalg.inv(cov.astype(np.float64))
    a = gpu["coeffs"].astype(np.float64)
    ao = ora.coeffs
    assert np.isfinite(a).all(), label
    # ---- the oracle's optimality in numpy, every pixel
    g = ((ao @ A64.T - Y64) @ Ci) @ A64
    F = ao > 0
    scale = np.abs(g).max(1) + 1e-4 * (np.abs(Y64 @ Ci) @ np.abs(A64)).max(1)
    if constraint == "sto":
        nu = -(g * ao).sum(1)
        assert np.abs(ao.sum(1) - 1).max() <= 1e-12
    elif constraint == "slo":
        s = ao.sum(1)
        nu = np.where(s >= 1 - 1e-12, -(g * ao).sum(1) / np.maximum(s, 1e-300), 0.0)
        assert s.max() <= 1 + 1e-12 and (nu / scale).min() >= -1e-9, (label, "oracle slo multiplier")
    else:
        nu = np.zeros(N)
    gn = g + nu[:, None]
    assert (np.abs(np.where(F, gn, 0.0)).max(1) / scale).max() <= 1e-9, (label, "oracle stationarity")
    assert (np.where(F, 0.0, gn).min(1) / scale).min() >= -1e-9, (label, "oracle multipliers")
    # ---- feasibility of the GPU answer
    assert a.min() >= -1e-6, (label, a.min())
    if constraint == "sto":
        assert np.abs(a.sum(1) - 1.0).max() <= 1e-5, (label, np.abs(a.sum(1) - 1.0).max())
    elif constraint == "slo":
        assert a.sum(1).max() <= 1.0 + 1e-5, (label, a.sum(1).max())
    # ---- objective in the C^-1 metric (R12)
    rg = Y64 - a @ A64.T; ro = Y64 - ao @ A64.T
    Fg = np.einsum("pl,lm,pm->p", rg, Ci, rg); Fo = np.einsum("pl,lm,pm->p", ro, Ci, ro)
    floor = 1e-12 * np.einsum("pl,lm,pm->p", Y64, Ci, Y64)
    rel = np.abs(Fg - Fo) / np.maximum(Fo, floor)
    assert rel.max() <= 1e-5, (label, "objective", rel.max(), int(rel.argmax()))
    sing = np.linalg.svd(A64, compute_uv=False)
    unique = ora.rank_margin > 1e-6 * sing[0] * (np.sqrt(np.linalg.eigvalsh(Ci).min()) if cov is not None else 1.0)
    assert unique.mean() >= 0.99, (label, "unique fraction", unique.mean())
    da = np.abs(a - ao).max(1)
    out = np.nonzero(unique & (da > 1e-4))[0]
    assert len(out) <= coeff_outliers[0] and da[unique].max() <= coeff_outliers[1], \
        (label, "coeffs", da[unique].max(), int(np.argmax(np.where(unique, da, 0))), len(out))
    stats = dict(pixels=int(N), max_da=float(da[unique].max()), max_rel_obj=float(rel.max()),
                 coeff_outliers=[int(p) for p in out])
    if gpu.get("resid") is not None:
        rr = np.abs(gpu["resid"].astype(np.float64) - ora.resid) / np.maximum(ora.resid, np.sqrt(floor / L))
        assert rr.max() <= 1e-5, (label, "resid", rr.max())
        stats["max_rel_resid"] = float(rr.max())
    if gpu.get("coeff_sigma") is not None:
        sg = gpu["coeff_sigma"].astype(np.float64)
        same = ((a > 0) == (ao > 0)).all(1)
        err = np.abs(sg - ora.coeff_sigma) - (0.01 * ora.coeff_sigma + 1e-7)
        m = same & unique
        assert err[m].max() <= 0, (label, "sigma", err[m].max())
        ties = np.nonzero(~same & unique)[0]
        assert len(ties) <= max(2, max_tie_frac * N), (label, "support mismatches", len(ties))
        for p in ties:
            diff = (a[p] > 0) ^ (ao[p] > 0)
            assert max(a[p][diff].max(), ao[p][diff].max()) < 1e-4, (label, p)
            # R10: the GPU's sigma is R3 on the GPU's support (slo: the sum bound counts as active when the sum is one;
            # within rounding of one either reading is a valid side of the tie)
            sp = None if (sigma is None or cov is not None) else (sigma[p] if sigma.ndim == 2 else sigma)
            if constraint == "sto":
                eqs = [True]
            elif constraint == "pos":
                eqs = [False]
            else:
                sm = a[p].sum()
                eqs = [True, False] if abs(sm - 1.0) <= 1e-5 else [sm > 1.0 - 1e-5]
            Fp = np.nonzero(a[p] > 0)[0]
            ok = False
            for eq in eqs:
                ref = sigma_reference_next(A64, Fp, eq, Ci if cov is not None else None, sp)
                ok = ok or bool((np.abs(sg[p] - ref) <= 0.01 * ref + 1e-7).all())
            assert ok, (label, "tie sigma", int(p))
        stats["n_support_ties"] = int(len(ties))
    return stats
