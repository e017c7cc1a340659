"""-m gpu: the CUDA path, called through the C ABI (ctypes binding), against the fp64 oracle on the
same seeded inputs.  Tolerances: tests/parity.py (north_star).  Nothing here reads /root/reference."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


@pytest.fixture(scope="module")
def lm():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_1402_2518_b200 import build, linmin
    build.build_library()
    linmin.load()
    return linmin


def run_gpu(lm, A, Y, sigma, **kw):
    dev = torch.device("cuda:0")
    At = torch.from_numpy(A).to(dev)
    Yt = torch.from_numpy(Y).to(dev)
    st = None if sigma is None else torch.from_numpy(sigma).to(dev)
    c, s, r, info, status = lm.unmix(At, Yt, st, **kw)
    torch.cuda.synchronize()
    return dict(coeffs=c.cpu().numpy(), coeff_sigma=None if s is None else s.cpu().numpy(),
                resid=None if r is None else r.cpu().numpy(), info=info.cpu().numpy(), status=status)


def subsample(g, sel):
    return {k: (v[sel] if isinstance(v, np.ndarray) else v) for k, v in g.items()}


# ------------------------------------------------------------------ the five configs
@pytest.mark.parametrize("name,stride", [("tiny", 1), ("omega", 1), ("crism", 1), ("stress", 1)])
def test_config_parity(lm, name, stride):
    """Full-size configs 0-3 (BASELINE.json configs[0..3]); the oracle checks EVERY pixel."""
    import oracle
    from paper_1402_2518_b200.synth import make_workload
    from parity import check_parity
    w = make_workload(name)
    g = run_gpu(lm, w.A, w.Y, w.sigma)
    sel = np.arange(0, w.N, stride)
    ora = oracle.solve(w.A, w.Y[sel], w.sigma[sel])
    stats = check_parity(w.A, w.Y[sel], w.sigma[sel], subsample(g, sel), ora, label=name)
    assert stats["pixels"] == w.N
    info = g["info"]
    assert ((info & lm.INFO_NONFINITE_INPUT) == 0).all()
    assert ((info & lm.INFO_FINISH_FALLBACK) == 0).mean() > 0.9999
    # exact zeros off the support, support size reported
    assert (((g["coeffs"] > 0).sum(1)) == ((info >> 24) & 0xff)).all()
    if name == "crism":      # pixels drawn on a simplex face are reported separately
        face = w.face[sel]
        da = np.abs(subsample(g, sel)["coeffs"] - ora.coeffs).max(1)
        assert da[face].max() <= 1e-4
    print(name, stats, "iters mean", ((info >> 8) & 0xff).mean(), "pivots mean", ((info >> 16) & 0xff).mean())


def test_throughput_config_sampled(lm):
    """Config 4 (a stack of OMEGA-like cubes): 8 cubes = 1,048,576 pixels on the GPU, every 64th
    pixel against the oracle."""
    import oracle
    from paper_1402_2518_b200.synth import make_workload
    from parity import check_parity
    w = make_workload("throughput", n_cubes=8)
    g = run_gpu(lm, w.A, w.Y, w.sigma)
    sel = np.arange(0, w.N, 64)
    ora = oracle.solve(w.A, w.Y[sel], w.sigma[sel])
    print(check_parity(w.A, w.Y[sel], w.sigma[sel], subsample(g, sel), ora, label="throughput"))


# ------------------------------------------------------------------ interfaces and edge cases
def test_library_handle_strides_shared_sigma_and_host_path(lm):
    import oracle
    from paper_1402_2518_b200.synth import make_workload
    from parity import check_parity
    w = make_workload("omega", N=1003)          # ragged: not a multiple of any tile size
    dev = torch.device("cuda:0")
    lib = lm.library_create(torch.from_numpy(w.A).to(dev))
    assert lib.status == 0
    # strided Y (ldY > L), shared sigma vector
    Ypad = torch.zeros((w.N, w.L + 5), device=dev)
    Ypad[:, :w.L] = torch.from_numpy(w.Y).to(dev)
    sig = w.sigma[0].copy()
    c, s, r, info, st = lm.unmix_lib(lib, Ypad[:, :w.L], torch.from_numpy(sig).to(dev))
    torch.cuda.synchronize()
    ora = oracle.solve(w.A, w.Y, sig)
    g = dict(coeffs=c.cpu().numpy(), coeff_sigma=s.cpu().numpy(), resid=r.cpu().numpy())
    check_parity(w.A, w.Y, sig, g, ora, label="strided/shared")
    assert lib.last_launches() >= 2
    # sigma == NULL -> noise amplification factors (sigma == 1)
    c1, s1, r1, _, _ = lm.unmix_lib(lib, torch.from_numpy(w.Y).to(dev), None)
    torch.cuda.synchronize()
    ora1 = oracle.solve(w.A, w.Y, None)
    check_parity(w.A, w.Y, np.ones(w.L, np.float32),
                 dict(coeffs=c1.cpu().numpy(), coeff_sigma=s1.cpu().numpy(), resid=r1.cpu().numpy()), ora1, label="nosigma")
    # outputs optional
    c2, s2, r2, i2, _ = lm.unmix_lib(lib, torch.from_numpy(w.Y).to(dev), None, want_sigma=False, want_resid=False, want_info=False)
    torch.cuda.synchronize()
    assert s2 is None and r2 is None and i2 is None
    assert torch.equal(c2, c1)
    # host entry point: same kernels, host buffers -> identical bits
    ch, sh, rh, ih, _ = lm.unmix_host(w.A, w.Y, w.sigma, want_info=True)
    cd, sd, rd, idv, _ = lm.unmix_lib(lib, torch.from_numpy(w.Y).to(dev), torch.from_numpy(w.sigma).to(dev))
    torch.cuda.synchronize()
    assert np.array_equal(ch.numpy(), cd.cpu().numpy())
    assert np.array_equal(sh.numpy(), sd.cpu().numpy())
    assert np.array_equal(rh.numpy(), rd.cpu().numpy())
    assert np.array_equal(ih.numpy(), idv.cpu().numpy())
    lib.destroy()


@pytest.mark.parametrize("constraint", [0, 1, 2])
def test_arrays_need_only_float_alignment(lm, constraint):
    """include/linmin.h, "Alignment": every array may sit on any 4-byte boundary.  R = 32 is the size whose IPLS kernel
    stores 16 bytes at a time; outputs (and Y, sigma) that are sub-views one float into a larger buffer must give the
    oracle's result, not a misaligned-address fault."""
    import oracle
    from paper_1402_2518_b200.synth import make_workload
    from parity import check_parity, check_parity_next
    w = make_workload("omega", N=1003)
    dev = torch.device("cuda:0")
    assert w.R == 32

    def off1(shape, dtype=torch.float32, src=None):
        n = int(np.prod(shape))
        buf = torch.zeros(n + 1, dtype=dtype, device=dev)
        v = buf[1:].view(*shape)
        if src is not None:
            v.copy_(torch.from_numpy(src).to(dev))
        assert v.data_ptr() % 16 == 4 and v.is_contiguous()
        return v

    Y, S = off1((w.N, w.L), src=w.Y), off1((w.N, w.L), src=w.sigma)
    out = dict(coeffs=off1((w.N, w.R)), coeff_sigma=off1((w.N, w.R)), resid=off1((w.N,)), info=off1((w.N,), torch.int32))
    c, s, r, info, st = lm.unmix(torch.from_numpy(w.A).to(dev), Y, S, out=out, constraint=constraint)
    torch.cuda.synchronize()
    assert c.data_ptr() == out["coeffs"].data_ptr()
    g = dict(coeffs=c.cpu().numpy(), coeff_sigma=s.cpu().numpy(), resid=r.cpu().numpy())
    if constraint == 0:
        check_parity(w.A, w.Y, w.sigma, g, oracle.solve(w.A, w.Y, w.sigma), label="misaligned")
    else:
        name = {1: "slo", 2: "pos"}[constraint]
        check_parity_next(w.A, w.Y, g, oracle.solve(w.A, w.Y, w.sigma, constraint=name), constraint=name,
                          label="misaligned/" + name, sigma=w.sigma)
    # same minimiser as with aligned arrays (another IPLS kernel hands over, the finish is exact)
    ca = lm.unmix(torch.from_numpy(w.A).to(dev), torch.from_numpy(w.Y).to(dev), torch.from_numpy(w.sigma).to(dev),
                  constraint=constraint)[0]
    assert float((ca - c).abs().max()) < 1e-5


def test_empty_single_and_determinism(lm):
    from paper_1402_2518_b200.synth import make_workload
    w = make_workload("tiny", N=9)
    g0 = run_gpu(lm, w.A, w.Y[:0], w.sigma[:0])
    assert g0["coeffs"].shape == (0, 8)
    g1 = run_gpu(lm, w.A, w.Y[:1], w.sigma[:1])
    g9 = run_gpu(lm, w.A, w.Y, w.sigma)
    g9b = run_gpu(lm, w.A, w.Y, w.sigma)
    assert np.array_equal(g1["coeffs"][0], g9["coeffs"][0])       # independent of N / tiling
    assert np.array_equal(g9["coeffs"], g9b["coeffs"])            # run-to-run deterministic
    assert np.array_equal(g9["coeff_sigma"], g9b["coeff_sigma"])


def test_degenerate_inputs(lm):
    import oracle
    from parity import check_parity
    rng = np.random.default_rng(9)
    L = 10
    # R = 1
    A1 = rng.uniform(0.1, 0.9, (L, 1)).astype(np.float32)
    y = rng.uniform(0, 1, (3, L)).astype(np.float32)
    g = run_gpu(lm, A1, y, np.full((3, L), 0.01, np.float32))
    assert (g["coeffs"] == 1.0).all() and (g["coeff_sigma"] == 0).all()
    r = y.astype(np.float64) - A1.astype(np.float64).T
    np.testing.assert_allclose(g["resid"], np.sqrt((r ** 2).mean(1)), rtol=1e-6)
    # R = 2: closed form of tests/test_oracle_pins.py::test_r2_closed_form
    A2 = rng.uniform(0.1, 0.9, (L, 2)).astype(np.float32)
    Y2 = rng.uniform(-0.2, 1.2, (64, L)).astype(np.float32)
    g2 = run_gpu(lm, A2, Y2, None)
    d = A2[:, 0].astype(np.float64) - A2[:, 1]
    t = np.clip((Y2.astype(np.float64) - A2[:, 1]) @ d / (d @ d), 0, 1)
    np.testing.assert_allclose(g2["coeffs"][:, 0], t, atol=1e-6)
    # duplicate column (rank-deficient library): objective parity, twins sum to the unique answer
    A = rng.uniform(0.1, 0.9, (L, 4)).astype(np.float32)
    Ad = np.concatenate([A, A[:, :1]], axis=1)
    a0 = np.array([0.5, 0.2, 0.3, 0.0])
    Y = (A.astype(np.float64) @ a0 + 0.01 * rng.standard_normal((20, L))).astype(np.float32)
    gd = run_gpu(lm, Ad, Y, None)
    ou = oracle.solve(A, Y)
    np.testing.assert_allclose(gd["coeffs"][:, 0] + gd["coeffs"][:, 4], ou.coeffs[:, 0], atol=1e-5)
    np.testing.assert_allclose(gd["resid"], ou.resid, rtol=1e-5)
    # R > L (LINMIN_WARN_RANK_DEFICIENT): objective parity only
    Aw = rng.uniform(0.1, 0.9, (4, 6)).astype(np.float32)
    Yw = rng.uniform(0.1, 0.9, (16, 4)).astype(np.float32)
    gw = run_gpu(lm, Aw, Yw, None)
    assert gw["status"] == lm.WARN_RANK_DEFICIENT
    ow = oracle.solve(Aw, Yw)
    Fg = ((Yw - gw["coeffs"].astype(np.float64) @ Aw.T.astype(np.float64)) ** 2).sum(1)
    Fo = ((Yw - ow.coeffs @ Aw.T.astype(np.float64)) ** 2).sum(1)
    assert (np.abs(Fg - Fo) <= 1e-5 * np.maximum(Fo, 1e-12 * (Yw.astype(np.float64) ** 2).sum(1))).all()
    assert np.abs(gw["coeffs"].sum(1) - 1).max() <= 1e-5 and gw["coeffs"].min() >= 0
    # NaN pixel and bad sigma: flagged, NaN outputs, neighbours untouched
    Yn = Y.copy(); Yn[3, 2] = np.nan
    S = np.full((20, L), 0.01, np.float32); S[5, 1] = 0.0
    gn = run_gpu(lm, A, Yn, S)
    gref = run_gpu(lm, A, Y, np.full((20, L), 0.01, np.float32))
    assert np.isnan(gn["coeffs"][3]).all() and np.isnan(gn["resid"][3]) and (gn["info"][3] & lm.INFO_NONFINITE_INPUT)
    assert np.isnan(gn["coeff_sigma"][5]).all() and (gn["info"][5] & lm.INFO_BAD_SIGMA)
    assert np.array_equal(gn["coeffs"][5], gref["coeffs"][5])
    assert np.array_equal(gn["coeffs"][4], gref["coeffs"][4]) and np.array_equal(gn["coeff_sigma"][4], gref["coeff_sigma"][4])
    # non-finite library: refused by linmin_library_create (status); the one-shot call, which never waits for the
    # device, poisons its outputs instead (NaN, LINMIN_INFO_LIBRARY_NONFINITE)
    Ab = A.copy(); Ab[0, 0] = np.inf
    with pytest.raises(lm.LinminError) as e:
        lm.library_create(torch.from_numpy(Ab).to("cuda:0"))
    assert e.value.code == lm.ERR_LIBRARY_NONFINITE
    gb = run_gpu(lm, Ab, Y, np.full((20, L), 0.01, np.float32))
    assert np.isnan(gb["coeffs"]).all() and np.isnan(gb["coeff_sigma"]).all() and np.isnan(gb["resid"]).all()
    assert (gb["info"] == lm.INFO_LIBRARY_NONFINITE).all()
    # same contract for a covariance that is not positive definite on the one-shot path: its own info bit
    Cbad = -np.eye(L, dtype=np.float32)
    t = lambda x: torch.from_numpy(x).to("cuda:0")
    with pytest.raises(lm.LinminError) as e:
        lm.library_create(t(A), cov=t(Cbad))
    assert e.value.code == lm.ERR_COVARIANCE
    for lib_arr, word in ((A, lm.INFO_COVARIANCE), (Ab, lm.INFO_COVARIANCE | lm.INFO_LIBRARY_NONFINITE)):
        c, s, r, info, _ = lm.unmix(t(lib_arr), t(Y), None, cov=t(Cbad))
        torch.cuda.synchronize()
        assert torch.isnan(c).all() and torch.isnan(s).all() and torch.isnan(r).all()
        assert (info.cpu().numpy() == word).all()
    sdiag = np.full(L, 0.01, np.float32); sdiag[2] = 0.0            # a zero noise std: diagonal covariance refused too
    c, s, r, info, _ = lm.unmix(t(A), t(Y), None, cov=t(sdiag))
    torch.cuda.synchronize()
    assert torch.isnan(c).all() and (info.cpu().numpy() == lm.INFO_COVARIANCE).all()
    # a zero endmember (what a sum-lower-than-one slack column looks like): results stay on the simplex
    Az = np.concatenate([A, np.zeros((L, 1), np.float32)], axis=1)
    gz = run_gpu(lm, Az, Y, None)
    oz = oracle.solve(Az, Y)
    assert np.abs(gz["coeffs"].sum(1) - 1).max() <= 1e-5 and gz["coeffs"].min() >= 0
    np.testing.assert_allclose(gz["resid"], oz.resid, rtol=1e-5)
    # ... element by element: coefficients, uncertainties, residual within the parity tolerances
    from parity import check_parity
    check_parity(Az, Y, np.ones(L, np.float32), gz, oz, label="zero endmember")
    assert (oz.coeffs[:, -1] > 0).any() and (oz.coeffs[:, -1] == 0).any()     # the slack is used by some pixels only


def test_boundary_is_asynchronous_graph_capturable_and_stream_safe(lm):
    """the device entry points enqueue and return.  Stream capture fails on any hidden
    synchronisation or host read, so capturing linmin_unmix_lib AND the one-shot linmin_unmix (precompute included)
    into CUDA graphs and replaying them proves it.  Then: a handle created on one stream, used on another and
    destroyed at once -- the frees must wait for the other stream's kernels."""
    from paper_1402_2518_b200.synth import make_workload
    w = make_workload("omega", N=5000)
    dev = torch.device("cuda:0")
    A, Y, S = (torch.from_numpy(x).to(dev) for x in (w.A, w.Y, w.sigma))
    ref = lm.unmix(A, Y, S)
    torch.cuda.synchronize()
    lib = lm.library_create(A)
    outs = dict(coeffs=torch.zeros((w.N, w.R), device=dev), coeff_sigma=torch.zeros((w.N, w.R), device=dev),
                resid=torch.zeros((w.N,), device=dev), info=torch.zeros((w.N,), dtype=torch.int32, device=dev))
    outs1 = {k: torch.zeros_like(v) for k, v in outs.items()}
    lm.unmix_lib(lib, Y, S, out=outs)            # warm-up outside the capture (function attributes, pool growth)
    torch.cuda.synchronize()
    for o in (outs, outs1):
        for v in o.values():
            v.zero_()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g):
        lm.unmix_lib(lib, Y, S, out=outs)
        lm.unmix(A, Y, S, out=outs1)
    for _ in range(2):
        g.replay()
    torch.cuda.synchronize()
    for o in (outs, outs1):
        assert torch.equal(o["coeffs"], ref[0]) and torch.equal(o["coeff_sigma"], ref[1])
        assert torch.equal(o["resid"], ref[2]) and torch.equal(o["info"], ref[3])
    del g
    lib.destroy()
    # handle used on a second stream, destroyed immediately; then the pool is churned on the creation stream
    side = torch.cuda.Stream()
    lib2 = lm.library_create(A)
    wbig = make_workload("omega", N=131072)
    Yb, Sb = torch.from_numpy(wbig.Y).to(dev), torch.from_numpy(wbig.sigma).to(dev)
    refb = lm.unmix_lib(lib2, Yb, Sb)
    torch.cuda.synchronize()
    with torch.cuda.stream(side):
        got = lm.unmix_lib(lib2, Yb, Sb)
    lib2.destroy()                                # kernels of `side` are still running
    junk = [lm.library_create(torch.rand((w.L, w.R), device=dev) + 0.1) for _ in range(4)]    # reuses freed blocks
    torch.cuda.synchronize()
    assert torch.equal(got[0], refb[0]) and torch.equal(got[1], refb[1]) and torch.equal(got[2], refb[2])
    for j in junk:
        j.destroy()
    # argument marshalling guards of the binding (wrong shapes / dtypes never reach the C ABI)
    with pytest.raises(ValueError):
        lm.unmix(A, Y[:, :100].contiguous(), None)
    with pytest.raises(ValueError):
        lm.unmix(A, Y, S, out=dict(info=torch.zeros((w.N,), dtype=torch.int64, device=dev)))
    with pytest.raises(ValueError):
        lm.unmix_host(w.A, w.Y, w.sigma[:, :64].copy())


def test_large_supports_take_the_overflow_path(lm):
    """Supports beyond finish_sweep's cap (16 members) are finished by the one-warp-per-pixel kernel:
    dense abundances on a well-conditioned random library, mixed with sparse pixels."""
    import oracle
    from parity import check_parity
    rng = np.random.default_rng(77)
    L, R, N = 128, 32, 600
    A = rng.uniform(0.1, 0.9, (L, R)).astype(np.float32)
    a0 = rng.dirichlet(5.0 * np.ones(R), size=N)
    sparse = rng.uniform(size=N) < 0.5
    for p in np.nonzero(sparse)[0]:
        a0[p] = 0.0
        kk = rng.integers(1, 6)
        a0[p, rng.choice(R, kk, replace=False)] = rng.dirichlet(np.ones(kk))
    sig = rng.uniform(0.0005, 0.002, (N, L)).astype(np.float32)
    Y = (a0 @ A.astype(np.float64).T + sig * rng.standard_normal((N, L))).astype(np.float32)
    g = run_gpu(lm, A, Y, sig)
    ora = oracle.solve(A, Y, sig)
    ksz = (g["info"] >> 24) & 0xff
    assert (ksz > 16).sum() > 100 and (ksz <= 16).sum() > 100
    print(check_parity(A, Y, sig, g, ora, label="overflow"))


def test_scale_and_offset_invariance(lm):
    """R13: relative stopping rules -> (cA, cy) gives the same coefficients; offset invariance (eq. 4)."""
    from paper_1402_2518_b200.synth import make_workload
    w = make_workload("omega", N=512)
    g = run_gpu(lm, w.A, w.Y, w.sigma)
    gs = run_gpu(lm, 4 * w.A, 4 * w.Y, 4 * w.sigma)
    np.testing.assert_allclose(gs["coeffs"], g["coeffs"], atol=2e-6)
    np.testing.assert_allclose(gs["resid"], 4 * g["resid"], rtol=1e-5)
    it, its = (g["info"] >> 8) & 0xff, (gs["info"] >> 8) & 0xff
    assert np.abs(it.astype(int) - its.astype(int)).max() <= 1
    go = run_gpu(lm, w.A + np.float32(0.25), w.Y + np.float32(0.25), w.sigma)
    np.testing.assert_allclose(go["coeffs"], g["coeffs"], atol=2e-5)


@pytest.mark.parametrize("L,R", [(110, 36), (56, 36), (33, 5), (200, 100), (110, 32), (240, 20), (400, 12), (512, 32),
                                 (150, 65), (260, 129), (240, 255)])
def test_odd_sizes(lm, L, R):
    """The paper's own sizes (110 or 56 channels, 36 endmembers) and others."""
    import oracle
    from parity import check_parity
    rng = np.random.default_rng(L * 1000 + R)
    lam = np.linspace(1.0, 2.5, L)
    cols = []
    for _ in range(R - 2):
        c0, c1 = rng.uniform(0.2, 0.6, 2)
        s = c0 + (c1 - c0) * (lam - 1.0) / 1.5
        for _ in range(rng.integers(1, 4)):
            s = s * (1 - rng.uniform(0.05, 0.4) * np.exp(-0.5 * ((lam - rng.uniform(1.0, 2.5)) / rng.uniform(0.01, 0.06)) ** 2))
        cols.append(s)
    cols += [np.ones(L), (lam - 1.0) / 1.5]
    A = np.stack(cols, 1).astype(np.float32)
    N = 777
    a0 = np.zeros((N, R))
    for p in range(N):
        k = rng.integers(1, 5)
        a0[p, rng.choice(R, k, replace=False)] = rng.dirichlet(0.3 * np.ones(k))
    sig = rng.uniform(0.002, 0.01, (N, L)).astype(np.float32)
    Y = (a0 @ A.astype(np.float64).T + sig * rng.standard_normal((N, L))).astype(np.float32)
    g = run_gpu(lm, A, Y, sig)
    ora = oracle.solve(A, Y, sig)
    print(check_parity(A, Y, sig, g, ora, label=f"L{L}R{R}"))


@pytest.mark.parametrize("name,N", [("omega", 40000), ("crism", 6000), ("tiny", 1000), ("stress", 900)])
def test_results_do_not_depend_on_neighbours_or_repeats(lm, name, N):
    """Stands in for racecheck (compute-sanitizer is closed on this pool): every pixel is an independent
    problem, so its outputs must be bit-identical run to run, under a random permutation of
    the pixels (other pixels share its warp, its 32-pixel chunk and its shared-memory scratch) and when it
    is solved alone in a shorter batch.  A missing barrier or a read of another pixel's scratch breaks this."""
    from paper_1402_2518_b200.synth import make_workload
    w = make_workload(name, N=N)
    g = run_gpu(lm, w.A, w.Y, w.sigma)
    g2 = run_gpu(lm, w.A, w.Y, w.sigma)
    rng = np.random.Generator(np.random.PCG64(7))
    perm = rng.permutation(N)
    gp = run_gpu(lm, w.A, np.ascontiguousarray(w.Y[perm]), np.ascontiguousarray(w.sigma[perm]))
    m = 777 if N > 777 else N // 2
    gs = run_gpu(lm, w.A, w.Y[:m], w.sigma[:m])
    for key in ("coeffs", "coeff_sigma", "resid"):
        assert np.array_equal(g[key], g2[key], equal_nan=True), f"{key}: run-to-run"
        assert np.array_equal(g[key][perm], gp[key], equal_nan=True), f"{key}: permutation"
        assert np.array_equal(g[key][:m], gs[key], equal_nan=True), f"{key}: shorter batch"
    it, it_p = (g["info"] >> 8) & 0xff, (gp["info"] >> 8) & 0xff
    assert np.array_equal(it[perm], it_p)


def test_throughput_full_size_sampled_and_properties(lm):
    """BASELINE.json configs[4] at its FULL size (128 cubes = 16,777,216 pixels, per-pixel sigma), in the launch
    configuration bench.py times: every 16th pixel (1,048,576 pixels) element by element against the
    oracle, and properties that hold at any size on ALL pixels (simplex feasibility, exact zeros off the support,
    finite outputs).  Also the multi-chunk host path (linmin_unmix_host, 5 chunks) bit for bit against the device path."""
    import os
    import sys
    import oracle
    from parity import check_parity
    sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
    from bench import CUBE, gen_cubes
    n_cubes, L, R = 128, 128, 32
    N = n_cubes * CUBE
    Yh = torch.empty((N, L), dtype=torch.float32)
    Sh = torch.empty((N, L), dtype=torch.float32)
    A = gen_cubes(0, n_cubes, Yh.numpy(), Sh.numpy(), max(1, (os.cpu_count() or 8)))
    dev = torch.device("cuda:0")
    Ad, Yd, Sd = torch.from_numpy(A).to(dev), Yh.to(dev), Sh.to(dev)
    c, s, r, info, status = lm.unmix(Ad, Yd, Sd)
    torch.cuda.synchronize()
    # properties on every pixel (computed on the device by torch: plumbing, not the product)
    assert bool(torch.isfinite(c).all()) and bool(torch.isfinite(s).all()) and bool(torch.isfinite(r).all())
    assert float((c.sum(1) - 1.0).abs().max()) <= 1e-5
    assert float(c.min()) >= 0.0
    assert bool(((c == 0) == (s == 0)).logical_or(c.gt(0).sum(1, keepdim=True) == 1).all())   # sigma is 0 exactly off the support (and all 0 when k = 1)
    assert float(r.min()) > 0.0
    flags = info & 0xff
    assert int(((flags & 0x10) != 0).sum()) == 0            # no finish fallback
    assert int(((flags & 0x04) != 0).sum()) == 0            # no non-finite input
    sel = np.arange(0, N, 16)
    assert len(sel) == 1048576
    sel_t = torch.from_numpy(sel).to(dev)
    g = dict(coeffs=c[sel_t].cpu().numpy(), coeff_sigma=s[sel_t].cpu().numpy(), resid=r[sel_t].cpu().numpy())
    Ys, Ss = Yh.numpy()[sel], Sh.numpy()[sel]
    ora = oracle.solve(A, Ys, Ss)
    print(check_parity(A, Ys, Ss, g, ora, label="throughput-full"))
    # host entry point over more than three chunks of its pipeline (2^18 pixels each), ragged tail included
    nh = 4 * (1 << 18) + 1003
    ch, sh, rh, ih, _ = lm.unmix_host(A, Yh[:nh], Sh[:nh], want_info=True)
    assert np.array_equal(ch.numpy(), c[:nh].cpu().numpy())
    assert np.array_equal(sh.numpy(), s[:nh].cpu().numpy())
    assert np.array_equal(rh.numpy(), r[:nh].cpu().numpy())
    assert np.array_equal(ih.numpy(), info[:nh].cpu().numpy())


def test_ipls_converges_in_few_iterations(lm):
    """Guards the start point and the stopping rule of the IPLS kernels: on the OMEGA-like and CRISM-like
    cubes the mean iteration count stays near the measured 5.9 / 7.5 and (almost) every pixel converges."""
    from paper_1402_2518_b200.synth import make_workload
    for name, N, bound in (("omega", 32768, 7.0), ("crism", 4096, 9.0), ("tiny", 1000, 6.0)):
        w = make_workload(name, N=N)
        g = run_gpu(lm, w.A, w.Y, w.sigma)
        it = (g["info"] >> 8) & 0xff
        conv = (g["info"] & 0x01) != 0
        assert it.mean() <= bound, (name, it.mean())
        assert conv.mean() >= 0.999, (name, conv.mean())
    lm.trim_memory()      # hands the cached staging memory back; the next call allocates again
    w = make_workload("tiny", N=64)
    run_gpu(lm, w.A, w.Y, w.sigma)
