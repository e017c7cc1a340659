"""Host-side checks that need no GPU: the C-ABI library builds, loads and exports every symbol
include/linmin.h declares; argument validation; loud failure without a device."""
import ctypes
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_1402_2518_b200 import build, linmin
    build.build_library()
    return linmin.load()


def declared_functions():
    src = open(os.path.join(ROOT, "include", "linmin.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(linmin_[a-z_0-9]+)\s*\(", src)))


def test_exports_match_header(lib):
    from paper_1402_2518_b200 import linmin
    names = declared_functions()
    assert set(names) == set(linmin.EXPORTS), (names, linmin.EXPORTS)
    for n in names:
        assert getattr(lib, n) is not None


def test_version_and_strerror(lib):
    from paper_1402_2518_b200 import linmin
    assert linmin.version() == 200
    for code in [0, -1, -2, -3, -4, -5, -6, -7, -8, 1]:
        assert "unknown" not in linmin.strerror(code)
    assert "unknown" in linmin.strerror(12345)


def test_opts_struct_layout(lib):
    from paper_1402_2518_b200 import linmin
    # must match include/linmin.h: 4+pad4, 8, 8, 8, 4, 4, 4, 4, 4 +pad4, 8, 4, 4, 8 = 80 bytes
    assert ctypes.sizeof(linmin.LinminOpts) == 80
    assert linmin.LinminOpts.cov.offset == 72
    assert linmin.LinminOpts.info_out.offset == 56


def test_argument_validation_without_device(lib):
    from paper_1402_2518_b200 import linmin
    one = ctypes.c_void_p(16)   # never dereferenced: validation fails first
    o = linmin._make_opts()
    f = lib.linmin_unmix
    assert f(None, one, None, 1, 4, 2, ctypes.byref(o), one, None, None) == linmin.ERR_INVALID_ARGUMENT
    assert f(one, one, None, -1, 4, 2, ctypes.byref(o), one, None, None) == linmin.ERR_INVALID_ARGUMENT
    assert f(one, one, None, 1, 0, 2, ctypes.byref(o), one, None, None) == linmin.ERR_INVALID_ARGUMENT
    assert f(one, one, None, 1, 4, 0, ctypes.byref(o), one, None, None) == linmin.ERR_INVALID_ARGUMENT
    assert f(one, one, None, 1, 4, 257, ctypes.byref(o), one, None, None) == linmin.ERR_UNSUPPORTED_SIZE
    assert f(one, one, None, 1, 513, 2, ctypes.byref(o), one, None, None) == linmin.ERR_UNSUPPORTED_SIZE
    assert f(one, None, None, 1, 4, 2, ctypes.byref(o), one, None, None) == linmin.ERR_INVALID_ARGUMENT
    assert f(one, one, None, 1, 4, 2, ctypes.byref(o), None, None, None) == linmin.ERR_INVALID_ARGUMENT
    bad = linmin._make_opts(); bad.struct_size = 8
    assert f(one, one, None, 1, 4, 2, ctypes.byref(bad), one, None, None) == linmin.ERR_INVALID_ARGUMENT
    for kw, code in [(dict(ldY=3), -1), (dict(sigma_pixel_stride=2), -1), (dict(max_iter=256), -1),
                     (dict(gap_tol=-1.0), -1), (dict(constraint=7), -1), (dict(constraint=-1), -1),
                     (dict(weighting=1), -1), (dict(weighting=2), -1),       # a weighting without opts->cov
                     (dict(weighting=9), -1)]:
        ob = linmin._make_opts(**kw)
        assert f(one, one, None, 1, 4, 2, ctypes.byref(ob), one, None, None) == code, kw
    h = ctypes.c_void_p()
    assert lib.linmin_library_create(None, 4, 2, None, ctypes.byref(h)) == linmin.ERR_INVALID_ARGUMENT
    assert lib.linmin_library_create(one, 4, 2, None, None) == linmin.ERR_INVALID_ARGUMENT
    assert lib.linmin_unmix_lib(None, one, None, 1, None, one, None, None) == linmin.ERR_INVALID_ARGUMENT
    lib.linmin_library_destroy(None)    # no-op


def test_fails_loudly_without_cuda_device(lib):
    """No CPU fallback: with valid arguments and no GPU the host entry point reports a CUDA error."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    from paper_1402_2518_b200 import linmin
    A = np.random.default_rng(0).uniform(0.1, 1, (8, 3)).astype(np.float32)
    Y = np.random.default_rng(1).uniform(0.1, 1, (5, 8)).astype(np.float32)
    with pytest.raises(linmin.LinminError) as e:
        linmin.unmix_host(A, Y)
    assert e.value.code == linmin.ERR_CUDA


def test_product_does_not_import_oracle():
    """The product path must never route through oracle/ (or any CPU solver)."""
    pkg = os.path.join(ROOT, "paper_1402_2518_b200")
    for dirpath, _, files in os.walk(pkg):
        for fn in files:
            if fn.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, fn)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", txt, flags=re.M), fn
                assert "linmin_oracle" not in txt, fn
    for fn in os.listdir(os.path.join(ROOT, "oracle")):
        if fn.endswith((".py", ".c")):
            txt = open(os.path.join(ROOT, "oracle", fn)).read()
            assert not re.search(r"^\s*(from|import)\s+paper_1402_2518_b200", txt, flags=re.M), fn


def test_trim_memory_without_pools(lib):
    # no pool exists before the first GPU call: trimming is a no-op that reports success
    assert lib.linmin_trim_memory() == 0
