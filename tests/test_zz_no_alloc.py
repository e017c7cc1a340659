"""linmin_detection_thresholds_static: the eq. 8 thresholds for callers that cannot let the
library allocate device memory -- an application that gave the whole GPU to its own arena, or a latency-bound loop
that cannot take an allocation's stall.  Its partial sums live in one fixed array inside liblinmin.so, shared by every
call on a device and still holding the previous call's contents; so the check is made on TWO calls in a row, on
different data (the second with fewer blocks than the first, so stale slots lie right behind the ones it uses),
each against linmin_detection_thresholds on the same arrays.

This file is named to be collected last: `pytest -x` stops at the first failure, and a failure here must not hide the
parity tests.  It passes alone in a fresh process (the first call on the device does the address look-up) and after
the other tests."""
import ctypes

import numpy as np
import pytest
import torch

pytestmark = pytest.mark.gpu

# the tolerance tests/test_gpu_next.py holds linmin_detection_thresholds to: the two paths add the same fp64 terms
# in a different block order, so their float32 results agree to rounding
RTOL, ATOL = 2e-6, 1e-9


@pytest.fixture(scope="module")
def lm():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_1402_2518_b200 import build, linmin
    build.build_library()
    linmin.load()
    return linmin


def labelled_set(n, r, seed, dev):
    """Estimated coefficients with exact zeros (as the finish returns them) and a presence label per entry."""
    g = np.random.default_rng(seed)
    present = g.random((n, r)) < 0.08
    c = np.where(present, 0.05 + 0.3 * g.random((n, r)), 0.0)
    false_pos = (~present) & (g.random((n, r)) < 0.1)
    c = np.where(false_pos, 0.02 * g.random((n, r)), c)
    c[present & (g.random((n, r)) < 0.05)] = 0.0            # missed detections
    return torch.from_numpy(c.astype(np.float32)).to(dev), torch.from_numpy(present).to(dev)


def test_static_scratch_matches_the_pooled_path_on_two_calls_in_a_row(lm):
    dev = torch.device("cuda:0")
    # first call: many blocks (every slot of the array written); second: a few pixels of another library size
    for n, r, seed in ((50000, 32, 1), (37, 36, 2)):
        c, present = labelled_set(n, r, seed, dev)
        want = lm.detection_thresholds(c, present)
        out = torch.full((r,), float("nan"), dtype=torch.float32, device=dev)
        got = lm.detection_thresholds_static(c, present, out)
        again = lm.detection_thresholds_static(c, present, torch.empty_like(out))
        torch.cuda.synchronize()
        assert got.data_ptr() == out.data_ptr()
        np.testing.assert_allclose(got.cpu().numpy(), want.cpu().numpy(), rtol=RTOL, atol=ATOL)
        assert torch.equal(got, again)                       # fixed summation order: same data, same bits
        assert np.isfinite(got.cpu().numpy()).all() and float(got.abs().max()) > 0.0


def test_static_scratch_limit_and_arguments(lm):
    dev = torch.device("cuda:0")
    r = lm.STATIC_MAX_R + 1
    c, present = labelled_set(8, r, 3, dev)
    out = torch.zeros(r, dtype=torch.float32, device=dev)
    with pytest.raises(lm.LinminError) as e:
        lm.detection_thresholds_static(c, present, out)
    assert e.value.code == lm.ERR_STATIC_SCRATCH and "64" in str(e.value)
    assert float(out.abs().max()) == 0.0                     # refused before anything was launched
    # the limit itself is served, and so is a set without detections in either class (every threshold is 0)
    c, present = labelled_set(300, lm.STATIC_MAX_R, 4, dev)
    got = lm.detection_thresholds_static(c, present, torch.empty(lm.STATIC_MAX_R, dtype=torch.float32, device=dev))
    np.testing.assert_allclose(got.cpu().numpy(), lm.detection_thresholds(c, present).cpu().numpy(), rtol=RTOL, atol=ATOL)
    none = lm.detection_thresholds_static(torch.zeros_like(c), present, torch.ones(lm.STATIC_MAX_R, dtype=torch.float32, device=dev))
    assert float(none.abs().max()) == 0.0
    one = ctypes.c_void_p(256)                               # never dereferenced: validation fails first
    f = lm.load().linmin_detection_thresholds_static
    assert f(None, one, 1, 4, one, None) == lm.ERR_INVALID_ARGUMENT
    assert f(one, one, -1, 4, one, None) == lm.ERR_INVALID_ARGUMENT
    assert f(one, one, 1, 0, one, None) == lm.ERR_INVALID_ARGUMENT
