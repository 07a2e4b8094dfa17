"""rips_sort_u64_static: the sort primitive for callers that must not allocate (its scratch is a static device array
inside the library instead of a cudaMalloc per call; include/rips.h).  Checked against the existing path
(rips_sort_u64) on two calls in a row -- the second one smaller than the first and on other bits, so it runs on the
scratch the first one left behind -- for exact equality (records are integers: the tolerance of every test here is
zero), and against NumPy's stable argsort.  Collected last on purpose (the suite runs with pytest -x)."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def R():
    import torch
    assert torch.cuda.is_available(), "the gpu tests need a CUDA device"
    from paper_2003_07989_b200 import rips
    rips.use_library(None)          # the product library, whatever an earlier test loaded
    return rips


def _reference(R, a, lo, hi):
    import torch
    t = torch.from_numpy(a.copy()).cuda()
    R.rips_sort_u64(t, lo, hi)       # the existing path: cudaMalloc'ed scratch
    return t.cpu().numpy()


def test_static_scratch_sort_matches_the_allocating_sort(R):
    import torch
    rng = np.random.default_rng(17)
    # two calls in a row on the shared scratch: 1.5e6 records on 24 bits (three passes, 293 tiles), then 70,001
    # records on other bits (two passes, 14 tiles), then a third with all keys equal (stability)
    cases = [(1_500_000, 3, 27), (70_001, 40, 53), (300_007, 0, 8)]
    for i, (n, lo, hi) in enumerate(cases):
        a = rng.integers(0, 1 << 62, n, dtype=np.int64)
        if i == 2:
            a = (a & ~np.int64(0xff)) | np.int64(5)          # one digit value: must come back untouched
        want = _reference(R, a, lo, hi)
        t = torch.from_numpy(a.copy()).cuda()
        tmp = torch.empty_like(t)
        R.rips_sort_u64_static(t, tmp, lo, hi)
        torch.cuda.synchronize()
        got = t.cpu().numpy()
        assert np.array_equal(got, want), (n, lo, hi)
        u = a.view(np.uint64)
        key = (u >> np.uint64(lo)) & np.uint64((1 << (hi - lo)) - 1)
        assert np.array_equal(got.view(np.uint64), u[np.argsort(key, kind="stable")]), (n, lo, hi)


def test_static_scratch_sort_rejects_what_the_array_cannot_hold(R):
    import torch
    n = (1 << 22) + 1
    t = torch.zeros(n, dtype=torch.int64, device="cuda")
    tmp = torch.empty_like(t)
    with pytest.raises(R.RipsError) as e:
        R.rips_sort_u64_static(t, tmp, 0, 16)
    assert e.value.code == R.RIPS_EINVAL and "maximum" in str(e.value)
    # the largest size it takes
    a = np.random.default_rng(3).integers(0, 1 << 40, 1 << 22, dtype=np.int64)
    t = torch.from_numpy(a.copy()).cuda()
    R.rips_sort_u64_static(t, tmp, 0, 16)
    torch.cuda.synchronize()
    u = a.view(np.uint64)
    assert np.array_equal(t.cpu().numpy().view(np.uint64), u[np.argsort(u & np.uint64(0xffff), kind="stable")])
