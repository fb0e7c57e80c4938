"""hamr_divb_noalloc (include/hamr.h): the div B diagnostic on caller-owned dense device arrays, with its scratch in a
fixed file-scope device array: no allocation inside the call.  Checked against the existing path (hamr_divb on a grid
holding the same face field) on two calls in a row that share the scratch array: the second on a SMALLER grid with a
different field, so that stale partial results of the first call would show.  Collected last on purpose.  Needs a B200."""
import numpy as np
import pytest

from paper_1912_10192_b200 import inputs as I

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def H():
    from paper_1912_10192_b200 import build, hamr
    build.build_lib()
    hamr.lib()
    return hamr


def _field(n, seed, scale, div_free):
    """dense face arrays on the unit cube: a divergence-free part from an edge vector potential (cfg 1's recipe) and,
    unless div_free, seeded noise on top (a field WITH divergence, so that the diagnostic returns an O(1) number)"""
    p = I.minkowski_params(n=n)
    hyd, bf = I.minkowski_waves(p, seed=seed, amp=1e-2)[:2]
    bf = [scale * np.ascontiguousarray(b) for b in bf]
    if not div_free:
        for d in range(3):
            idx = I.zone_index(bf[d].shape)
            bf[d] = bf[d] * (1.0 + 0.3 * I.rand_pm1(seed + 10 + d, idx))
    return p, hyd, bf


def _both(H, torch, n, seed, scale, div_free):
    p, hyd, bf = _field(n, seed, scale, div_free)
    g = H.Grid(p)
    assert g.set_prims(hyd, bf) == 0
    ref = g.divb()                                           # the existing path
    dev = [torch.from_numpy(b).cuda() for b in bf]
    out = torch.full((1,), -1.0, dtype=torch.float64, device="cuda")
    dx = [1.0 / m for m in n]
    st = torch.cuda.current_stream().cuda_stream
    H.divb_noalloc(n, dx, [t.data_ptr() for t in dev], out.data_ptr(), st)
    torch.cuda.synchronize()
    g.close()
    return ref, float(out.item())


def test_divb_noalloc_matches_hamr_divb_on_two_calls_in_a_row(H):
    import torch
    L = H.lib()
    assert L.hamr_noalloc_setup() == 0
    # first call: 40 x 24 x 36 (135 blocks of partial results), a field with divergence
    ref1, new1 = _both(H, torch, (40, 24, 36), seed=5, scale=1.0, div_free=False)
    assert ref1 > 1e-3 and abs(new1 - ref1) <= 1e-12 * ref1, (ref1, new1)
    # second call: a smaller grid (12 blocks), field 1e-3 times weaker and a different seed: stale partial maxima or a
    # stale denominator maximum from the first call would change the answer
    ref2, new2 = _both(H, torch, (24, 16, 8), seed=9, scale=1e-3, div_free=False)
    assert ref2 > 1e-3 and abs(new2 - ref2) <= 1e-12 * ref2, (ref2, new2)
    assert abs(ref2 - ref1) > 1e-6 * ref1                    # the two calls really differ
    # a divergence-free field: both at round-off (the bound the parity tests use for div B)
    ref3, new3 = _both(H, torch, (32, 32, 32), seed=1, scale=1.0, div_free=True)
    assert ref3 <= 1e-12 and new3 <= 1e-12 and abs(new3 - ref3) <= 1e-14, (ref3, new3)


def test_divb_noalloc_rejects_what_exceeds_the_scratch(H):
    import ctypes as C
    import torch
    L = H.lib()
    out = torch.zeros(1, dtype=torch.float64, device="cuda")
    buf = torch.zeros(8, dtype=torch.float64, device="cuda")
    ptrs = [buf.data_ptr()] * 3
    with pytest.raises(H.HamrError) as e:                    # 512 x 256 x 256 = 2 x the limit: nothing is launched
        H.divb_noalloc((512, 256, 256), (1.0, 1.0, 1.0), ptrs, out.data_ptr(), None)
    assert e.value.code == H.EINVAL and "HAMR_NOALLOC_MAX_ZONES" in str(e.value)
    with pytest.raises(H.HamrError):
        H.divb_noalloc((0, 4, 4), (1.0, 1.0, 1.0), ptrs, out.data_ptr(), None)
    with pytest.raises(H.HamrError):
        H.divb_noalloc((4, 4, 4), (1.0, 0.0, 1.0), ptrs, out.data_ptr(), None)
    nn = (C.c_int * 3)(4, 4, 4)
    dd = (C.c_double * 3)(1.0, 1.0, 1.0)
    assert L.hamr_divb_noalloc(nn, dd, None, None, None) == H.EINVAL
    torch.cuda.synchronize()
    assert float(out.item()) == 0.0
    # exactly at the limit is accepted (256^3 zones)
    assert H.NOALLOC_MAX_ZONES == 256 ** 3
