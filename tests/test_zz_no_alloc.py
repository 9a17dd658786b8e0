"""ib_bin_sort_static (include/ibcouple.h): the bin sort for callers that must not allocate.

Its scratch is a fixed file-scope device array of the library, so it has a size limit and all calls share the
array.  Checked here: bit-identical keys and permutation to the existing path (ib_bin_sort, integer work: the
bar is equality) on two calls in a row -- a large cloud first, then a smaller one on another grid, so the second
call runs over the first call's leftovers -- the limit, the latch of a non-finite coordinate and its clearing.
The file is named so that pytest collects it last.
"""
import ctypes

import numpy as np
import pytest

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def ib():
    import torch
    assert torch.cuda.is_available(), "gpu tests need a CUDA device"
    from paper_2503_22695_b200 import build, ibcouple
    build.build()
    ibcouple.lib()
    return ibcouple


def _t(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _cloud(n, h, org, P, seed):
    rng = np.random.default_rng(seed)
    xp = np.asarray(org)[:, None] + rng.uniform(-0.2, 1.2, (3, P)) * (np.array(n) * h)[:, None]
    if P > 100:
        xp[:, :50] = np.asarray(org)[:, None] + rng.integers(0, 8, (3, 50)) * h     # exact cell boundaries
        xp[:, 50:100] = xp[:, 100:101]                                              # many ties
    return xp


def _existing_path(ib, n, h, org, xp):
    import torch
    P = xp.shape[1]
    ctx = ib.Context(*n, h, org, np.zeros((0, 8), np.int32), np.zeros((3, 0)), None, None, None, [])
    key = torch.empty(P, dtype=torch.int64, device="cuda")
    perm = torch.empty(P, dtype=torch.int32, device="cuda")
    ctx.ib_bin_sort(_t(xp) if P else None, P, key, perm)
    ctx.check()
    out = key.cpu().numpy(), perm.cpu().numpy()
    ctx.close()
    return out


def test_static_bin_sort_matches_the_existing_path_on_two_calls_in_a_row(ib):
    import torch
    cases = [((64, 64, 64), 0.25, (-1.0, 0.5, 2.0), ib.BIN_SORT_STATIC_MAX_POINTS, 11),     # the limit itself
             ((16, 8, 24), 0.125, (0.0, -3.0, 1.0), 5000, 12),                              # smaller, other grid: stale scratch
             ((16, 8, 24), 0.125, (0.0, -3.0, 1.0), 1, 13),
             ((16, 8, 24), 0.125, (0.0, -3.0, 1.0), 0, 14)]
    for n, h, org, P, seed in cases:
        xp = _cloud(n, h, org, P, seed)
        k_ref, p_ref = _existing_path(ib, n, h, org, xp)
        key = torch.full((P,), -1, dtype=torch.int64, device="cuda")
        perm = torch.full((P,), -1, dtype=torch.int32, device="cuda")
        ib.ib_bin_sort_static((*n, h, org, 1), _t(xp) if P else None, P, key, perm, check=1)
        assert np.array_equal(key.cpu().numpy(), k_ref), (n, P)
        assert np.array_equal(perm.cpu().numpy(), p_ref), (n, P)
        if P > 1:
            assert np.array_equal(np.sort(p_ref), np.arange(P))         # the reference itself is a permutation
    # asynchronous form (check = 0) on a side stream, outputs optional
    n, h, org, P, seed = cases[1]
    xp = _cloud(n, h, org, P, seed)
    k_ref, p_ref = _existing_path(ib, n, h, org, xp)
    x_d = _t(xp)
    perm = torch.empty(P, dtype=torch.int32, device="cuda")
    st = torch.cuda.Stream()
    st.wait_stream(torch.cuda.current_stream())
    ib.ib_bin_sort_static((*n, h, org, 1), x_d, P, None, perm, check=0, stream=st)
    st.synchronize()
    assert np.array_equal(perm.cpu().numpy(), p_ref)


def test_static_bin_sort_limit_arguments_and_latch(ib):
    import torch
    n, h, org = (16, 8, 24), 0.125, (0.0, -3.0, 1.0)
    P = 300
    xp = _cloud(n, h, org, P, 21)
    x_d = _t(xp)
    key = torch.empty(P, dtype=torch.int64, device="cuda")
    perm = torch.empty(P, dtype=torch.int32, device="cuda")
    # beyond the limit: a clear error, nothing enqueued (the pointers are never touched)
    with pytest.raises(ib.IbError) as e:
        ib.ib_bin_sort_static((*n, h, org, 1), x_d, ib.BIN_SORT_STATIC_MAX_POINTS + 1, key, perm)
    assert e.value.code == 8 and "IB_ERR_TOO_LARGE" in str(e.value)
    L = ib.lib()
    g = ib.GridDesc(30, 8, 24, h, 0, 0, 0, 1)                   # nx not a multiple of 8
    assert L.ib_bin_sort_static(ctypes.byref(g), None, 0, None, None, 0, None) == 1
    g = ib.GridDesc(16, 8, 24, h, 0, 0, 0, 1)
    assert L.ib_bin_sort_static(ctypes.byref(g), None, 5, None, None, 0, None) == 1     # P > 0 without points
    assert L.ib_bin_sort_static(None, None, 0, None, None, 0, None) == 1
    # a NaN coordinate is latched, reported with check != 0, and the latch is cleared by the next call
    xn = xp.copy()
    xn[1, 7] = np.nan
    with pytest.raises(ib.IbError) as e:
        ib.ib_bin_sort_static((*n, h, org, 1), _t(xn), P, key, perm, check=1)
    assert e.value.code == 6
    ib.ib_bin_sort_static((*n, h, org, 1), x_d, P, key, perm, check=1)
    k_ref, p_ref = _existing_path(ib, n, h, org, xp)
    assert np.array_equal(key.cpu().numpy(), k_ref) and np.array_equal(perm.cpu().numpy(), p_ref)
