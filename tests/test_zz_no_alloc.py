"""hlc2_crossmatch_static (include/hlc2.h): the match with its scratch in a static device array inside the library, for
callers that cannot allocate device memory.  Its output is compared with the existing path's (hlc2_crossmatch with a
caller buffer) on two calls in a row -- the second call finds the first one's contents in the shared array -- on both match
kernels (same grid, two grids); the size limit is checked, and that the call leaves the device's free memory unchanged.

Collected last on purpose (the file name): the suite runs with `pytest -x`."""
import numpy as np
import pytest

import hlc2_synth as S
from tests import parity

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def P():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("gpu tests selected but no CUDA device")
    import paper_2301_07331_b200 as P
    from paper_2301_07331_b200 import build
    build.build()
    return P


def dev(c):
    import torch
    return (torch.from_numpy(c.ra).cuda(), torch.from_numpy(c.dec).cuda(), torch.from_numpy(c.id).cuda())


def rows(oa, ob, os_, n):
    """Result rows in a canonical order (the kernels emit pairs in no fixed order)."""
    a, b, s = oa[:n].cpu().numpy(), ob[:n].cpu().numpy(), os_[:n].cpu().numpy()
    k = np.lexsort((b, a))
    return a[k], b[k], s[k]


def both_paths(P, ia, ib, r, mode, cap):
    import torch
    out = []
    for static in (False, True):
        oa = torch.full((cap,), -7, dtype=torch.int64, device="cuda"); ob = torch.full_like(oa, -7)
        os_ = torch.full((cap,), -7.0, dtype=torch.float64, device="cuda"); cnt = torch.zeros(1, dtype=torch.int64, device="cuda")
        if static:
            P.hlc2_crossmatch_static(ia, ib, r, mode, oa, ob, os_, cnt)
        else:
            P.hlc2_crossmatch(ia, ib, r, mode, oa, ob, os_, cnt)
        torch.cuda.synchronize()
        n = int(cnt.item())
        assert 0 < n <= cap
        out.append(rows(oa, ob, os_, n))
    return out


def assert_same(ref, got):
    assert len(ref[0]) == len(got[0])
    assert np.array_equal(ref[0], got[0]) and np.array_equal(ref[1], got[1])          # ids: bit-exact
    assert np.max(np.abs(ref[2] - got[2])) <= parity.TOL_SEP                            # separations (arcsec)


@pytest.mark.parametrize("grid", ["same", "two"])
def test_static_scratch_matches_the_caller_buffer_path_twice_in_a_row(P, grid):
    """Two different catalogue pairs back to back, all_pairs then nearest on each: every call of the static entry point
    starts from whatever the previous one left in the array."""
    for scale in (0.5, 0.3):
        w = S.config(1, scale=scale)
        r = w.radius_arcsec
        ib = P.hlc2_build_index(*dev(w.B), opts=P.make_opts(r))
        ia = P.hlc2_build_index(*dev(w.A), opts=P.make_opts(r, target_occupancy=0.0 if grid == "same" else 0.7),
                                like=ib if grid == "same" else None)
        assert P.hlc2_crossmatch_sizes(ia, ib) <= P.HLC2_STATIC_SCRATCH_BYTES
        for mode in (P.HLC2_ALL_PAIRS, P.HLC2_NEAREST):
            ref, got = both_paths(P, ia, ib, r, mode, 4 * max(len(w.A), len(w.B)))
            assert len(ref[0]) > 10_000
            assert_same(ref, got)


def test_static_scratch_allocates_nothing_and_has_a_stated_limit(P):
    import torch
    # 1.5 million A rows: the match's scratch is 6 MB, so an allocation hidden in the call would move the device's free
    # memory by more than the 4 MiB allowed below (the driver hands memory out in 2 MiB pieces)
    rng = np.random.default_rng(90)
    n = 1_500_000
    rb, db = S.uniform_patch(rng, n, 40.0, 44.0, 20.0, 24.0)
    pr, pd = S.perturb(rng, rb, db, 0.3)
    pr = np.clip(pr, 40.0, 44.0); pd = np.clip(pd, 20.0, 24.0)
    r = 1.0
    ib = P.hlc2_build_index(torch.from_numpy(rb).cuda(), torch.from_numpy(db).cuda(), None, opts=P.make_opts(r))
    ia = P.hlc2_build_index(torch.from_numpy(pr).cuda(), torch.from_numpy(pd).cuda(), None, opts=P.make_opts(r), like=ib)
    assert 4 << 20 < P.hlc2_crossmatch_sizes(ia, ib) <= P.HLC2_STATIC_SCRATCH_BYTES
    cap = 2 * n
    oa = torch.empty(cap, dtype=torch.int64, device="cuda"); ob = torch.empty_like(oa)
    os_ = torch.empty(cap, dtype=torch.float64, device="cuda"); cnt = torch.zeros(1, dtype=torch.int64, device="cuda")
    P.hlc2_crossmatch_static(ia, ib, r, 0, oa, ob, os_, cnt); torch.cuda.synchronize()     # first call: address resolved, modules loaded
    n1 = int(cnt.item())
    free0, _ = torch.cuda.mem_get_info()
    reserved0 = torch.cuda.memory_reserved()
    for _ in range(3):
        P.hlc2_crossmatch_static(ia, ib, r, 0, oa, ob, os_, cnt)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] >= free0 - (4 << 20) and torch.cuda.memory_reserved() == reserved0
    assert int(cnt.item()) == n1 > 0.9 * n
    # the same rows as the caller-buffer path at this size too
    ref = torch.zeros(1, dtype=torch.int64, device="cuda")
    oa2 = torch.empty_like(oa); ob2 = torch.empty_like(oa); os2 = torch.empty_like(os_)
    P.hlc2_crossmatch(ia, ib, r, 0, oa2, ob2, os2, ref); torch.cuda.synchronize()
    assert int(ref.item()) == n1
    assert_same(rows(oa2, ob2, os2, n1), rows(oa, ob, os_, n1))

    # beyond the limit: 4 bytes per A row + 256 > 8 MiB -> refused with its own status, outputs untouched
    n_big = P.HLC2_STATIC_SCRATCH_BYTES // 4 + 1000
    rng = np.random.default_rng(91)
    ra, dec = S.uniform_patch(rng, n_big, 10.0, 14.0, -2.0, 2.0)
    big = P.hlc2_build_index(torch.from_numpy(ra).cuda(), torch.from_numpy(dec).cuda(), None, opts=P.make_opts(r))
    assert P.hlc2_crossmatch_sizes(big, big) > P.HLC2_STATIC_SCRATCH_BYTES
    cnt.fill_(-5)
    with pytest.raises(P.Hlc2Error) as e:
        P.hlc2_crossmatch_static(big, big, r, 0, oa, ob, os_, cnt)
    assert e.value.status == P.HLC2_ERR_STATIC_LIMIT and "8 MiB" in str(e.value)
    torch.cuda.synchronize()
    assert int(cnt.item()) == -5
    # and the same pair goes through the existing entry point
    a, b, s = P.crossmatch(big, big, r, 0, capacity=2 * n_big)
    assert a.shape[0] >= n_big                               # every source matches itself
