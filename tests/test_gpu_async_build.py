"""opts.async_like (include/hlc2.h): an index built on another index's grid without the extent pass and without any host
synchronisation (the build is a stream-ordered call).  Checked: the index is the one the synchronous
build makes, hlc2_index_status reports bad rows and an out-of-box catalogue after the fact, and build + match capture
into ONE CUDA graph that is replayed on new catalogue contents (which a call that synchronises cannot do)."""
import numpy as np
import pytest

import hlc2_synth as S
import oracle
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


def test_async_like_build_is_the_synchronous_index(P):
    w = S.config(1, scale=0.5)
    r = w.radius_arcsec
    ib = P.hlc2_build_index(*dev(w.B), opts=P.make_opts(r))
    ia_sync = P.hlc2_build_index(*dev(w.A), opts=P.make_opts(r), like=ib)
    ia = P.hlc2_build_index(*dev(w.A), opts=P.make_opts(r, async_like=True), like=ib)
    assert P.hlc2_index_status(ia) == (P.HLC2_OK, -1)
    s, a = P.hlc2_index_arrays(ia_sync), P.hlc2_index_arrays(ia)
    for k in ("x", "y", "z", "id", "cell_start", "cell_key"):      # the sort is stable: identical row order too
        assert bool((s[k] == a[k]).all()), k
    sep_of = parity.make_sep_of(w.A, w.B)
    for mode in (0, 1):
        got = P.crossmatch(ia, ib, r, mode)
        oa, ob, os_, _ = oracle.match(w.A.ra, w.A.dec, w.A.id, w.B.ra, w.B.dec, w.B.id, r, mode)
        cmp = parity.compare_nearest if mode else parity.compare_all_pairs
        rep = cmp(tuple(t.cpu().numpy() for t in got), (oa, ob, os_), r, sep_of)
        assert len(rep["borderline"]) <= 2 and rep["n_gpu"] > 30_000


def test_async_like_status_reports_bad_rows_and_out_of_box(P):
    import torch
    rng = np.random.default_rng(71)
    ra, dec = S.uniform_patch(rng, 50_000, 30.0, 31.0, -5.0, -4.0)
    ib = P.hlc2_build_index(torch.from_numpy(ra).cuda(), torch.from_numpy(dec).cuda(), None, opts=P.make_opts(2.0))
    o = P.make_opts(2.0, async_like=True)

    def status(ra2, dec2):
        return P.hlc2_index_status(P.hlc2_build_index(torch.from_numpy(ra2).cuda(), torch.from_numpy(dec2).cuda(), None, opts=o, like=ib))

    assert status(ra[:1000].copy(), dec[:1000].copy()) == (P.HLC2_OK, -1)
    bad = dec[:1000].copy(); bad[[17, 400]] = [np.nan, 91.0]
    assert status(ra[:1000].copy(), bad) == (P.HLC2_ERR_BAD_COORD, 17)
    east = ra[:1000].copy(); east[5] = 40.0                         # outside the RA box
    assert status(east, dec[:1000].copy())[0] == P.HLC2_ERR_GRID_MISMATCH
    north = dec[:1000].copy(); north[999] = 20.0                    # beyond the last zone: filed in it, as in any build
    assert status(ra[:1000].copy(), north) == (P.HLC2_OK, -1)
    # the synchronous build refuses the RA case at the call
    with pytest.raises(P.Hlc2Error):
        P.hlc2_build_index(torch.from_numpy(east).cuda(), torch.from_numpy(dec[:1000].copy()).cuda(), None, opts=P.make_opts(2.0), like=ib)


def test_build_and_match_replay_as_one_cuda_graph(P):
    """Capture hlc2_build_index(async_like) + hlc2_crossmatch once; replay on two other catalogues copied into the same
    input buffers.  Each replay's pairs are the oracle's for that catalogue."""
    import torch
    rng = np.random.default_rng(72)
    box = (200.0, 201.5, 44.0, 45.5)
    nb, na, r = 300_000, 60_000, 1.5
    rb, db = S.uniform_patch(rng, nb, *box)
    B = S.Catalogue(rb, db, np.arange(nb, dtype=np.int64) * 5 + 2 * 10**12)
    ib = P.hlc2_build_index(*dev(B), opts=P.make_opts(r))

    def make_a(seed):
        g = np.random.default_rng(seed)
        k = g.choice(nb, na, replace=False)
        pr, pd = S.perturb(g, B.ra[k], B.dec[k], 0.8)
        lo = np.array([box[0], box[2]]); hi = np.array([box[1], box[3]])
        pr = np.clip(pr, lo[0], hi[0]); pd = np.clip(pd, lo[1], hi[1])     # stay inside B's box
        return S.Catalogue(pr, pd, np.arange(na, dtype=np.int64) * 3 + 10**12)

    cats = [make_a(s) for s in (1, 2, 3)]
    ra_d, dec_d, id_d = dev(cats[0])
    o = P.make_opts(r, async_like=True)
    ibytes, tbytes = P.hlc2_index_sizes(na, o)
    buf = torch.empty(ibytes, dtype=torch.uint8, device="cuda"); temp = torch.empty(tbytes, dtype=torch.uint8, device="cuda")
    cap = 4 * na
    oa = torch.empty(cap, dtype=torch.int64, device="cuda"); ob = torch.empty_like(oa)
    os_ = torch.empty(cap, dtype=torch.float64, device="cuda"); cnt = torch.zeros(1, dtype=torch.int64, device="cuda")
    # scratch for the match is sized from a throw-away index of the same shape (sizes depend on n and the grid only)
    probe = P.hlc2_build_index(ra_d, dec_d, id_d, opts=o, like=ib)
    mtemp = torch.empty(max(P.hlc2_crossmatch_sizes(probe, ib), 16), dtype=torch.uint8, device="cuda")
    torch.cuda.synchronize()

    side = torch.cuda.Stream()
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.stream(side):
        graph.capture_begin()
        ia = P.hlc2_build_index(ra_d, dec_d, id_d, opts=o, like=ib, stream=side, temp=temp, buf=buf)
        P.hlc2_crossmatch(ia, ib, r, 0, oa, ob, os_, cnt, stream=side, temp=mtemp)
        graph.capture_end()
    for c in cats:
        ra_d.copy_(torch.from_numpy(c.ra)); dec_d.copy_(torch.from_numpy(c.dec)); id_d.copy_(torch.from_numpy(c.id))
        torch.cuda.synchronize()
        graph.replay()
        torch.cuda.synchronize()
        n = int(cnt.item())
        assert 0 < n <= cap
        ea, eb, es, _ = oracle.match(c.ra, c.dec, c.id, B.ra, B.dec, B.id, r, 0)
        rep = parity.compare_all_pairs((oa[:n].cpu().numpy(), ob[:n].cpu().numpy(), os_[:n].cpu().numpy()), (ea, eb, es), r,
                                       parity.make_sep_of(c, B))
        assert len(rep["borderline"]) <= 2 and rep["n_gpu"] >= na * 0.9
    assert P.hlc2_index_status(ia)[0] == P.HLC2_OK


def test_async_like_index_against_an_index_on_another_grid(P):
    """An index built asynchronously on C's grid, matched with B whose grid is its own (the two-grid kernel): the
    declination extent of the asynchronous index is the whole sphere, so the tiles of its first and last zone plan their
    windows over every B zone beyond the grid -- slower, and the pairs must still be the oracle's.  B reaches far beyond
    C's box on both sides."""
    rng = np.random.default_rng(73)
    rb, db = S.uniform_patch(rng, 200_000, 80.0, 84.0, -3.0, 3.0)
    B = S.Catalogue(rb, db, np.arange(len(rb), dtype=np.int64) * 5 + 2 * 10**12)
    inside = (rb > 81.0) & (rb < 83.0) & (db > -0.5) & (db < 0.5)
    k = np.flatnonzero(inside)
    pr, pd = S.perturb(rng, B.ra[k], B.dec[k], 1.0)
    keep = (pr > 81.0) & (pr < 83.0) & (pd > -0.5) & (pd < 0.5)
    A = S.Catalogue(pr[keep], pd[keep], np.arange(int(keep.sum()), dtype=np.int64) * 3 + 10**12)
    rc, dc = S.uniform_patch(rng, 30_000, 81.0, 83.0, -0.5, 0.5)
    C = S.Catalogue(rc, dc, np.arange(len(rc), dtype=np.int64))
    r = 2.0
    ib = P.hlc2_build_index(*dev(B), opts=P.make_opts(r))
    ic = P.hlc2_build_index(*dev(C), opts=P.make_opts(r, target_occupancy=0.6))
    ia = P.hlc2_build_index(*dev(A), opts=P.make_opts(r, async_like=True), like=ic)
    assert P.hlc2_index_status(ia) == (P.HLC2_OK, -1)
    assert P.hlc2_grid_describe(ia)["n_cells"] != P.hlc2_grid_describe(ib)["n_cells"]
    sep_of = parity.make_sep_of(A, B)
    for mode in (0, 1):
        got = P.crossmatch(ia, ib, r, mode)
        oa, ob, os_, _ = oracle.match(A.ra, A.dec, A.id, B.ra, B.dec, B.id, r, mode)
        cmp = parity.compare_nearest if mode else parity.compare_all_pairs
        rep = cmp(tuple(t.cpu().numpy() for t in got), (oa, ob, os_), r, sep_of)
        assert len(rep["borderline"]) <= 2 and rep["n_gpu"] > 0.8 * len(A)
