"""Parity cases for match paths the named configurations never reach (boundary loss is THE failure
mode of a partitioned cross-match): catalogues whose grids have different RA boxes / declination
extents, several radii r < r_max against one pair of indices, a forced overflow of the job pool, a seam-crossing tile
next to a one-cell polar zone (a pair must not be reported twice), rows with bad coordinates."""
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


def box_cat(rng, n, box, id0, step):
    ra, dec = S.uniform_patch(rng, n, *box)
    return S.Catalogue(np.mod(ra, 360.0), dec, np.arange(n, dtype=np.int64) * step + id0)


def with_copies(rng, A, B_uniform, sigma, box_b, margin_deg=0.05):
    """B = its own uniform sources + perturbed copies of the A sources that fall inside (or just outside) B's box."""
    ra_lo, ra_hi, d_lo, d_hi = box_b
    u = np.mod(A.ra - ra_lo, 360.0)
    inside = (u <= (ra_hi - ra_lo) + margin_deg) & (A.dec >= d_lo - margin_deg) & (A.dec <= d_hi + margin_deg)
    pr, pd = S.perturb(rng, A.ra[inside], A.dec[inside], sigma)
    ra = np.concatenate([pr, B_uniform.ra]); dec = np.clip(np.concatenate([pd, B_uniform.dec]), -90.0, 90.0)
    o = rng.permutation(len(ra))
    return S.Catalogue(ra[o], dec[o], np.arange(len(ra), dtype=np.int64) * 5 + 2 * 10**12)


def check(P, A, B, radius, mode, opts_a=None, opts_b=None, ia=None, ib=None, engine=oracle.ENGINE_VOXEL):
    if ia is None:
        ia = P.hlc2_build_index(*dev(A), opts=opts_a or P.make_opts(radius))
    if ib is None:
        ib = P.hlc2_build_index(*dev(B), opts=opts_b or P.make_opts(radius))
    a, b, s = P.crossmatch(ia, ib, radius, mode, capacity=max(1024, 4 * max(len(A), len(B))))
    oa, ob, os_, _ = oracle.match(A.ra, A.dec, A.id, B.ra, B.dec, B.id, radius, mode, engine)
    cmp = parity.compare_nearest if mode else parity.compare_all_pairs
    rep = cmp((a.cpu().numpy(), b.cpu().numpy(), s.cpu().numpy()), (oa, ob, os_), radius, parity.make_sep_of(A, B))
    assert len(rep["borderline"]) <= 2
    return rep, ia, ib


FULL = (0.0, 360.0, -90.0, 90.0)
CASES = {
    # name: (box of A, n_A, box of B, n_B uniform, radius)
    "fullsky_A_patch_B": (FULL, 150_000, (10.0, 40.0, -20.0, 10.0), 60_000, 20.0),
    "patch_A_fullsky_B": ((10.0, 40.0, -20.0, 10.0), 60_000, FULL, 150_000, 20.0),
    "overlapping_patches": ((100.0, 130.0, 0.0, 30.0), 80_000, (120.0, 150.0, 20.0, 50.0), 80_000, 15.0),
    "seam_patch_vs_plain_patch": ((350.0, 370.0, -10.0, 10.0), 60_000, (0.0, 30.0, -5.0, 15.0), 60_000, 15.0),
    "plain_patch_vs_seam_patch": ((0.0, 30.0, -5.0, 15.0), 60_000, (350.0, 370.0, -10.0, 10.0), 60_000, 15.0),
    "dec_extents_touch": ((50.0, 60.0, 0.0, 10.0), 50_000, (50.0, 60.0, 10.0, 20.0), 50_000, 30.0),
    "polar_cap_vs_fullsky": ((0.0, 360.0, 85.0, 90.0), 40_000, FULL, 150_000, 25.0),
}


@pytest.mark.parametrize("name", sorted(CASES))
@pytest.mark.parametrize("mode", [0, 1])
def test_different_boxes(P, name, mode):
    """A and B carry grids with different RA boxes / declination extents: the planner's box-frame shift, its second
    RA interval and the general path's partly-outside windows all see boxes that are not their own."""
    box_a, n_a, box_b, n_b, r = CASES[name]
    rng = np.random.default_rng(abs(hash(name)) % 2**31)
    A = box_cat(rng, n_a, box_a, 10**12, 3)
    if name == "dec_extents_touch":          # sources planted within r of the shared edge, on both sides
        k = len(A) // 2
        A.dec[:k] = 10.0 - rng.uniform(0.0, 2 * r, k) / 3600.0
    B = with_copies(rng, A, box_cat(rng, n_b, box_b, 0, 1), r / 3, box_b)
    rep, ia, ib = check(P, A, B, r, mode)
    assert rep["n_gpu"] > 500, rep["n_gpu"]
    ga, gb = P.hlc2_grid_describe(ia), P.hlc2_grid_describe(ib)
    assert (ga["span"], ga["ra0"], ga["dec_lo"]) != (gb["span"], gb["ra0"], gb["dec_lo"])


@pytest.mark.parametrize("mode", [0, 1])
def test_radii_below_r_max_on_one_index_pair(P, mode):
    """Build once with r_max, query several radii (the ABI's stated use): windows come from the query radius, the
    grid from r_max."""
    w = S.config(2, scale=0.02)
    r_max = 30.0
    ia = P.hlc2_build_index(*dev(w.A), opts=P.make_opts(r_max)); ib = P.hlc2_build_index(*dev(w.B), opts=P.make_opts(r_max))
    last = -1
    for r in (0.05, 0.7, 2.0, 11.0, 30.0):
        rep, _, _ = check(P, w.A, w.B, r, mode, ia=ia, ib=ib)
        assert rep["n_gpu"] >= last
        last = rep["n_gpu"]
    assert last > 130_000
    with pytest.raises(P.Hlc2Error) as e:
        P.crossmatch(ia, ib, 30.0001, mode)
    assert e.value.status == P.HLC2_ERR_RADIUS_TOO_LARGE
    # A filed on B's grid (opts.grid_like), same radii
    ia2 = P.hlc2_build_index(*dev(w.A), opts=P.make_opts(r_max), like=ib)
    for r in (0.7, 30.0):
        check(P, w.A, w.B, r, mode, ia=ia2, ib=ib)


@pytest.mark.parametrize("mode", [0, 1])
def test_job_pool_overflow_falls_back(P, mode):
    """A few A tiles whose windows hold ~1e6 B rows each: the chained jobs exceed the pool (3 x tiles + 4096), the
    planner marks the tiles it could not finish DIRECT and nothing is lost."""
    import torch
    rng = np.random.default_rng(77)
    box = (30.0, 30.2, 40.0, 40.2)
    A = box_cat(rng, 100, box, 10**12, 3)
    B = with_copies(rng, A, box_cat(rng, 3_000_000, box, 0, 1), 1.0, box)
    o = P.make_opts(5.0, cell_arcsec=60.0)
    ia = P.hlc2_build_index(*dev(A), opts=o); ib = P.hlc2_build_index(*dev(B), opts=o)
    need = P.hlc2_crossmatch_sizes(ia, ib)
    temp = torch.zeros(need, dtype=torch.uint8, device="cuda")
    cap = 1 << 20
    oa = torch.empty(cap, dtype=torch.int64, device="cuda"); ob = torch.empty_like(oa)
    os_ = torch.empty(cap, dtype=torch.float64, device="cuda"); cnt = torch.zeros(1, dtype=torch.int64, device="cuda")
    P.hlc2_crossmatch(ia, ib, 5.0, mode, oa, ob, os_, cnt, temp=temp)
    n = int(cnt.item()); assert n <= cap
    pool_n = int(temp[:4].view(torch.int32).item())
    pool_cap = 3 * (len(A) // 128 + P.hlc2_grid_describe(ia)["n_zones"] + 1) + 4096        # of the driving catalogue's tiles
    assert pool_n > pool_cap, (pool_n, pool_cap)          # the counter ran past the pool: the overflow branch was taken
    oa_, ob_, os2, _ = oracle.match(A.ra, A.dec, A.id, B.ra, B.dec, B.id, 5.0, mode)
    cmp = parity.compare_nearest if mode else parity.compare_all_pairs
    rep = cmp((oa[:n].cpu().numpy(), ob[:n].cpu().numpy(), os_[:n].cpu().numpy()), (oa_, ob_, os2), 5.0, parity.make_sep_of(A, B))
    assert rep["n_gpu"] == (100 if mode else rep["n_oracle"]) and rep["n_oracle"] > (50 if mode else 20_000)


@pytest.mark.parametrize("mode", [0, 1])
def test_seam_tile_next_to_one_cell_polar_zone(P, mode):
    """Full-sky grid with 160-arcsec cells: the last zone has one RA cell, the one below it six.  A rows just under
    that zone edge within the RA window of the seam reach the polar cell through both images of their window; every
    pair must be reported exactly once (tests/parity.py asserts uniqueness)."""
    rng = np.random.default_rng(160)
    o = P.make_opts(3.0, cell_arcsec=160.0, full_sky=True, zone_aspect=1)       # square cells: zones 160 arcsec high
    parts_ra, parts_dec = [], []
    for sign in (1.0, -1.0):
        edge = 90.0 - 160.0 / 3600.0
        n = 4000
        ra = np.concatenate([rng.uniform(0.0, 1.2, n // 2), rng.uniform(358.8, 360.0, n // 2)])
        dec = sign * (edge - rng.uniform(-3.0, 3.0, n) / 3600.0)
        parts_ra.append(ra); parts_dec.append(dec)
    ura, udec = S.uniform_sphere(rng, 20_000)
    ra = np.concatenate(parts_ra + [ura]); dec = np.concatenate(parts_dec + [udec])
    A = S.Catalogue(ra, dec, np.arange(len(ra), dtype=np.int64) * 3 + 10**12)
    pr, pd = S.perturb(rng, A.ra, A.dec, 1.0)
    B = S.Catalogue(pr, np.clip(pd, -90.0, 90.0), np.arange(len(pr), dtype=np.int64) * 5 + 2 * 10**12)
    rep, ia, ib = check(P, A, B, 3.0, mode, opts_a=o, opts_b=o, engine=oracle.ENGINE_BRUTE)
    g = P.hlc2_grid_describe(ib)
    assert g["n_ra"][-1] == 1 and g["n_ra"][0] == 1 and 2 <= g["n_ra"][-2] <= 8
    assert rep["n_gpu"] > 20_000


def test_bad_rows_never_appear(P):
    """Rows with a non-finite coordinate or |dec| > 90 are reported by hlc2_index_status and appear in no result,
    neither as idA nor as idB, in either mode; the other rows are matched as usual."""
    w = S.config(1, scale=0.2)
    rng = np.random.default_rng(9)
    A = w.A.take(np.arange(len(w.A))); B = w.B.take(np.arange(len(w.B)))
    bad_a = rng.choice(len(A), 300, replace=False); bad_b = rng.choice(len(B), 300, replace=False)
    A.dec[bad_a[:100]] = np.nan; A.ra[bad_a[100:200]] = np.inf; A.dec[bad_a[200:]] = 90.5
    B.ra[bad_b[:150]] = np.nan; B.dec[bad_b[150:]] = -123.0
    ia = P.hlc2_build_index(*dev(A), opts=P.make_opts(1.0)); ib = P.hlc2_build_index(*dev(B), opts=P.make_opts(1.0))
    assert P.hlc2_index_status(ia) == (P.HLC2_ERR_BAD_COORD, int(bad_a.min()))
    assert P.hlc2_index_status(ib) == (P.HLC2_ERR_BAD_COORD, int(bad_b.min()))
    ga = np.delete(np.arange(len(A)), bad_a); gb = np.delete(np.arange(len(B)), bad_b)
    Ag, Bg = A.take(ga), B.take(gb)
    for mode in (0, 1):
        a, b, s = P.crossmatch(ia, ib, 1.0, mode)
        a, b, s = a.cpu().numpy(), b.cpu().numpy(), s.cpu().numpy()
        assert not np.isin(a, A.id[bad_a]).any() and not np.isin(b, B.id[bad_b]).any()
        oa, ob, os_, _ = oracle.match(Ag.ra, Ag.dec, Ag.id, Bg.ra, Bg.dec, Bg.id, 1.0, mode)
        cmp = parity.compare_nearest if mode else parity.compare_all_pairs
        rep = cmp((a, b, s), (oa, ob, os_), 1.0, parity.make_sep_of(Ag, Bg))
        assert rep["n_gpu"] > 10_000
    # a catalogue of bad rows only, and one bad row matched against itself
    import torch
    nanv = torch.full((5,), float("nan"), dtype=torch.float64, device="cuda")
    ix = P.hlc2_build_index(nanv, nanv.clone(), None, opts=P.make_opts(1.0))
    assert P.hlc2_index_status(ix)[0] == P.HLC2_ERR_BAD_COORD
    for mode in (0, 1):
        assert len(P.crossmatch(ix, ix, 1.0, mode)[0]) == 0
        assert len(P.crossmatch(ia, ix, 1.0, mode)[0]) == 0
