"""Parity of the CUDA path (through the C ABI) with the CPU oracle, element by element, on the same
seeded inputs.  Run on the B200 box: python -m pytest tests -m gpu.

Bar (north_star): pair sets bit-exact as (idA, idB) sets except pairs with |sep - r| < 1e-9 arcsec
(listed separately); separations within 1e-9 arcsec (tests/parity.py).
"""
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


def dev(cat):
    import torch
    return (torch.from_numpy(cat.ra).cuda(), torch.from_numpy(cat.dec).cuda(), torch.from_numpy(cat.id).cuda())


def gpu_match(P, A, B, radius, mode, opts_a=None, opts_b=None, same_grid=False, **kw):
    ib = P.hlc2_build_index(*dev(B), opts=opts_b or P.make_opts(radius, **kw))
    ia = P.hlc2_build_index(*dev(A), opts=opts_a or P.make_opts(radius, **kw), like=ib if same_grid else None)
    assert P.hlc2_index_status(ia)[0] == 0 and P.hlc2_index_status(ib)[0] == 0
    a, b, s = P.crossmatch(ia, ib, radius, mode)
    return a.cpu().numpy(), b.cpu().numpy(), s.cpu().numpy(), ia, ib


def check(P, A, B, radius, mode, engine=oracle.ENGINE_VOXEL, **kw):
    ga, gb, gs, ia, ib = gpu_match(P, A, B, radius, mode, **kw)
    oa, ob, os_, _ = oracle.match(A.ra, A.dec, A.id, B.ra, B.dec, B.id, radius, mode, engine)
    cmp = parity.compare_nearest if mode == P.HLC2_NEAREST else parity.compare_all_pairs
    rep = cmp((ga, gb, gs), (oa, ob, os_), radius, parity.make_sep_of(A, B))
    assert len(rep["borderline"]) <= 2, rep["borderline"]
    return rep, ia, ib


# ------------------------------------------------------------------------------ index build (rows a1-a4)
@pytest.mark.parametrize("cfg,scale", [(1, 1.0), (2, 0.03), (3, 0.003)])
def test_index_invariants(P, cfg, scale):
    """Keys sorted, rows a permutation of the input, cell table monotone and consistent with the keys,
    unit vectors equal to the definition (cos d cos a, cos d sin a, sin d) to a few ulp."""
    import torch
    w = S.config(cfg, scale=scale)
    ra, dec, ids = dev(w.B)
    idx = P.hlc2_build_index(ra, dec, ids, opts=P.make_opts(w.radius_arcsec))
    assert P.hlc2_index_status(idx) == (0, -1)
    arr = P.hlc2_index_arrays(idx)
    n, nc = arr["n"], arr["n_cells"]
    assert n == len(w.B)
    key = arr["cell_key"].cpu().numpy().view(np.uint32).astype(np.int64)
    flags = key >> 28                                  # window flags ride in the top bits (include/hlc2.h, HLC2_KEY_MASK)
    key = key & P.HLC2_KEY_MASK
    assert flags.max() <= 15
    cs = arr["cell_start"].cpu().numpy().view(np.uint32).astype(np.int64)
    assert (np.diff(key) >= 0).all() and key.max() < nc
    assert cs[0] == 0 and cs[-1] == n and (np.diff(cs) >= 0).all()
    assert np.array_equal(np.searchsorted(key, np.arange(nc + 1), side="left"), cs)
    sid = arr["id"].cpu().numpy()
    assert np.array_equal(np.sort(sid), np.sort(w.B.id))
    row = (sid - w.B.id[0]) // 2                       # ids of the generator are 2*row + const
    a, d = np.deg2rad(w.B.ra[row]), np.deg2rad(w.B.dec[row])
    x, y, z = (arr[k].cpu().numpy() for k in "xyz")
    assert np.abs(x - np.cos(d) * np.cos(a)).max() < 2e-15
    assert np.abs(y - np.cos(d) * np.sin(a)).max() < 2e-15
    assert np.abs(z - np.sin(d)).max() < 2e-15
    g = P.hlc2_grid_describe(idx)
    assert g["n_cells"] == nc and g["n_ra"].sum() == nc and g["cell_arcsec"] >= w.radius_arcsec
    # window flags (bits 30 / 31: the window reaches the zone below / above; both: general path): a row within r_max of
    # a zone edge must carry that edge's flag, a row further than r_max (+ slop) from both edges must carry neither
    dec_s = np.rad2deg(np.arcsin(np.clip(z, -1.0, 1.0)))
    zone = np.clip(np.floor((dec_s - g["dec_lo"]) / g["zone_h"]).astype(np.int64), 0, g["n_zones"] - 1)
    d_lo = dec_s - (g["dec_lo"] + zone * g["zone_h"]); d_hi = (g["dec_lo"] + (zone + 1) * g["zone_h"]) - dec_s
    r_deg = w.radius_arcsec / 3600.0
    general = (flags >> 2) == 3
    need_lo = (d_lo < r_deg - 1e-7) & (zone > 0); need_hi = (d_hi < r_deg - 1e-7) & (zone < g["n_zones"] - 1)
    assert (((flags >> 2) & 1)[need_lo] == 1).all() and (((flags >> 3) & 1)[need_hi] == 1).all()
    far = (d_lo > r_deg + 1e-6) & (d_hi > r_deg + 1e-6) & ~general
    assert ((flags >> 2)[far] == 0).all()
    # occupancy near the target (1 source per cell over the occupied box)
    assert 0.2 < n / nc < 5.0


# ------------------------------------------------------------------------------ parity, the five configs (scaled)
@pytest.mark.parametrize("mode", ["all_pairs", "nearest"])
def test_cfg1_tiny_patch(P, mode):
    w = S.config(1)
    m = P.HLC2_NEAREST if mode == "nearest" else P.HLC2_ALL_PAIRS
    rep, _, _ = check(P, w.A, w.B, w.radius_arcsec, m)
    assert rep["n_gpu"] > 75_000
    # the same patch matched with cells forced to the minimum size (= r) and with huge cells, each also with A filed
    # on B's grid (opts.grid_like: the same-grid path of the match)
    check(P, w.A, w.B, w.radius_arcsec, m, same_grid=True)
    for cell in (1.0, 900.0):
        check(P, w.A, w.B, w.radius_arcsec, m, cell_arcsec=cell)
        check(P, w.A, w.B, w.radius_arcsec, m, cell_arcsec=cell, same_grid=True)


@pytest.mark.parametrize("same_grid", [False, True])
@pytest.mark.parametrize("mode", ["all_pairs", "nearest"])
def test_cfg2_full_sky_scaled(P, mode, same_grid):
    w = S.config(2, scale=0.1)          # 1e6 x 1e6: several hundred tiles and a ragged tail
    m = P.HLC2_NEAREST if mode == "nearest" else P.HLC2_ALL_PAIRS
    rep, _, _ = check(P, w.A, w.B, w.radius_arcsec, m, same_grid=same_grid)
    assert rep["n_gpu"] > 690_000


@pytest.mark.parametrize("same_grid", [False, True])
def test_cfg3_gaia_like_scaled(P, same_grid):
    w = S.config(3, scale=0.012)        # 1.2e6 x 6e5, galactic-plane density contrast
    rep, _, _ = check(P, w.A, w.B, w.radius_arcsec, P.HLC2_ALL_PAIRS, same_grid=same_grid)
    assert rep["n_gpu"] > 355_000


def test_cfg4_boundary_stress_vs_brute_force(P):
    """Sources pushed onto the IMPLEMENTATION's own cell / zone edges and corners, the poles and the RA seam
    (grid taken from hlc2_grid_describe), completeness against brute force (the paper's 'No Index')."""
    import torch
    scale = 0.01                                                     # 2e5 x 2e5, r = 3 arcsec
    n_b = int(round(20_000_000 * scale))
    opts = P.make_opts(3.0, cell_arcsec=160.0, full_sky=True, zone_aspect=1)   # config 4's nominal grid: square 160" cells, full sky
    prelim_ra, prelim_dec = S.uniform_sphere(np.random.default_rng(1), n_b)
    pre = P.hlc2_build_index(torch.from_numpy(prelim_ra).cuda(), torch.from_numpy(prelim_dec).cuda(), None, opts=opts)
    grid = P.hlc2_grid_describe(pre)
    w = S.config(4, scale=scale, grid=grid)
    ia = P.hlc2_build_index(*dev(w.A), opts=P.make_opts(3.0, cell_arcsec=160.0, full_sky=True, zone_aspect=1))
    ib = P.hlc2_build_index(*dev(w.B), opts=P.make_opts(3.0), like=pre)          # exactly the described grid
    gb_grid = P.hlc2_grid_describe(ib)
    assert gb_grid["n_cells"] == grid["n_cells"] and np.array_equal(gb_grid["n_ra"], grid["n_ra"])
    ia_same = P.hlc2_build_index(*dev(w.A), opts=P.make_opts(3.0), like=pre)     # A on the same grid: the same-grid path
    sep_of = parity.make_sep_of(w.A, w.B)
    for mode in (P.HLC2_ALL_PAIRS, P.HLC2_NEAREST):
        oa, ob, os_, _ = oracle.match(w.A.ra, w.A.dec, w.A.id, w.B.ra, w.B.dec, w.B.id, 3.0, mode, oracle.ENGINE_BRUTE)
        cmp = parity.compare_nearest if mode == P.HLC2_NEAREST else parity.compare_all_pairs
        for ixa in (ia, ia_same):
            a, b, s = P.crossmatch(ixa, ib, 3.0, mode)
            rep = cmp((a.cpu().numpy(), b.cpu().numpy(), s.cpu().numpy()), (oa, ob, os_), 3.0, sep_of)
            assert rep["n_oracle"] > 150_000 and len(rep["borderline"]) <= 2


# ------------------------------------------------------------------------------ poles, seam, degenerate inputs
def _tiny(seed=11):
    rng = np.random.default_rng(seed)
    ra = np.concatenate([rng.uniform(0, 360, 150), rng.uniform(-0.002, 0.002, 120) % 360.0,
                         rng.uniform(0, 360, 100), rng.uniform(0, 360, 100), [0.0, 360.0, 10.0, 10.0, -0.0, 719.999999]])
    dec = np.concatenate([np.rad2deg(np.arcsin(rng.uniform(-1, 1, 150))), rng.uniform(-0.002, 0.002, 120),
                          90.0 - np.abs(rng.normal(0, 0.001, 100)), -90.0 + np.abs(rng.normal(0, 0.001, 100)),
                          [90.0, -90.0, 20.0, 20.0, 0.0, 0.0]])
    ra_b, dec_b = S.perturb(rng, ra, dec, 1.5)
    ra_b = np.concatenate([ra_b, ra[:50]]); dec_b = np.concatenate([dec_b, dec[:50]])
    A = S.Catalogue(ra, dec, S.ids_a(len(ra))); B = S.Catalogue(ra_b, dec_b, S.ids_b(len(ra_b)))
    return A, B


@pytest.mark.parametrize("radius", [0.5, 3.0, 40.0, 3000.0, 36000.0])
@pytest.mark.parametrize("mode", [0, 1])
def test_poles_seam_duplicates_micro(P, radius, mode):
    """Both poles, the RA = 0/360 seam, exact duplicates, RA given as 360.0 / -0.0 / 719.99..., against the
    all-long-double brute force; radii from sub-cell to 10 degrees (windows wider than the polar cap)."""
    A, B = _tiny()
    for kw in ({}, {"full_sky": True}, {"cell_arcsec": radius}, {"cell_arcsec": 20000.0}):
        check(P, A, B, radius, mode, engine=oracle.ENGINE_BRUTE_LD, **kw)
        try:
            check(P, A, B, radius, mode, engine=oracle.ENGINE_BRUTE_LD, same_grid=True, **kw)
        except P.Hlc2Error as e:        # B's few hundred sources leave RA gaps: its box may not hold all of A
            assert e.status == P.HLC2_ERR_GRID_MISMATCH and not kw.get("full_sky")


def test_patch_across_ra_seam_and_on_pole(P):
    """Config 1's patch rotated onto RA = 0 (box straddles the seam) and onto the north pole."""
    w = S.config(1, scale=0.3)
    th = np.deg2rad(89.0)
    Rz = lambda t: np.array([[np.cos(t), -np.sin(t), 0], [np.sin(t), np.cos(t), 0], [0, 0, 1]])
    Ry = lambda t: np.array([[np.cos(t), 0, -np.sin(t)], [0, 1, 0], [np.sin(t), 0, np.cos(t)]])

    def rot(c, R):
        a, d = np.deg2rad(c.ra), np.deg2rad(c.dec)
        x, y, z = R @ np.stack([np.cos(d) * np.cos(a), np.cos(d) * np.sin(a), np.sin(d)])
        ra = np.mod(np.rad2deg(np.arctan2(y, x)), 360.0); ra[ra >= 360.0] = 0.0
        return S.Catalogue(ra, np.rad2deg(np.arctan2(z, np.hypot(x, y))), c.id)

    for R in (Rz(np.deg2rad(179.0)), Ry(th) @ Rz(np.deg2rad(-181.0))):
        A, B = rot(w.A, R), rot(w.B, R)
        for mode in (0, 1):
            rep, ia, ib = check(P, A, B, 1.0, mode)
            assert rep["n_gpu"] > 20_000
    g = P.hlc2_grid_describe(ib)
    assert g["span"] == 360.0                      # polar patch: all RAs occur
    A, B = rot(w.A, Rz(np.deg2rad(179.0))), rot(w.B, Rz(np.deg2rad(179.0)))
    _, ia, ib = check(P, A, B, 1.0, 0)
    g = P.hlc2_grid_describe(ib)
    assert g["span"] < 5.0 and g["ra0"] > 350.0   # a box of a few degrees that starts west of RA = 0


def test_self_match_and_symmetry(P):
    w = S.config(1, scale=0.2)
    ga, gb, gs, ia, _ = gpu_match(P, w.A, w.A, 1.0, P.HLC2_ALL_PAIRS)
    diag = ga == gb
    assert diag.sum() == len(w.A) and (gs[diag] == 0.0).all()
    a1, b1, s1, _, _ = gpu_match(P, w.A, w.B, 1.0, 0)
    b2, a2, s2, _, _ = gpu_match(P, w.B, w.A, 1.0, 0)
    o1 = np.lexsort((b1, a1)); o2 = np.lexsort((b2, a2))
    assert np.array_equal(a1[o1], a2[o2]) and np.array_equal(b1[o1], b2[o2])
    assert np.abs(s1[o1] - s2[o2]).max() < 1e-10


def test_inclusive_threshold_either_side(P):
    """Eq. (4) is inclusive; 2^-10 deg = 3.515625 arcsec apart on the equator: in at +2e-9, out at -2e-9."""
    A = S.Catalogue(np.array([100.0]), np.array([0.0]), np.array([7], np.int64))
    B = S.Catalogue(np.array([100.0 + 2.0 ** -10]), np.array([0.0]), np.array([9], np.int64))
    sep = 3.515625
    for r, want in ((sep + 2e-9, 1), (sep - 2e-9, 0)):
        ga, gb, gs, _, _ = gpu_match(P, A, B, r, 0, opts_a=P.make_opts(4.0), opts_b=P.make_opts(4.0))
        assert len(ga) == want
        if want:
            assert abs(gs[0] - sep) < 1e-9 and ga[0] == 7 and gb[0] == 9


# ------------------------------------------------------------------------------ ABI behaviour on the device
def test_empty_and_single(P):
    import torch
    e = S.Catalogue(np.zeros(0), np.zeros(0), np.zeros(0, np.int64))
    one = S.Catalogue(np.array([10.0]), np.array([-45.0]), np.array([5], np.int64))
    for A, B, want in ((e, e, 0), (e, one, 0), (one, e, 0), (one, one, 1)):
        for mode in (0, 1):
            ga, gb, gs, _, _ = gpu_match(P, A, B, 1.0, mode)
            assert len(ga) == want
    # ids = None -> row numbers
    ra = torch.tensor([1.0, 2.0, 1.0], dtype=torch.float64).cuda(); dec = torch.zeros(3, dtype=torch.float64).cuda()
    ia = P.hlc2_build_index(ra, dec, None, opts=P.make_opts(1.0))
    a, b, s = P.crossmatch(ia, ia, 1.0, 0)
    got = sorted(zip(a.tolist(), b.tolist()))
    assert got == [(0, 0), (0, 2), (1, 1), (2, 0), (2, 2)]


def test_capacity_overflow_counts_everything(P):
    import torch
    w = S.config(1, scale=0.1)
    ia = P.hlc2_build_index(*dev(w.A), opts=P.make_opts(1.0)); ib = P.hlc2_build_index(*dev(w.B), opts=P.make_opts(1.0))
    full = P.crossmatch(ia, ib, 1.0, 0)
    n = len(full[0])
    cap = n // 3
    oa = torch.full((cap,), -1, dtype=torch.int64).cuda(); ob = torch.full((cap,), -1, dtype=torch.int64).cuda()
    os_ = torch.zeros(cap, dtype=torch.float64).cuda(); cnt = torch.zeros(1, dtype=torch.int64).cuda()
    P.hlc2_crossmatch(ia, ib, 1.0, 0, oa, ob, os_, cnt)
    assert int(cnt.item()) == n                      # counted past capacity, nothing written out of bounds
    got = set(zip(oa.tolist(), ob.tolist())); ref = set(zip(full[0].tolist(), full[1].tolist()))
    assert len(got) == cap and got <= ref
    P.hlc2_crossmatch(ia, ib, 1.0, 0, oa[:0], ob[:0], os_[:0], cnt)     # capacity 0: count only
    assert int(cnt.item()) == n


def test_bad_coordinates_and_errors(P):
    import torch
    ra = torch.tensor([1.0, 2.0, float("nan"), 4.0], dtype=torch.float64).cuda()
    dec = torch.tensor([0.0, 91.0, 0.0, 0.0], dtype=torch.float64).cuda()
    idx = P.hlc2_build_index(ra, dec, None, opts=P.make_opts(1.0))
    assert P.hlc2_index_status(idx) == (P.HLC2_ERR_BAD_COORD, 1)
    a, b, s = P.crossmatch(idx, idx, 1.0, 0)          # bad rows appear in no result
    assert set(zip(a.tolist(), b.tolist())) == {(0, 0), (3, 3)}
    good = P.hlc2_build_index(ra[:1], dec[:1], None, opts=P.make_opts(1.0))
    with pytest.raises(P.Hlc2Error) as e:
        P.crossmatch(good, good, 2.0, 0)
    assert e.value.status == P.HLC2_ERR_RADIUS_TOO_LARGE
    for bad_r in (0.0, -1.0, float("nan")):
        with pytest.raises(P.Hlc2Error) as e:
            P.crossmatch(good, good, bad_r, 0)
        assert e.value.status == P.HLC2_ERR_INVALID_ARG
    with pytest.raises(P.Hlc2Error):
        P.crossmatch(good, good, 1.0, 7)
    # grid_like with a catalogue outside that grid's RA box
    w = S.config(1, scale=0.05)
    box = P.hlc2_build_index(*dev(w.A), opts=P.make_opts(1.0))
    far = S.Catalogue(np.array([10.0]), np.array([1.0]), np.array([1], np.int64))
    with pytest.raises(P.Hlc2Error) as e:
        P.hlc2_build_index(*dev(far), opts=P.make_opts(1.0), like=box)
    assert e.value.status == P.HLC2_ERR_GRID_MISMATCH


def test_launch_counter_moves(P):
    w = S.config(1, scale=0.05)
    n0 = P.kernel_launches()
    gpu_match(P, w.A, w.B, 1.0, 0)
    assert P.kernel_launches() - n0 >= 10


def test_match_kernel_events(P):
    """hlc2_crossmatch_events records the caller's events around k_match on the caller's stream; results are unaffected."""
    import torch
    w = S.config(1, scale=0.3)
    ga, gb, gs, ia, ib = gpu_match(P, w.A, w.B, w.radius_arcsec, 0)
    cap = len(ga) + 10
    oa = torch.empty(cap, dtype=torch.int64, device="cuda"); ob = torch.empty_like(oa)
    os_ = torch.empty(cap, dtype=torch.float64, device="cuda"); cnt = torch.zeros(1, dtype=torch.int64, device="cuda")
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(); e1.record()
    P.hlc2_crossmatch(ia, ib, w.radius_arcsec, 0, oa, ob, os_, cnt, events=(e0, e1))
    e1.synchronize()
    ms = e0.elapsed_time(e1)
    assert 0.0 < ms < 50.0 and int(cnt.item()) == len(ga)
