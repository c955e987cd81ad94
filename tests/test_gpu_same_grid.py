"""Parity on inputs built to drive the same-grid match (csrc/hlc2_match_same.cu) through each of its
paths: row chunks (a piece larger than a stage), the neighbour-zone stages, wide tiles (a tile spanning more cells than a
stage holds), general rows, explicit zone aspects, a second pair for one A row within a tile, output capacity overflow."""
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


def patch(rng, n, box, id0, step=3):
    ra, dec = S.uniform_patch(rng, n, *box)
    return S.Catalogue(ra, dec, np.arange(n, dtype=np.int64) * step + id0)


def check_same(P, A, B, r, opts_b, modes=(0, 1), engine=oracle.ENGINE_VOXEL, min_rows=1):
    ib = P.hlc2_build_index(*dev(B), opts=opts_b)
    ia = P.hlc2_build_index(*dev(A), opts=P.make_opts(r), like=ib)
    flags = (P.hlc2_index_arrays(ia)["cell_key"].cpu().numpy().view(np.uint32) >> 28)
    sep_of = parity.make_sep_of(A, B)
    out = {}
    for mode in modes:
        a, b, s = P.crossmatch(ia, ib, r, mode, capacity=8 * max(len(A), len(B)) + 1024)
        oa, ob, os_, _ = oracle.match(A.ra, A.dec, A.id, B.ra, B.dec, B.id, r, mode, engine)
        cmp = parity.compare_nearest if mode else parity.compare_all_pairs
        rep = cmp((a.cpu().numpy(), b.cpu().numpy(), s.cpu().numpy()), (oa, ob, os_), r, sep_of)
        assert len(rep["borderline"]) <= 2 and rep["n_gpu"] >= min_rows
        out[mode] = rep
    return out, flags, P.hlc2_grid_describe(ib)


def test_dense_b_cells_are_cut_into_row_chunks(P):
    """B 30x denser than the grid's cells were planned for (the grid is B's own at occupancy 40): a tile's own-zone piece
    and its neighbour-zone pieces hold thousands of rows -> many 96-row chunks per piece, nearest carried across them."""
    rng = np.random.default_rng(31)
    box = (50.0, 50.6, 10.0, 10.6)
    A = patch(rng, 20_000, box, 10**12)
    pr, pd = S.perturb(rng, A.ra, A.dec, 0.5)
    e = patch(rng, 200_000, box, 0)
    B = S.Catalogue(np.concatenate([pr, e.ra]), np.concatenate([pd, e.dec]), np.arange(len(pr) + len(e), dtype=np.int64) * 5 + 2 * 10**12)
    rep, flags, g = check_same(P, A, B, 2.0, P.make_opts(2.0, target_occupancy=40.0), min_rows=15_000)
    assert len(B) / g["n_cells"] > 20                      # tens of rows per cell: pieces of several hundred rows
    assert ((flags >> 2) & 3 != 0).sum() > 50              # rows that reach a neighbouring zone exist


def test_sparse_a_tiles_span_more_cells_than_a_stage(P):
    """A 500x sparser than B on B's grid: 128 consecutive A rows span thousands of cells -> the tile's rows read
    cell_start and B through global memory (no staged slice)."""
    rng = np.random.default_rng(32)
    box = (120.0, 124.0, -40.0, -36.0)
    B = patch(rng, 400_000, box, 2 * 10**12, 5)
    k = rng.choice(len(B), 800, replace=False)
    pr, pd = S.perturb(rng, B.ra[k], B.dec[k], 0.4)
    A = S.Catalogue(pr, pd, np.arange(800, dtype=np.int64) * 3 + 10**12)
    rep, flags, g = check_same(P, A, B, 1.5, P.make_opts(1.5), min_rows=700)
    assert g["n_cells"] / len(A) > 520                     # > 512 cells per A row on average: wider than a stage's slice


@pytest.mark.parametrize("aspect", [1, 4, 32])
def test_explicit_zone_aspects(P, aspect):
    w = S.config(1, scale=0.5)
    rep, flags, g = check_same(P, w.A, w.B, w.radius_arcsec, P.make_opts(w.radius_arcsec, zone_aspect=aspect), min_rows=35_000)
    top = g["dec_lo"] + g["zone_h"]                        # poleward edge of zone 0 (the patch lies north of the equator)
    cell_w = g["span"] * 3600.0 * np.cos(np.deg2rad(top)) / g["n_ra"][0]
    a_eff = min(aspect, g["cell_arcsec"] / w.radius_arcsec)
    assert cell_w >= w.radius_arcsec * (1 - 1e-9)          # cells never narrower than r_max, zones a_eff^2 times as high as wide
    assert 0.5 * a_eff ** 2 < g["zone_h"] * 3600.0 / cell_w < 2.0 * a_eff ** 2


def test_ra_concentrated_catalogue_gets_square_cells(P):
    """The automatic aspect is scaled back when the coarse RA histogram shows a dense strip along a meridian."""
    import torch
    rng = np.random.default_rng(33)
    ra_u, dec_u = S.uniform_sphere(rng, 300_000)
    dec_s = np.rad2deg(np.arcsin(rng.uniform(-0.99, 0.99, 100_000)))
    ra_s = np.mod(rng.uniform(-6.0, 6.0, 100_000) / 3600.0 / np.cos(np.deg2rad(dec_s)), 360.0)
    uni = P.hlc2_grid_describe(P.hlc2_build_index(torch.from_numpy(ra_u).cuda(), torch.from_numpy(dec_u).cuda(), None, opts=P.make_opts(3.0)))
    mix = P.hlc2_grid_describe(P.hlc2_build_index(torch.from_numpy(np.concatenate([ra_u, ra_s])).cuda(),
                                                  torch.from_numpy(np.concatenate([dec_u, dec_s])).cuda(), None, opts=P.make_opts(3.0)))
    assert uni["zone_h"] * 3600.0 > 8.0 * uni["cell_arcsec"] and mix["zone_h"] * 3600.0 < 1.6 * mix["cell_arcsec"]


def test_several_pairs_per_row_and_capacity_overflow(P):
    """Five B copies of every A source: a lane holds its first pair, the others go straight out; with a capacity below
    the result the count is still the full one and the rows written are valid pairs."""
    import torch
    rng = np.random.default_rng(34)
    box = (10.0, 11.0, 60.0, 61.0)
    A = patch(rng, 30_000, box, 10**12)
    parts = [S.perturb(rng, A.ra, A.dec, 0.3) for _ in range(5)]
    B = S.Catalogue(np.concatenate([p[0] for p in parts]), np.concatenate([p[1] for p in parts]), np.arange(5 * len(A), dtype=np.int64) * 5 + 2 * 10**12)
    rep, _, _ = check_same(P, A, B, 1.5, P.make_opts(1.5), modes=(0, 1), min_rows=29_000)
    assert rep[0]["n_gpu"] > 140_000
    ib = P.hlc2_build_index(*dev(B), opts=P.make_opts(1.5)); ia = P.hlc2_build_index(*dev(A), opts=P.make_opts(1.5), like=ib)
    cap = 50_000
    oa = torch.full((cap,), -1, dtype=torch.int64, device="cuda"); ob = torch.full_like(oa, -1); os_ = torch.full((cap,), -1.0, dtype=torch.float64, device="cuda")
    cnt = torch.zeros(1, dtype=torch.int64, device="cuda")
    P.hlc2_crossmatch(ia, ib, 1.5, 0, oa, ob, os_, cnt)
    assert int(cnt.item()) == rep[0]["n_gpu"]
    oa_, ob_, os2, _ = oracle.match(A.ra, A.dec, A.id, B.ra, B.dec, B.id, 1.5, 0)
    truth = set(zip(oa_.tolist(), ob_.tolist()))
    got = list(zip(oa.cpu().tolist(), ob.cpu().tolist()))
    assert all(g in truth for g in got) and len(set(got)) == cap
