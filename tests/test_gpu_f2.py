"""Self-match of one catalogue and per-record error radii (PAPER.md D4 L286 / L295, Eq. (4)) against
the oracle's extensions (oracle.match(..., self_mode=, err_a=, err_b=)), through the C ABI."""
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


def dev(*arrs):
    import torch
    return tuple(torch.from_numpy(np.ascontiguousarray(a)).cuda() for a in arrs)


def unordered(a, b, s):
    """(idA, idB, sep) rows with every pair written smaller id first."""
    lo, hi = np.minimum(a, b), np.maximum(a, b)
    return lo, hi, s


def _cat(seed=5, n=60_000, dup=300, box=(100.0, 101.0, -30.0, -29.0)):
    rng = np.random.default_rng(seed)
    ra, dec = S.uniform_patch(rng, n, *box)
    pr, pd = S.perturb(rng, ra[: n // 2], dec[: n // 2], 0.6)                # companions within a few arcsec
    ra = np.concatenate([ra, pr, ra[:dup]]); dec = np.concatenate([dec, pd, dec[:dup]])      # + exact duplicates
    o = rng.permutation(len(ra))
    return S.Catalogue(ra[o], dec[o], np.arange(len(ra), dtype=np.int64))


@pytest.mark.parametrize("kw", [{}, {"zone_aspect": 1, "cell_arcsec": 2.5}], ids=["same-grid kernel", "per-lane path (zones 1 r high)"])
def test_selfmatch_all_pairs(P, kw):
    c = _cat()
    r = 2.5
    idx = P.hlc2_build_index(*dev(c.ra, c.dec, c.id), opts=P.make_opts(r, **kw))
    for include_self in (False, True):
        ga, gb, gs = (t.cpu().numpy() for t in P.selfmatch(idx, r, P.HLC2_ALL_PAIRS, include_self=include_self, capacity=4 * len(c)))
        oa, ob, os_, _ = oracle.match(c.ra, c.dec, c.id, c.ra, c.dec, c.id, r, 0, oracle.ENGINE_VOXEL,
                                      self_mode=oracle.SELF_PAIRS_AND_DIAGONAL if include_self else oracle.SELF_PAIRS)
        rep = parity.compare_all_pairs(unordered(ga, gb, gs), unordered(oa, ob, os_), r, parity.make_sep_of(c, c))
        assert rep["n_gpu"] == rep["n_oracle"] + len(rep["borderline"]) or len(rep["borderline"]) <= 2
        assert rep["n_oracle"] > 30_000 + (len(c) if include_self else 0)
    # half of the ordinary cross-match of the catalogue with itself, diagonal removed
    fa, fb, fs = (t.cpu().numpy() for t in P.crossmatch(idx, idx, r, P.HLC2_ALL_PAIRS, capacity=8 * len(c)))
    assert (len(fa) - len(c)) // 2 == rep["n_gpu"] - len(c)


def test_selfmatch_nearest_excludes_the_source_itself(P):
    c = _cat(seed=6)
    r = 3.0
    idx = P.hlc2_build_index(*dev(c.ra, c.dec, c.id), opts=P.make_opts(r))
    ga, gb, gs = (t.cpu().numpy() for t in P.selfmatch(idx, r, P.HLC2_NEAREST))
    oa, ob, os_, _ = oracle.match(c.ra, c.dec, c.id, c.ra, c.dec, c.id, r, 1, oracle.ENGINE_VOXEL, self_mode=oracle.SELF_EXCLUDE_OWN)
    rep = parity.compare_nearest((ga, gb, gs), (oa, ob, os_), r, parity.make_sep_of(c, c))
    assert (ga != gb).all() and rep["n_gpu"] > 30_000


def test_selfmatch_full_sky_poles_and_seam(P):
    """General rows (polar, RA seam) of a self-match go through the follow-up kernel: still every pair once."""
    rng = np.random.default_rng(8)
    ra = np.concatenate([rng.uniform(0, 360, 3000), rng.uniform(-0.003, 0.003, 400) % 360.0, rng.uniform(0, 360, 600)])
    dec = np.concatenate([np.rad2deg(np.arcsin(rng.uniform(-1, 1, 3000))), rng.uniform(-1, 1, 400), np.where(rng.random(600) < 0.5, 1, -1) * (90.0 - np.abs(rng.normal(0, 0.003, 600)))])
    c = S.Catalogue(ra, dec, np.arange(len(ra), dtype=np.int64))
    for r in (5.0, 60.0):
        idx = P.hlc2_build_index(*dev(c.ra, c.dec, c.id), opts=P.make_opts(r, full_sky=True))
        ga, gb, gs = (t.cpu().numpy() for t in P.selfmatch(idx, r, capacity=1 << 20))
        oa, ob, os_, _ = oracle.match(c.ra, c.dec, c.id, c.ra, c.dec, c.id, r, 0, oracle.ENGINE_BRUTE, self_mode=1)
        rep = parity.compare_all_pairs(unordered(ga, gb, gs), unordered(oa, ob, os_), r, parity.make_sep_of(c, c))
        assert rep["n_oracle"] > 100


@pytest.mark.parametrize("mode", [0, 1])
def test_crossmatch_radii_is_eq4_per_pair(P, mode):
    w = S.config(1, scale=0.5)
    rng = np.random.default_rng(44)
    ea = rng.uniform(0.02, 0.35, len(w.A)); eb = rng.uniform(0.02, 0.35, len(w.B))
    cap_r = 3.0 * np.sqrt(0.35 ** 2 + 0.35 ** 2) + 1e-6                         # the largest threshold any pair can have
    ia = P.hlc2_build_index(*dev(w.A.ra, w.A.dec, w.A.id), opts=P.make_opts(cap_r), err_arcsec=dev(ea)[0])
    ib = P.hlc2_build_index(*dev(w.B.ra, w.B.dec, w.B.id), opts=P.make_opts(cap_r), err_arcsec=dev(eb)[0])
    for k in (3.0, 1.5):
        ga, gb, gs = (t.cpu().numpy() for t in P.crossmatch_radii(ia, ib, cap_r, k, mode, capacity=4 * len(w.A)))
        oa, ob, os_, _ = oracle.match(w.A.ra, w.A.dec, w.A.id, w.B.ra, w.B.dec, w.B.id, cap_r, mode, oracle.ENGINE_VOXEL,
                                      err_a=ea, err_b=eb, k_factor=k)
        # borderline = within 1e-9 arcsec of the PAIR's threshold: classify with the oracle's separation
        ia_row = {int(v): i for i, v in enumerate(w.A.id)}; ib_row = {int(v): i for i, v in enumerate(w.B.id)}
        thr = lambda a, b: min(cap_r, k * float(np.hypot(ea[ia_row[int(a)]], eb[ib_row[int(b)]])))
        gset = {(int(a), int(b)): s for a, b, s in zip(ga, gb, gs)}; oset = {(int(a), int(b)): s for a, b, s in zip(oa, ob, os_)}
        assert len(gset) == len(ga)
        if mode == 0:
            for key in set(gset) ^ set(oset):
                sep = oracle.sep_arcsec(w.A.ra[ia_row[key[0]]], w.A.dec[ia_row[key[0]]], w.B.ra[ib_row[key[1]]], w.B.dec[ib_row[key[1]]])
                assert abs(sep - thr(*key)) < 1e-9, (key, sep, thr(*key))
            common = set(gset) & set(oset)
            assert len(common) > 10_000 and max(abs(gset[q] - oset[q]) for q in common) < 1e-9
        else:
            assert len(gset) == len(oset) and sum(1 for q in gset if q not in oset) <= 2
    with pytest.raises(P.Hlc2Error):                                          # an index without radii is refused
        P.crossmatch_radii(P.hlc2_build_index(*dev(w.A.ra, w.A.dec, w.A.id), opts=P.make_opts(cap_r)), ib, cap_r)
