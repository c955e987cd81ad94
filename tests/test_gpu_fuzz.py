"""Randomised parity: patches, a box across the RA seam, both polar caps and the full sky, random sizes (3e2 .. 2e5),
density ratios and radii (0.05 .. 300 arcsec, capped so that a case holds at most ~2e6 chance pairs), both modes, against
the oracle.  A contiguous range of seeds; the cases drive the
planner through wrap / ring jobs, chained jobs, exchanged roles and the general path in combinations the named
configurations do not reach."""
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


def make_case(seed):
    rng = np.random.default_rng(seed)
    kind = int(rng.integers(0, 5))
    na = int(10 ** rng.uniform(2.5, 5.3)); nb = int(10 ** rng.uniform(2.5, 5.3))
    r = float(10 ** rng.uniform(-0.5, 2.5))
    if kind == 0:
        ra0, d0, w = rng.uniform(0, 350), rng.uniform(-80, 70), 10 ** rng.uniform(-1, 1.3)
        box = (ra0, ra0 + w, d0, d0 + min(w, 89 - d0))
    elif kind == 1: box = (355.0, 365.0, -5.0, 5.0)          # across the seam (RA taken mod 360)
    elif kind == 2: box = (0.0, 360.0, 88.0, 90.0)           # polar caps
    elif kind == 3: box = (0.0, 360.0, -90.0, -87.0)
    else:           box = (0.0, 360.0, -90.0, 90.0)

    def cat(n, id0, step):
        ra, dec = S.uniform_patch(rng, n, *box)
        return S.Catalogue(np.mod(ra, 360.0), dec, np.arange(n, dtype=np.int64) * step + id0)
    # keep the expected number of chance pairs bounded (a 0.1-degree box with r = 300 arcsec would pair everything)
    area = max((box[1] - box[0]) * 3600.0 * (np.sin(np.deg2rad(box[3])) - np.sin(np.deg2rad(box[2]))) * 206264.8, 1.0)
    r = float(min(r, np.sqrt(2.0e6 * area / (np.pi * na * max(nb, 1)))))
    r = max(r, 0.05)
    A = cat(na, 10**12, 3)
    k = rng.random(na) < 0.6
    pr, pd = S.perturb(rng, A.ra[k], A.dec[k], r / 3)
    E = cat(nb, 0, 1)
    ra = np.concatenate([pr, E.ra]); dec = np.clip(np.concatenate([pd, E.dec]), -90.0, 90.0)
    B = S.Catalogue(ra, dec, np.arange(len(ra), dtype=np.int64) * 5 + 2 * 10**12)
    return A, B, r


@pytest.mark.parametrize("seed", list(range(1000, 1036)))
def test_random_geometry_parity(P, seed):
    import torch
    A, B, r = make_case(seed)
    dev = lambda c: (torch.from_numpy(c.ra).cuda(), torch.from_numpy(c.dec).cuda(), torch.from_numpy(c.id).cuda())
    ia = P.hlc2_build_index(*dev(A), opts=P.make_opts(r)); ib = P.hlc2_build_index(*dev(B), opts=P.make_opts(r))
    # A filed on B's grid as well (the same-grid path), when A fits inside B's RA box
    try:
        ia_same = P.hlc2_build_index(*dev(A), opts=P.make_opts(r), like=ib)
    except P.Hlc2Error as e:
        assert e.status == P.HLC2_ERR_GRID_MISMATCH
        ia_same = None
    sep_of = parity.make_sep_of(A, B)
    for mode in (0, 1):
        oa, ob, os_, _ = oracle.match(A.ra, A.dec, A.id, B.ra, B.dec, B.id, r, mode)
        cmp = parity.compare_nearest if mode else parity.compare_all_pairs
        for ixa in (ia, ia_same):
            if ixa is None:
                continue
            a, b, s = P.crossmatch(ixa, ib, r, mode, capacity=max(1024, 4 * max(len(A), len(B))))
            rep = cmp((a.cpu().numpy(), b.cpu().numpy(), s.cpu().numpy()), (oa, ob, os_), r, sep_of)
            assert len(rep["borderline"]) <= 2
