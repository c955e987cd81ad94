"""Parity on inputs built to drive the match through each of its paths: chained jobs (windows
larger than one shared-memory stage), the general per-lane path (a tile reaching more than 8 zones of B's grid),
exchanged roles (B much smaller than A), wrap / ring jobs, nearest mode across the jobs of a tile."""
import numpy as np
import pytest

import hlc2_synth as S
import oracle
from tests import parity

pytestmark = pytest.mark.gpu

JOB_WORDS = 32
F_DIRECT, F_RING, F_WRAP = 1 << 8, 1 << 9, 1 << 10


@pytest.fixture(scope="module")
def P():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("gpu tests selected but no CUDA device")
    import paper_2301_07331_b200 as P
    from paper_2301_07331_b200 import build
    build.build()
    return P


def patch(rng, n, ra0, ra1, d0, d1, id0):
    ra, dec = S.uniform_patch(rng, n, ra0, ra1, d0, d1)
    return S.Catalogue(ra, dec, np.arange(n, dtype=np.int64) * 3 + id0)


def run(P, A, B, radius, mode):
    """-> (gpu rows, job flag words of the first jobs, number of chained jobs)"""
    import torch
    dev = lambda c: (torch.from_numpy(c.ra).cuda(), torch.from_numpy(c.dec).cuda(), torch.from_numpy(c.id).cuda())
    # white-box tests of the general (two-grid) path: square cells, and B's occupancy a little off A's so that two
    # catalogues of equal size never end up on structurally identical grids (which would take the same-grid path)
    ia = P.hlc2_build_index(*dev(A), opts=P.make_opts(radius, zone_aspect=1))
    ib = P.hlc2_build_index(*dev(B), opts=P.make_opts(radius, zone_aspect=1, target_occupancy=0.8))
    need = P.hlc2_crossmatch_sizes(ia, ib)
    temp = torch.zeros(need, dtype=torch.uint8, device="cuda")
    cap = 4 * max(len(A), len(B)) + 1024
    oa = torch.empty(cap, dtype=torch.int64, device="cuda"); ob = torch.empty_like(oa)
    os_ = torch.empty(cap, dtype=torch.float64, device="cuda"); cnt = torch.zeros(1, dtype=torch.int64, device="cuda")
    P.hlc2_crossmatch(ia, ib, radius, mode, oa, ob, os_, cnt, temp=temp)
    n = int(cnt.item()); assert n <= cap
    # white box: the scratch is a 256-byte header (counter of chained jobs) followed by 128-byte job records
    words = temp[256:].view(torch.int32).view(-1, JOB_WORDS).cpu().numpy().view(np.uint32)
    pool_n = int(temp[:4].view(torch.int32).item())
    live = words[words[:, 1] > 0]
    return (oa[:n].cpu().numpy(), ob[:n].cpu().numpy(), os_[:n].cpu().numpy()), live[:, 2], pool_n


def check(P, A, B, radius, mode):
    got, flags, pool_n = run(P, A, B, radius, mode)
    ora = oracle.match(A.ra, A.dec, A.id, B.ra, B.dec, B.id, radius, mode)[:3]
    cmp = parity.compare_nearest if mode == 1 else parity.compare_all_pairs
    rep = cmp(got, ora, radius, parity.make_sep_of(A, B))
    assert len(rep["borderline"]) <= 2
    return rep, flags, pool_n


def copies_plus(rng, A, frac, sigma, extra, id0, box):
    k = rng.random(len(A)) < frac
    pr, pd = S.perturb(rng, A.ra[k], A.dec[k], sigma)
    e = patch(rng, extra, *box, 0)
    ra = np.concatenate([pr, e.ra]); dec = np.concatenate([pd, e.dec])
    o = rng.permutation(len(ra))
    return S.Catalogue(ra[o], dec[o], np.arange(len(ra), dtype=np.int64) * 5 + id0)


@pytest.mark.parametrize("mode", [0, 1])
def test_chained_jobs_dense_b(P, mode):
    """B 20x denser than A: a tile's window holds thousands of B rows -> many jobs per tile, nearest carried across."""
    rng = np.random.default_rng(21)
    box = (40.0, 41.0, -10.0, -9.0)
    A = patch(rng, 6_000, *box, 10**12)
    B = copies_plus(rng, A, 0.7, 0.4, 120_000, 2 * 10**12, box)
    rep, flags, pool_n = check(P, A, B, 2.0, mode)
    assert rep["n_gpu"] > 3_500
    assert pool_n > 50 and not (flags & F_DIRECT).any()


@pytest.mark.parametrize("mode", [0, 1])
def test_general_path_many_zones(P, mode):
    """B ~1000x denser than A: an A zone covers more than 8 zones of B's grid -> the general per-lane path."""
    rng = np.random.default_rng(22)
    box = (200.0, 202.0, 30.0, 32.0)
    A = patch(rng, 400, *box, 10**12)
    B = copies_plus(rng, A, 0.8, 0.5, 400_000, 2 * 10**12, box)
    rep, flags, pool_n = check(P, A, B, 2.5, mode)
    assert rep["n_gpu"] > 250
    assert (flags & F_DIRECT).any()


def test_exchanged_roles_small_b(P):
    """all_pairs with B more than 3x smaller than A: B rows drive the lanes, the id columns come back in place."""
    w = S.config(2, scale=0.02)                     # 2e5 x 2e5 full sky
    rng = np.random.default_rng(23)
    keep = rng.random(len(w.B)) < 0.2
    B = w.B.take(np.flatnonzero(keep))
    rep, flags, pool_n = check(P, w.A, B, w.radius_arcsec, 0)
    assert rep["n_gpu"] > 20_000
    # the same pairs with the arguments exchanged by the caller
    got2, _, _ = run(P, B, w.A, w.radius_arcsec, 0)
    assert set(zip(got2[1].tolist(), got2[0].tolist())) == set(zip(*[x.tolist() for x in run(P, w.A, B, w.radius_arcsec, 0)[0][:2]]))


@pytest.mark.parametrize("mode", [0, 1])
def test_wrap_and_ring_jobs_are_staged(P, mode):
    """Full-sky catalogues: tiles at the RA seam produce WRAP jobs, polar tiles RING jobs, (almost) none falls back."""
    w = S.config(2, scale=0.03)
    rep, flags, pool_n = check(P, w.A, w.B, w.radius_arcsec, mode)
    # (a seam tile whose two window images meet in a few-cell polar zone takes the general path: a handful at most)
    assert (flags & F_WRAP).any() and (flags & F_RING).any() and ((flags & F_DIRECT) != 0).sum() <= 8


def test_cfg3_nearest_scaled(P):
    w = S.config(3, scale=0.004)
    rep, _, _ = check(P, w.A, w.B, w.radius_arcsec, 1)
    assert rep["n_gpu"] > 100_000
