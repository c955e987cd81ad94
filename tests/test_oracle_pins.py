"""Pins of the CPU oracle against things other than itself (CPU only).

Each test states what a plausible mistake it would catch.  Citations: PAPER.md lines
(P:L..), north_star (NS) of BASELINE.json, DESIGN.md readings.
"""
import os

import mpmath as mp
import numpy as np
import pytest

import hlc2_synth as S
import oracle

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")
mp.mp.dps = 50


def mp_sep_eq1(ra1, dec1, ra2, dec2):
    """PAPER.md Eq. (1), the law of spherical cosines, at 50 digits, arcsec.
    Inputs are the exact fp64 values."""
    d2r = mp.pi / 180
    a1, d1, a2, d2 = (mp.mpf(float(v)) * d2r for v in (ra1, dec1, ra2, dec2))
    c = mp.sin(d1) * mp.sin(d2) + mp.cos(d1) * mp.cos(d2) * mp.cos(a1 - a2)
    c = max(min(c, mp.mpf(1)), mp.mpf(-1))
    return mp.acos(c) * 648000 / mp.pi


def mp_sep_vincenty(ra1, dec1, ra2, dec2):
    """A third algebraic form (atan2 of the cross/dot products), 50 digits, arcsec."""
    d2r = mp.pi / 180
    a1, d1, a2, d2 = (mp.mpf(float(v)) * d2r for v in (ra1, dec1, ra2, dec2))
    da = a1 - a2
    num = mp.sqrt((mp.cos(d2) * mp.sin(da)) ** 2 +
                  (mp.cos(d1) * mp.sin(d2) - mp.sin(d1) * mp.cos(d2) * mp.cos(da)) ** 2)
    den = mp.sin(d1) * mp.sin(d2) + mp.cos(d1) * mp.cos(d2) * mp.cos(da)
    return mp.atan2(num, den) * 648000 / mp.pi


def oracle_sep_mp(ra1, dec1, ra2, dec2):
    hi, lo = oracle.sep_arcsec_hilo(ra1, dec1, ra2, dec2)
    return mp.mpf(hi) + mp.mpf(lo)


def _pairs_close(rng, n, sep_arcsec, dec_lo, dec_hi, ra_lo=0.0, ra_hi=360.0):
    ra = rng.uniform(ra_lo, ra_hi, n)
    dec = rng.uniform(dec_lo, dec_hi, n)
    ra2, dec2 = S.perturb(rng, ra, dec, sep_arcsec)
    return ra, dec, ra2, dec2


# ----------------------------------------------------------------------------- separation
def test_golden_closed_forms():
    """Hand-derived textbook angles of Eq. (1): catches a wrong sign, a dropped cos(dec) factor,
    degrees/radians mix-ups, a missing modulo on RA, transposed arguments."""
    rows = [l.split("#")[0].split() for l in open(os.path.join(GOLDEN, "sep_closed_forms.txt"))]
    rows = [list(map(float, r)) for r in rows if len(r) == 5]
    assert len(rows) >= 12
    for ra1, d1, ra2, d2, want in rows:
        got = oracle.sep_arcsec(ra1, d1, ra2, d2)
        assert abs(got - want) <= 1e-10 * max(1.0, want / 3600.0), (ra1, d1, ra2, d2, got, want)
        # the 180-degree cases sit on asin's vertical tangent: allow its rounding there only
        assert abs(oracle.sep_arcsec(ra2, d2, ra1, d1) - got) <= 1e-9


@pytest.mark.parametrize("case", ["fullsky", "close", "seam", "polar", "very_polar"])
def test_sep_matches_eq1_at_50_digits(case):
    """Oracle haversine == Eq. (1) == Vincenty form at 50 digits to 1e-12 arcsec on the exact fp64
    inputs: catches any algebraic slip in the haversine restatement and loss of precision in the
    degree->radian path (a plain fp64 haversine fails this at ~2e-10 arcsec)."""
    rng = np.random.default_rng(7331)
    n = 300
    if case == "fullsky":
        ra, dec = S.uniform_sphere(rng, n); ra2, dec2 = S.uniform_sphere(rng, n)
    elif case == "close":
        ra, dec, ra2, dec2 = _pairs_close(rng, n, 1.5, -85, 85)
    elif case == "seam":
        ra, dec, ra2, dec2 = _pairs_close(rng, n, 2.0, -80, 80, -0.0003, 0.0003)
        ra = np.mod(ra, 360.0)
    elif case == "polar":
        ra, dec, ra2, dec2 = _pairs_close(rng, n, 2.0, 89.5, 90.0)
    else:
        ra, dec, ra2, dec2 = _pairs_close(rng, n, 1.0, 89.999, 90.0)
        dec = -dec; dec2 = -dec2
    worst = 0
    for k in range(n):
        o = oracle_sep_mp(ra[k], dec[k], ra2[k], dec2[k])
        v = mp_sep_vincenty(ra[k], dec[k], ra2[k], dec2[k])
        worst = max(worst, abs(o - v))
        assert abs(o - v) < mp.mpf("1e-12"), (case, k, o, v)
        e1 = mp_sep_eq1(ra[k], dec[k], ra2[k], dec2[k])
        assert abs(e1 - v) < mp.mpf("1e-20")          # the two 50-digit forms are the same quantity
    assert worst < mp.mpf("1e-12")


def test_small_angle_eq3_sanity():
    """Eq. (3) agrees with the oracle to ~1e-9 arcsec for arcsec pairs at |dec| <= 60 and
    is expected to drift toward the poles (the reason Eq. (1) is the definition, reading 1)."""
    rng = np.random.default_rng(3)
    ra, dec, ra2, dec2 = _pairs_close(rng, 2000, 1.0, -60, 60, 1.0, 359.0)
    dbar = np.deg2rad(0.5 * (dec + dec2))
    d3 = np.sqrt(((ra - ra2) * np.cos(dbar)) ** 2 + (dec - dec2) ** 2) * 3600.0
    d1 = np.array([oracle.sep_arcsec(*v) for v in zip(ra, dec, ra2, dec2)])
    assert np.max(np.abs(d3 - d1)) < 5e-9
    ra, dec, ra2, dec2 = _pairs_close(rng, 500, 1.0, 89.9, 89.99, 1.0, 359.0)
    dbar = np.deg2rad(0.5 * (dec + dec2))
    d3 = np.sqrt(((ra - ra2) * np.cos(dbar)) ** 2 + (dec - dec2) ** 2) * 3600.0
    d1 = np.array([oracle.sep_arcsec(*v) for v in zip(ra, dec, ra2, dec2)])
    assert np.max(np.abs(d3 - d1)) > 1e-8        # Eq. (3) is not usable at the 1e-9 bar there


def test_ra_periodic_and_pole_degenerate():
    assert oracle.sep_arcsec(370.0, 12.0, 10.0, 12.0) == 0.0
    assert oracle.sep_arcsec(-350.0, 12.0, 10.0, 12.0) == 0.0
    assert oracle.sep_arcsec(0.0, 90.0, 271.3, 90.0) < 1e-13     # every RA is the same point at the pole


# ----------------------------------------------------------------------------- pair sets
def _tiny_inputs(seed=11):
    """Tiny catalogue covering both poles, the RA seam, exact duplicates and ordinary sky."""
    rng = np.random.default_rng(seed)
    ra = np.concatenate([rng.uniform(0, 360, 150), rng.uniform(-0.002, 0.002, 120) % 360.0,
                         rng.uniform(0, 360, 100), rng.uniform(0, 360, 100), [0.0, 360.0, 10.0, 10.0]])
    dec = np.concatenate([np.rad2deg(np.arcsin(rng.uniform(-1, 1, 150))), rng.uniform(-0.002, 0.002, 120),
                          90.0 - np.abs(rng.normal(0, 0.001, 100)), -90.0 + np.abs(rng.normal(0, 0.001, 100)),
                          [90.0, -90.0, 20.0, 20.0]])
    ra_b, dec_b = S.perturb(rng, ra, dec, 1.5)
    ra_b = np.concatenate([ra_b, ra[:50]]); dec_b = np.concatenate([dec_b, dec[:50]])    # exact copies too
    return ra, dec, ra_b, dec_b


@pytest.mark.parametrize("mode", [oracle.ALL_PAIRS, oracle.NEAREST])
def test_engines_agree_on_tiny_inputs(mode):
    """Voxel-hash engine == brute force with pre-filter == brute force all-long-double, on inputs with
    poles, seam and duplicates: catches a dropped neighbour voxel, a too-tight pre-filter, a wrong key."""
    ra, dec, ra_b, dec_b = _tiny_inputs()
    for r in (0.5, 3.0, 40.0, 3000.0):
        res = [oracle.match(ra, dec, None, ra_b, dec_b, None, r, mode, e) for e in (0, 1, 2)]
        for k in (1, 2):
            assert np.array_equal(res[0][0], res[k][0]) and np.array_equal(res[0][1], res[k][1]), (r, k)
            assert np.array_equal(res[0][2], res[k][2])
        assert len(res[0][0]) > 0


def test_brute_force_is_the_definition():
    """Engine 0 against a direct transcription of the definition in Python over the 50-digit Eq. (1)."""
    ra, dec, ra_b, dec_b = _tiny_inputs(5)
    ra, dec, ra_b, dec_b = ra[::9], dec[::9], ra_b[::7], dec_b[::7]
    r = 600.0
    want = [(i, j) for i in range(len(ra)) for j in range(len(ra_b))
            if mp_sep_eq1(ra[i], dec[i], ra_b[j], dec_b[j]) <= r]
    a, b, s, _ = oracle.match(ra, dec, None, ra_b, dec_b, None, r, oracle.ALL_PAIRS, 0)
    assert sorted(want) == list(zip(a.tolist(), b.tolist()))


def test_symmetry_and_selfmatch():
    """match(A,B) == transpose(match(B,A)); match(A,A) holds every (i,i) at 0 (D4 self-match)."""
    w = S.config(1, scale=0.05)
    A, B, r = w.A, w.B, w.radius_arcsec
    a, b, s, _ = oracle.match(A.ra, A.dec, A.id, B.ra, B.dec, B.id, r)
    b2, a2, s2, _ = oracle.match(B.ra, B.dec, B.id, A.ra, A.dec, A.id, r)
    o = np.lexsort((b2, a2))
    assert np.array_equal(a, a2[o]) and np.array_equal(b, b2[o]) and np.allclose(s, s2[o], atol=1e-12, rtol=0)
    a, b, s, _ = oracle.match(A.ra, A.dec, A.id, A.ra, A.dec, A.id, r)
    diag = a == b
    assert diag.sum() == len(A) and np.all(s[diag] == 0.0)


@pytest.mark.parametrize("cfg,scale", [(1, 0.2), (2, 0.01), (3, 0.002), (4, 0.005)])
def test_planted_truth_is_found(cfg, scale):
    """Every planted (parent, copy) whose separation is <= r must be in the result; and the fraction
    inside r matches the Rayleigh law 1 - exp(-r^2 / 2 sigma^2) of the generator."""
    w = S.config(cfg, scale=scale)
    A, B, r = w.A, w.B, w.radius_arcsec
    a, b, s, _ = oracle.match(A.ra, A.dec, A.id, B.ra, B.dec, B.id, r)
    got = set(zip(a.tolist(), b.tolist()))
    sep = np.array([oracle.sep_arcsec(A.ra[i], A.dec[i], B.ra[j], B.dec[j])
                    for i, j in zip(w.planted_a, w.planted_b)])
    inside = sep <= r
    for i, j in zip(w.planted_a[inside], w.planted_b[inside]):
        assert (int(A.id[i]), int(B.id[j])) in got
    p = 1.0 - np.exp(-r * r / (2 * w.sigma_arcsec ** 2))
    n = len(sep)
    assert abs(inside.mean() - p) < 5 * np.sqrt(max(p * (1 - p), 1e-6) / n) + 1e-3


def test_chance_pair_count_is_poisson():
    """Two independent uniform catalogues: E[pairs] = N_A N_B (1 - cos r)/2 (cap area fraction).
    Catches systematically lost neighbours (a missing voxel column loses ~1/3 of these)."""
    rng = np.random.default_rng(99)
    n = 150_000
    ra, dec = S.uniform_sphere(rng, n); ra_b, dec_b = S.uniform_sphere(rng, n)
    r = 90.0
    a, b, s, _ = oracle.match(ra, dec, None, ra_b, dec_b, None, r)
    lam = n * n * (1 - np.cos(np.deg2rad(r / 3600.0))) / 2
    assert abs(len(a) - lam) < 5 * np.sqrt(lam), (len(a), lam)
    # separations of chance pairs are distributed with density ~ s: mean = 2r/3
    assert abs(s.mean() - 2 * r / 3) < 5 * (r / np.sqrt(18)) / np.sqrt(len(s))


def _rotate(ra, dec, R):
    a, d = np.deg2rad(ra), np.deg2rad(dec)
    v = np.stack([np.cos(d) * np.cos(a), np.cos(d) * np.sin(a), np.sin(d)])
    x, y, z = R @ v
    return np.mod(np.rad2deg(np.arctan2(y, x)), 360.0), np.rad2deg(np.arctan2(z, np.hypot(x, y)))


def test_rotation_invariance():
    """Moving the patch of config 1 onto the north pole and across RA = 0 preserves the pair set (up to
    pairs within 1e-6 arcsec of r, which re-rounding the rotated coordinates may flip)."""
    w = S.config(1, scale=0.05)
    A, B, r = w.A, w.B, w.radius_arcsec
    a0, b0, s0, _ = oracle.match(A.ra, A.dec, A.id, B.ra, B.dec, B.id, r)
    th = np.deg2rad(89.0)       # patch centre (181, 1) -> the pole
    Rz = lambda t: np.array([[np.cos(t), -np.sin(t), 0], [np.sin(t), np.cos(t), 0], [0, 0, 1]])
    Ry = lambda t: np.array([[np.cos(t), 0, -np.sin(t)], [0, 1, 0], [np.sin(t), 0, np.cos(t)]])
    for R in (Ry(th) @ Rz(np.deg2rad(-181.0)), Rz(np.deg2rad(179.0))):
        ra_a, dec_a = _rotate(A.ra, A.dec, R); ra_b, dec_b = _rotate(B.ra, B.dec, R)
        a1, b1, s1, _ = oracle.match(ra_a, dec_a, A.id, ra_b, dec_b, B.id, r)
        p0 = {(x, y): z for x, y, z in zip(a0.tolist(), b0.tolist(), s0.tolist())}
        p1 = {(x, y): z for x, y, z in zip(a1.tolist(), b1.tolist(), s1.tolist())}
        for k in set(p0) ^ set(p1):
            z = p0.get(k, p1.get(k))
            assert abs(z - r) < 1e-6
        common = set(p0) & set(p1)
        assert len(common) > 0.99 * len(p0)
        assert max(abs(p0[k] - p1[k]) for k in common) < 1e-8     # fp64 rotation noise, not oracle error


def test_inclusive_threshold_either_side():
    """Eq. (4) is inclusive.  Two equator points 2^-10 deg = 3.515625 arcsec apart (exact):
    in at r = sep + 2e-9, out at r = sep - 2e-9.  (Exactly at r it is exempt by NS: parity-unpinned.)"""
    ra = np.array([100.0]); dec = np.array([0.0])
    ra_b = np.array([100.0 + 2.0 ** -10]); dec_b = np.array([0.0])
    sep = 3.515625
    assert oracle.sep_arcsec(ra[0], 0.0, ra_b[0], 0.0) == pytest.approx(sep, abs=1e-13)
    for eng in (0, 1, 2):
        assert len(oracle.match(ra, dec, None, ra_b, dec_b, None, sep + 2e-9, 0, eng)[0]) == 1
        assert len(oracle.match(ra, dec, None, ra_b, dec_b, None, sep - 2e-9, 0, eng)[0]) == 0
        assert len(oracle.match(ra, dec, None, ra_b, dec_b, None, sep, 0, eng)[0]) == 1    # inclusive reading


def test_nearest_is_argmin_of_all_pairs():
    w = S.config(4, scale=0.002)
    A, B, r = w.A, w.B, 30.0
    a, b, s, _ = oracle.match(A.ra, A.dec, A.id, B.ra, B.dec, B.id, r, oracle.ALL_PAIRS)
    na, nb, ns, _ = oracle.match(A.ra, A.dec, A.id, B.ra, B.dec, B.id, r, oracle.NEAREST)
    assert np.array_equal(na, np.unique(a))
    first = np.searchsorted(a, na)
    for k, lo in enumerate(first):
        hi = lo
        while hi < len(a) and a[hi] == na[k]:
            hi += 1
        j = lo + int(np.lexsort((b[lo:hi], s[lo:hi]))[0])
        assert nb[k] == b[j] and ns[k] == s[j]
    assert (np.diff(first) > 1).any()          # some rows really had a choice to make


def test_rejects_bad_input():
    ok = np.array([1.0]); z = np.array([0.0])
    for bad_dec in (90.0000001, -91.0, np.nan, np.inf):
        with pytest.raises(ValueError):
            oracle.match(ok, np.array([bad_dec]), None, ok, z, None, 1.0)
    with pytest.raises(ValueError):
        oracle.match(np.array([np.nan]), z, None, ok, z, None, 1.0)
    for bad_r in (0.0, -1.0, np.nan):
        with pytest.raises(ValueError):
            oracle.match(ok, z, None, ok, z, None, bad_r)
    a, b, s, _ = oracle.match(np.zeros(0), np.zeros(0), None, ok, z, None, 1.0)
    assert len(a) == 0


# ----------------------------------------------------------------------------- generators
def test_generators_are_seeded_and_shaped():
    w1 = S.config(3, scale=0.001); w2 = S.config(3, scale=0.001)
    assert np.array_equal(w1.A.ra, w2.A.ra) and np.array_equal(w1.B.dec, w2.B.dec)
    assert len(w1.A) == 100_000 and len(w1.B) == 50_000 and len(w1.planted_a) == 30_000
    assert w1.A.id[0] == 10**12 and w1.B.id[0] == 2 * 10**12 + 1
    assert (w1.A.ra >= 0).all() and (w1.A.ra < 360).all() and (np.abs(w1.A.dec) <= 90).all()
    # galactic-plane concentration: fraction of sources within |b| < 10 deg well above the uniform 17.4%
    w = S.config(4, scale=0.002)
    assert (np.abs(w.A.dec) > 89.5).mean() == pytest.approx(0.1, abs=0.01)


# ------------------------------------------------------------------------------------------------------
# extensions: per-record error radii (Eq. (4)) and self-match (L286, L295)
# ------------------------------------------------------------------------------------------------------
def _mp_sep_arcsec(ra1, dec1, ra2, dec2):
    """Eq. (1) itself (law of cosines) in 50-digit arithmetic -- not the oracle's haversine form."""
    import mpmath as mp
    mp.mp.dps = 50
    d2r = mp.pi / 180
    a1, d1, a2, d2 = (mp.mpf(float(v)) * d2r for v in (ra1, dec1, ra2, dec2))
    # Vincenty form of the same angle: well conditioned at arcsecond separations
    num = mp.sqrt((mp.cos(d2) * mp.sin(a2 - a1)) ** 2 + (mp.cos(d1) * mp.sin(d2) - mp.sin(d1) * mp.cos(d2) * mp.cos(a2 - a1)) ** 2)
    den = mp.sin(d1) * mp.sin(d2) + mp.cos(d1) * mp.cos(d2) * mp.cos(a2 - a1)
    return mp.atan2(num, den) * 648000 / mp.pi


def test_error_radii_hand_cases():
    """Two equator points 3.6 arcsec apart (theta = dRA exactly).  Eq. (4): 3 sqrt(e1^2 + e2^2)."""
    ra_a, dec_a = np.array([10.0]), np.array([0.0])
    ra_b, dec_b = np.array([10.001]), np.array([0.0])                     # 3.6 arcsec
    for e1, e2, inside in ((1.0, 0.2, False),     # 3 sqrt(1.04) = 3.0594 < 3.6
                           (1.0, 0.7, True),      # 3 sqrt(1.49) = 3.6620 >= 3.6
                           (0.0, 1.2, True),      # 3 * 1.2 = 3.6 + 4e-16: the threshold within an ulp of theta -> in or out, so test 1.2000001
                           (0.0, 1.19, False)):
        e2 = 1.2000001 if (e1, e2) == (0.0, 1.2) else e2
        a, b, s, _ = oracle.match(ra_a, dec_a, None, ra_b, dec_b, None, 100.0, 0, oracle.ENGINE_BRUTE_LD,
                                  err_a=np.array([e1]), err_b=np.array([e2]))
        assert (len(a) == 1) == inside, (e1, e2, len(a))
    # a different factor k, and the radius as a cap on the threshold
    a, *_ = oracle.match(ra_a, dec_a, None, ra_b, dec_b, None, 100.0, 0, 0, err_a=np.array([1.0]), err_b=np.array([0.7]), k_factor=2.0)
    assert len(a) == 0                                                     # 2 sqrt(1.49) = 2.44
    a, *_ = oracle.match(ra_a, dec_a, None, ra_b, dec_b, None, 3.5, 0, 0, err_a=np.array([1.0]), err_b=np.array([0.7]))
    assert len(a) == 0                                                     # threshold 3.66 capped at 3.5 < 3.6


def test_error_radii_against_the_written_out_definition():
    """Random tiny catalogues with random error radii: every pair decided by Eq. (4) with Eq. (1) in 50 digits."""
    import mpmath as mp
    rng = np.random.default_rng(77)
    n = 60
    ra_a = rng.uniform(30.0, 30.004, n); dec_a = rng.uniform(-60.0, -59.996, n)
    ra_b = ra_a + rng.normal(0, 2e-4, n); dec_b = dec_a + rng.normal(0, 2e-4, n)
    ea = rng.uniform(0.05, 0.8, n); eb = rng.uniform(0.05, 0.8, n)
    want = set()
    for i in range(n):
        for j in range(n):
            th = _mp_sep_arcsec(ra_a[i], dec_a[i], ra_b[j], dec_b[j])
            thr = 3 * mp.sqrt(mp.mpf(float(ea[i])) ** 2 + mp.mpf(float(eb[j])) ** 2)
            assert abs(th - thr) > 1e-9                                    # no pair sits on its threshold
            if th <= thr and th <= 50:
                want.add((i, j))
    for eng in (0, 1, 2):
        a, b, s, _ = oracle.match(ra_a, dec_a, None, ra_b, dec_b, None, 50.0, 0, eng, err_a=ea, err_b=eb)
        assert set(zip(a.tolist(), b.tolist())) == want and len(want) > 30


def test_error_radii_constant_reduces_to_a_single_radius():
    """e1 = e2 = e for every record: Eq. (4) is the single radius 3 sqrt(2) e (the pinned plain match)."""
    w = S.config(1, scale=0.05)
    e = 0.21
    a0, b0, s0, _ = oracle.match(w.A.ra, w.A.dec, w.A.id, w.B.ra, w.B.dec, w.B.id, 3.0 * np.sqrt(2.0) * e + 1e-12, 0, 2)
    a1, b1, s1, _ = oracle.match(w.A.ra, w.A.dec, w.A.id, w.B.ra, w.B.dec, w.B.id, 5.0, 0, 2,
                                 err_a=np.full(len(w.A), e), err_b=np.full(len(w.B), e))
    assert np.array_equal(a0, a1) and np.array_equal(b0, b1) and np.array_equal(s0, s1) and len(a0) > 1000


def test_self_match_is_the_upper_triangle():
    """One catalogue with exact duplicates: self_mode 1 = the pairs i < j of the full matrix, 2 = those plus the diagonal,
    3 (nearest) = nearest OTHER source; counts: 2 |upper| + n = |all_pairs(A, A)|."""
    w = S.config(1, scale=0.05)
    ra = np.concatenate([w.A.ra, w.A.ra[:40]]); dec = np.concatenate([w.A.dec, w.A.dec[:40]])      # 40 exact duplicates
    n = len(ra)
    fa, fb, fs, _ = oracle.match(ra, dec, None, ra, dec, None, 20.0, 0, 2)
    ua, ub, us, _ = oracle.match(ra, dec, None, ra, dec, None, 20.0, 0, 2, self_mode=oracle.SELF_PAIRS)
    da, db, ds, _ = oracle.match(ra, dec, None, ra, dec, None, 20.0, 0, 2, self_mode=oracle.SELF_PAIRS_AND_DIAGONAL)
    up = fa < fb
    assert np.array_equal(ua, fa[up]) and np.array_equal(ub, fb[up]) and np.array_equal(us, fs[up])
    assert 2 * len(ua) + n == len(fa) and len(da) == len(ua) + n and (ua < ub).all()
    dup = set(zip(ua[us == 0.0].tolist(), ub[us == 0.0].tolist()))
    assert dup == {(i, len(w.A.ra) + i) for i in range(40)}               # each duplicate pair once, no (i, i)
    # brute force agrees on a slice
    ba, bb, bs, _ = oracle.match(ra[:400], dec[:400], None, ra[:400], dec[:400], None, 20.0, 0, 0, self_mode=1)
    va, vb, vs, _ = oracle.match(ra[:400], dec[:400], None, ra[:400], dec[:400], None, 20.0, 0, 2, self_mode=1)
    assert np.array_equal(ba, va) and np.array_equal(bb, vb)
    # nearest other source = argmin over the off-diagonal of the full matrix
    na, nb_, ns, _ = oracle.match(ra, dec, None, ra, dec, None, 20.0, 1, 2, self_mode=oracle.SELF_EXCLUDE_OWN)
    off = fa != fb
    best = {}
    for i, j, s_ in zip(fa[off].tolist(), fb[off].tolist(), fs[off].tolist()):
        if i not in best or (s_, j) < best[i]:
            best[i] = (s_, j)
    assert len(na) == len(best) and all(best[i][1] == j for i, j in zip(na.tolist(), nb_.tolist())) and (na != nb_).all()
