"""The paper's partitioners as a completeness study (Alg. 1, Table 4): pins of
the HEALPix restatement, then the qualitative ordering of Table 4 on boundary-stress data (CPU only)."""
import numpy as np

import hlc2_synth as S
import oracle
from oracle import partition_study as ps


def test_ang2pix_nest_base_faces_and_hierarchy():
    # the twelve base pixels (nside = 1): north cap faces 0-3, equatorial 4-7 centred on RA 0, 90, 180, 270, south 8-11
    assert ps.ang2pix_nest([45.0, 135.0, 225.0, 315.0], [60.0] * 4, 0).tolist() == [0, 1, 2, 3]
    assert ps.ang2pix_nest([0.0, 90.0, 180.0, 270.0], [0.0] * 4, 0).tolist() == [4, 5, 6, 7]
    assert ps.ang2pix_nest([45.0, 135.0, 225.0, 315.0], [-60.0] * 4, 0).tolist() == [8, 9, 10, 11]
    assert ps.ang2pix_nest([10.0], [90.0], 0)[0] in (0, 1, 2, 3) and ps.ang2pix_nest([10.0], [-90.0], 0)[0] in (8, 9, 10, 11)
    # nested scheme: a pixel's parent is its index >> 2, at every level; all indices in range
    rng = np.random.default_rng(3)
    ra, dec = S.uniform_sphere(rng, 200_000)
    prev = ps.ang2pix_nest(ra, dec, 0)
    for k in range(1, 13):
        cur = ps.ang2pix_nest(ra, dec, k)
        assert cur.min() >= 0 and cur.max() < 12 * 4 ** k and np.array_equal(cur >> 2, prev)
        prev = cur


def test_ang2pix_nest_pixels_have_equal_area():
    # HEALPix = equal-area pixels: uniform points fill the 768 pixels of nside = 8 evenly (chi-square), and every pixel is hit
    rng = np.random.default_rng(4)
    ra, dec = S.uniform_sphere(rng, 768 * 500)
    cnt = np.bincount(ps.ang2pix_nest(ra, dec, 3), minlength=768)
    chi2 = ((cnt - 500.0) ** 2 / 500.0).sum()
    assert cnt.min() > 380 and 768 - 5 * np.sqrt(2 * 768) < chi2 < 768 + 5 * np.sqrt(2 * 768)


def test_table4_ordering_on_boundary_stress_data():
    """No Index >= quad-direction >= HEALPix only, the plain partition loses more the finer the pixels, and the
    quad-direction strategy recovers most but not all of it (it probes four directions with an RA offset that ignores
    cos(Dec): the diagonal and polar pairs stay lost) -- the qualitative content of Table 4."""
    w = S.config(4, scale=0.01)                                  # 2e5 x 2e5 stress mix, r = 3 arcsec
    a, b, s, _ = oracle.match(w.A.ra, w.A.dec, None, w.B.ra, w.B.dec, None, w.radius_arcsec, 0, oracle.ENGINE_VOXEL)
    rows = [ps.completeness(w.A.ra, w.A.dec, w.B.ra, w.B.dec, a, b, k, w.radius_arcsec) for k in (6, 9, 12)]
    for r_ in rows:
        assert r_["no_index"] >= r_["quad_direction"] >= r_["healpix_only"] > 0
    assert rows[0]["lost_healpix_only"] < rows[1]["lost_healpix_only"] < rows[2]["lost_healpix_only"]
    assert rows[2]["lost_healpix_only"] > 100 and 0 < rows[2]["lost_quad_direction"] < rows[2]["lost_healpix_only"]
    # on uniform full-sky data (no polar / seam clusters) the replication recovers most of what the plain partition loses
    u = S.config(2, scale=0.02)
    a, b, s, _ = oracle.match(u.A.ra, u.A.dec, None, u.B.ra, u.B.dec, None, u.radius_arcsec, 0, oracle.ENGINE_VOXEL)
    r12 = ps.completeness(u.A.ra, u.A.dec, u.B.ra, u.B.dec, a, b, 12, u.radius_arcsec)
    assert r12["lost_healpix_only"] > 500 and r12["lost_quad_direction"] < 0.2 * r12["lost_healpix_only"]
