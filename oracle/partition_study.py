"""The paper's own partitioners as a completeness study -- TEST / ANALYSIS INFRASTRUCTURE, CPU only.

PAPER.md partitions both catalogues by HEALPix nested pixel (L104, L255) and, to recover pairs that straddle a pixel
boundary, replicates every record of one catalogue into the pixels of four offset positions (RA +- R, Dec +- R: the
"quad-direction strategy", Algorithm 1); Table 4 (L326-334) counts what each strategy still loses against the
"No Index" nested loop.  This module restates both partitioners in numpy and counts, for a set of TRUE pairs (the
oracle's), which of them each strategy can see: a partition-based matcher finds a pair exactly when the two records
share a pixel (after replication), so no distance is recomputed here.  It shares nothing with the CUDA path, whose
zone / cell windows are complete by construction (reading 7).

ang2pix_nest follows the published HEALPix construction (Gorski et al. 2005, cited by the paper at L402): twelve base
faces, equatorial belt |z| <= 2/3 and polar caps, pixel = face * nside^2 + bit-interleave(ix, iy).
"""
from __future__ import annotations

import numpy as np


def _interleave(ix, iy, k):
    ix = ix.astype(np.int64); iy = iy.astype(np.int64)
    out = np.zeros_like(ix)
    for b in range(k):
        out |= ((ix >> b) & 1) << (2 * b)
        out |= ((iy >> b) & 1) << (2 * b + 1)
    return out


def ang2pix_nest(ra_deg, dec_deg, level: int):
    """HEALPix nested pixel index at nside = 2**level of positions given in degrees."""
    ra = np.mod(np.asarray(ra_deg, np.float64), 360.0)
    z = np.sin(np.deg2rad(np.asarray(dec_deg, np.float64)))
    za = np.abs(z)
    nside = 1 << level
    tt = np.mod(ra / 90.0, 4.0)                                   # phi in units of pi/2, in [0, 4)
    face = np.zeros(ra.shape, np.int64); ix = np.zeros(ra.shape, np.int64); iy = np.zeros(ra.shape, np.int64)

    eq = za <= 2.0 / 3.0
    t1 = nside * (0.5 + tt[eq]); t2 = nside * z[eq] * 0.75
    jp = np.floor(t1 - t2).astype(np.int64); jm = np.floor(t1 + t2).astype(np.int64)     # ascending / descending edge lines
    ifp = jp >> level; ifm = jm >> level
    f = np.where(ifp == ifm, (ifp & 3) + 4, np.where(ifp < ifm, ifp & 3, (ifm & 3) + 8))
    face[eq] = f; ix[eq] = jm & (nside - 1); iy[eq] = nside - (jp & (nside - 1)) - 1

    po = ~eq
    ntt = np.minimum(3, np.floor(tt[po]).astype(np.int64)); tp = tt[po] - ntt
    tmp = nside * np.sqrt(3.0 * (1.0 - za[po]))
    jp = np.minimum(np.floor(tp * tmp).astype(np.int64), nside - 1)
    jm = np.minimum(np.floor((1.0 - tp) * tmp).astype(np.int64), nside - 1)
    north = z[po] >= 0
    face[po] = np.where(north, ntt, ntt + 8)
    ix[po] = np.where(north, nside - jm - 1, jp); iy[po] = np.where(north, nside - jp - 1, jm)
    return face * (nside * nside) + _interleave(ix, iy, level)


def quad_direction_pixels(ra_deg, dec_deg, level: int, offset_arcsec: float):
    """Algorithm 1 (L126-169), read as in DESIGN.md section 2 (readings 5-7): the record's own pixel and the pixels of
    (RA + R, Dec), (RA - R, Dec), (RA, Dec + R), (RA, Dec - R) -- R added to RA as printed, without 1 / cos(Dec), the
    declinations clipped to the sphere.  Returns an [n, 5] array of pixel indices (duplicates allowed)."""
    ra = np.asarray(ra_deg, np.float64); dec = np.asarray(dec_deg, np.float64)
    R = offset_arcsec / 3600.0
    cols = [ang2pix_nest(ra, dec, level),
            ang2pix_nest(ra + R, dec, level), ang2pix_nest(ra - R, dec, level),
            ang2pix_nest(ra, np.clip(dec + R, -90.0, 90.0), level), ang2pix_nest(ra, np.clip(dec - R, -90.0, 90.0), level)]
    return np.stack(cols, axis=1)


def completeness(ra_a, dec_a, ra_b, dec_b, pair_rows_a, pair_rows_b, level: int, offset_arcsec: float) -> dict:
    """Of the true pairs (row numbers into A and B; the oracle's "No Index" result), how many does each of the paper's
    partition strategies see at this HEALPix level?  (the analogue of Table 4)"""
    pa = ang2pix_nest(ra_a, dec_a, level)
    qb = quad_direction_pixels(ra_b, dec_b, level, offset_arcsec)
    ia = np.asarray(pair_rows_a, np.int64); jb = np.asarray(pair_rows_b, np.int64)
    same = pa[ia] == qb[jb, 0]
    quad = (pa[ia][:, None] == qb[jb]).any(axis=1)
    n = int(ia.shape[0])
    return {"level": level, "nside": 1 << level, "no_index": n, "healpix_only": int(same.sum()), "quad_direction": int(quad.sum()),
            "lost_healpix_only": n - int(same.sum()), "lost_quad_direction": n - int(quad.sum())}
