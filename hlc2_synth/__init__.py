"""Seeded synthetic catalogue generators for the HLC2 cross-match workloads.

This module only *makes inputs*.  It holds none of the method's arithmetic
(no separations, no cell keys, no matching) and is the one piece of code that
both the CPU oracle (``oracle/``) and the CUDA path
(``paper_2301_07331_b200``) are fed from; it imports neither of them.

What the inputs stand in for
----------------------------
The paper measures on survey extracts that are not in this repository: SDSS,
2MASS and Gaia catalogues of 2e5 .. 4.7e8 records, patches and full sky
(Table 2), plus "simulated" sets pushed toward partition
edges.  The five configurations of ``BASELINE.json`` take
their shapes from those (patch vs full sky, self- vs cross-match, galactic
plane concentration, edge-heavy stress) and are generated here from a seed.
No survey record is reproduced.

Recipe (also stated in DESIGN.md)
---------------------------------
* RNG: ``numpy.random.Generator(Philox(key=[seed, stream]))``; chunk ``j`` of
  catalogue ``c`` uses stream ``(c << 40) | j`` so any chunk can be regenerated
  on its own.  ``seed = 230107331 + config number``.
* Coordinates are fp64 degrees, ``ra in [0, 360)``, ``dec in [-90, 90]``.
* ids: ``idA[i] = 10**12 + 2 i``, ``idB[j] = 2*10**12 + 2 j + 1`` (row numbers
  of the final arrays; > 2**32, disjoint).  B is randomly permuted so a copy is
  never index-aligned with its parent.
* "isotropic Gaussian sigma": per-axis sigma in the tangent plane (east/north),
  re-normalised, converted back to (ra, dec); the catalogue *is* the resulting
  fp64 degree values.
"""
from __future__ import annotations

import os
from concurrent.futures import ThreadPoolExecutor
from dataclasses import dataclass, field

import numpy as np

BASE_SEED = 230107331
CHUNK = 1 << 20
ARCSEC = 1.0 / 3600.0

# J2000 galactic pole / node used to tilt the galactic-plane band onto the
# equatorial sky (standard IAU 1958 system expressed in J2000).
_GP_RA = np.deg2rad(192.85948)
_GP_DEC = np.deg2rad(27.12825)
_L_NCP = np.deg2rad(122.93192)
# probability that a source of the "1 + 9 exp(-(b/10deg)^2)" density belongs
# to the plane component: 9 I / (2 + 9 I), I = sqrt(pi) beta exp(-beta^2/4),
# beta = 10 deg in radians.
_BETA = np.deg2rad(10.0)
_I_PLANE = np.sqrt(np.pi) * _BETA * np.exp(-_BETA * _BETA / 4.0)
P_PLANE = 9.0 * _I_PLANE / (2.0 + 9.0 * _I_PLANE)


@dataclass
class Catalogue:
    ra: np.ndarray   # fp64 degrees
    dec: np.ndarray  # fp64 degrees
    id: np.ndarray   # int64

    def __len__(self) -> int:
        return int(self.ra.shape[0])

    def take(self, rows) -> "Catalogue":
        return Catalogue(self.ra[rows].copy(), self.dec[rows].copy(), self.id[rows].copy())


@dataclass
class Workload:
    name: str
    A: Catalogue
    B: Catalogue
    radius_arcsec: float
    modes: tuple
    # planted truth: B row planted_b[k] is a perturbed copy of A row planted_a[k]
    planted_a: np.ndarray = field(default_factory=lambda: np.zeros(0, np.int64))
    planted_b: np.ndarray = field(default_factory=lambda: np.zeros(0, np.int64))
    sigma_arcsec: float = 0.0
    notes: str = ""


def _rng(seed: int, cat: int, j: int) -> np.random.Generator:
    return np.random.Generator(np.random.Philox(key=[int(seed), (int(cat) << 40) | int(j)]))


def ids_a(n: int) -> np.ndarray:
    return 10**12 + 2 * np.arange(n, dtype=np.int64)


def ids_b(n: int) -> np.ndarray:
    return 2 * 10**12 + 2 * np.arange(n, dtype=np.int64) + 1


# ----------------------------------------------------------------------------
# point samplers (each returns fp64 degrees)
# ----------------------------------------------------------------------------
def uniform_sphere(rng, n):
    ra = 360.0 * rng.random(n)
    dec = np.rad2deg(np.arcsin(rng.uniform(-1.0, 1.0, n)))
    return ra, dec


def uniform_patch(rng, n, ra_lo, ra_hi, dec_lo, dec_hi):
    ra = rng.uniform(ra_lo, ra_hi, n)
    s0, s1 = np.sin(np.deg2rad(dec_lo)), np.sin(np.deg2rad(dec_hi))
    dec = np.rad2deg(np.arcsin(rng.uniform(s0, s1, n)))
    return ra, dec


def _gal_to_equ(l, b):
    """Galactic (l, b) radians -> equatorial (ra, dec) degrees."""
    sb, cb = np.sin(b), np.cos(b)
    dl = _L_NCP - l
    sd = np.sin(_GP_DEC) * sb + np.cos(_GP_DEC) * cb * np.cos(dl)
    dec = np.arcsin(np.clip(sd, -1.0, 1.0))
    yy = cb * np.sin(dl)
    xx = np.cos(_GP_DEC) * sb - np.sin(_GP_DEC) * cb * np.cos(dl)
    ra = np.arctan2(yy, xx) + _GP_RA
    ra = np.mod(np.rad2deg(ra), 360.0)
    ra[ra >= 360.0] = 0.0
    return ra, np.rad2deg(dec)


def galactic_density(rng, n):
    """Density proportional to 1 + 9 exp(-(b/10deg)^2) in galactic latitude b."""
    plane = rng.random(n) < P_PLANE
    n_pl = int(plane.sum())
    l = 2.0 * np.pi * rng.random(n)
    b = np.arcsin(rng.uniform(-1.0, 1.0, n))          # uniform-sphere component
    # plane component: b ~ N(0, (10deg/sqrt2)^2) accepted with probability cos b
    got = np.zeros(0)
    sig = _BETA / np.sqrt(2.0)
    while got.shape[0] < n_pl:
        need = n_pl - got.shape[0]
        cand = rng.normal(0.0, sig, int(need * 1.1) + 16)
        keep = (np.abs(cand) < np.pi / 2) & (rng.random(cand.shape[0]) < np.cos(cand))
        got = np.concatenate([got, cand[keep]])
    b[plane] = got[:n_pl]
    return _gal_to_equ(l, b)


def perturb(rng, ra_deg, dec_deg, sigma_arcsec):
    """Tangent-plane Gaussian offset (per-axis sigma) of each position."""
    n = ra_deg.shape[0]
    a, d = np.deg2rad(ra_deg), np.deg2rad(dec_deg)
    sa, ca, sd, cd = np.sin(a), np.cos(a), np.sin(d), np.cos(d)
    sig = np.deg2rad(sigma_arcsec * ARCSEC)
    xi = rng.normal(0.0, sig, n)    # east
    eta = rng.normal(0.0, sig, n)   # north
    # p + xi * e_east + eta * e_north
    x = cd * ca - xi * sa - eta * sd * ca
    y = cd * sa + xi * ca - eta * sd * sa
    z = sd + eta * cd
    ra = np.mod(np.rad2deg(np.arctan2(y, x)), 360.0)
    ra[ra >= 360.0] = 0.0
    dec = np.rad2deg(np.arctan2(z, np.hypot(x, y)))
    return ra, dec


# ----------------------------------------------------------------------------
# config 4: boundary-stress mixture
# ----------------------------------------------------------------------------
def default_grid(cell_arcsec: float = 160.0) -> dict:
    """A stand-in grid description with the same fields as ``hlc2_grid_describe``
    (equal-height declination zones, per-zone number of RA cells).  Only used
    to place stress sources when no implementation grid is supplied; it is
    input-shaping data, not part of the method."""
    h = cell_arcsec * ARCSEC
    n_z = int(np.floor(180.0 / h))
    h = 180.0 / n_z
    edges = -90.0 + h * np.arange(n_z + 1)
    worst = np.maximum(np.abs(edges[:-1]), np.abs(edges[1:]))
    n_ra = np.maximum(1, np.floor(360.0 * np.cos(np.deg2rad(np.minimum(worst, 90.0))) / h)).astype(np.int64)
    return dict(dec_lo=-90.0, zone_h=h, n_zones=n_z, ra0=0.0, span=360.0, n_ra=n_ra)


def stress_mix(rng, n, grid: dict):
    """40% near cell/zone edges (a quarter of those at corners), 10% polar caps,
    10% RA=0/360 seam, 40% uniform.  Returns ra, dec, cls (0 edge, 1 cap, 2 seam, 3 uniform)."""
    n_edge = int(round(0.4 * n)); n_cap = int(round(0.1 * n)); n_seam = int(round(0.1 * n))
    n_uni = n - n_edge - n_cap - n_seam
    ra_out, dec_out, cls = [], [], []

    # --- edges and corners of the supplied grid
    ra, dec = uniform_sphere(rng, n_edge)
    h, d0, nz = grid["zone_h"], grid["dec_lo"], grid["n_zones"]
    z = np.clip(np.floor((dec - d0) / h).astype(np.int64), 0, nz - 1)
    nra = np.asarray(grid["n_ra"])[z].astype(np.float64)
    cw = grid["span"] / nra
    u = np.mod(ra - grid["ra0"], 360.0)
    k = np.clip(np.floor(u / cw), 0, nra - 1)
    kind = rng.integers(0, 4, n_edge)           # 0: RA edge, 1: zone edge, 2: RA edge, 3: corner
    side_r = rng.integers(0, 2, n_edge); side_z = rng.integers(0, 2, n_edge)
    off_r = rng.uniform(-2.0, 2.0, n_edge) * ARCSEC
    off_z = rng.uniform(-2.0, 2.0, n_edge) * ARCSEC
    cosd = np.maximum(np.cos(np.deg2rad(dec)), 1e-6)
    ra_edge = grid["ra0"] + (k + side_r) * cw + off_r / cosd
    dec_edge = d0 + (z + side_z) * h + off_z
    use_r = (kind == 0) | (kind == 2) | (kind == 3)
    use_z = (kind == 1) | (kind == 3)
    ra = np.where(use_r, ra_edge, ra)
    dec = np.where(use_z, dec_edge, dec)
    dec = np.clip(dec, -90.0, 90.0)
    ra = np.mod(ra, 360.0); ra[ra >= 360.0] = 0.0
    ra_out.append(ra); dec_out.append(dec); cls.append(np.zeros(n_edge, np.int8))

    # --- polar caps |dec| > 89.5, uniform in area, + exact poles + exact duplicates
    ra = 360.0 * rng.random(n_cap)
    c0 = np.cos(np.deg2rad(0.5))
    colat = np.rad2deg(np.arccos(rng.uniform(c0, 1.0, n_cap)))
    sign = np.where(rng.random(n_cap) < 0.5, -1.0, 1.0)
    dec = sign * (90.0 - colat)
    m = min(100, n_cap // 4)
    if m > 0:
        dec[:m] = np.where(np.arange(m) % 2 == 0, 90.0, -90.0)      # exactly at the poles
        ra[m:2 * m] = ra[2 * m:3 * m]; dec[m:2 * m] = dec[2 * m:3 * m]  # exact duplicates
    ra_out.append(ra); dec_out.append(dec); cls.append(np.ones(n_cap, np.int8))

    # --- RA = 0/360 seam: |dRA| cos(dec) <= 5 arcsec
    dec = np.clip(np.rad2deg(np.arcsin(rng.uniform(-1.0, 1.0, n_seam))), -89.5, 89.5)
    dra = rng.uniform(-5.0, 5.0, n_seam) * ARCSEC / np.cos(np.deg2rad(dec))
    ra = np.mod(dra, 360.0); ra[ra >= 360.0] = 0.0
    if n_seam >= 6:
        ra[0] = 0.0; ra[1] = 360.0; ra[2] = np.nextafter(360.0, 0.0)
        ra[3] = -0.0; ra[4] = np.nextafter(0.0, 1.0); ra[5] = 359.99999999999994
    ra_out.append(ra); dec_out.append(dec); cls.append(np.full(n_seam, 2, np.int8))

    ra, dec = uniform_sphere(rng, n_uni)
    ra_out.append(ra); dec_out.append(dec); cls.append(np.full(n_uni, 3, np.int8))

    ra = np.concatenate(ra_out); dec = np.concatenate(dec_out); cls = np.concatenate(cls)
    p = rng.permutation(n)
    return ra[p], dec[p], cls[p]


# ----------------------------------------------------------------------------
# chunked, threaded assembly
# ----------------------------------------------------------------------------
def _threads() -> int:
    return max(1, min(32, (os.cpu_count() or 1)))


def _chunks(n):
    return [(j, min(CHUNK, n - j * CHUNK)) for j in range((n + CHUNK - 1) // CHUNK)]


def _parallel(fn, jobs):
    if len(jobs) <= 1:
        return [fn(*j) for j in jobs]
    with ThreadPoolExecutor(_threads()) as ex:
        return list(ex.map(lambda a: fn(*a), jobs))


def _build(name, seed, n_a, n_copy, n_extra, sampler, sigma, radius, modes, notes=""):
    """A from ``sampler``; B = perturbed copies of a random subset of A (exactly
    n_copy of them, spread over A's chunks) + n_extra independent sources."""
    chunks = _chunks(n_a)
    # copies per A chunk: proportional, exact total
    base = np.array([c[1] for c in chunks], dtype=np.int64)
    quota = np.floor(base * (n_copy / max(n_a, 1))).astype(np.int64)
    short = n_copy - int(quota.sum())
    for t in range(short):
        quota[t % len(quota)] += 1

    def gen_a(j, m):
        rng = _rng(seed, 0, j)
        ra, dec = sampler(rng, m)
        q = int(min(quota[j], m))
        rows = np.sort(rng.permutation(m)[:q])
        cra, cdec = perturb(_rng(seed, 1, j), ra[rows], dec[rows], sigma)
        return ra, dec, rows + j * CHUNK, cra, cdec

    parts = _parallel(gen_a, chunks)
    A = Catalogue(np.concatenate([p[0] for p in parts]), np.concatenate([p[1] for p in parts]), ids_a(n_a))
    parent = np.concatenate([p[2] for p in parts]).astype(np.int64)
    cra = np.concatenate([p[3] for p in parts]); cdec = np.concatenate([p[4] for p in parts])
    del parts

    def gen_x(j, m):
        return sampler(_rng(seed, 2, j), m)

    xs = _parallel(gen_x, _chunks(n_extra)) if n_extra > 0 else []
    bra = np.concatenate([cra] + [x[0] for x in xs]); bdec = np.concatenate([cdec] + [x[1] for x in xs])
    n_b = bra.shape[0]
    perm = _rng(seed, 3, 0).permutation(n_b)            # final row r holds pre-permutation row perm[r]
    bra = bra[perm]; bdec = bdec[perm]
    inv = np.empty(n_b, np.int64); inv[perm] = np.arange(n_b, dtype=np.int64)
    planted_b = inv[: parent.shape[0]]
    B = Catalogue(bra, bdec, ids_b(n_b))
    return Workload(name, A, B, radius, modes, parent, planted_b, sigma, notes)


def config(k: int, scale: float = 1.0, grid: dict | None = None, seed: int | None = None) -> Workload:
    """Build configuration ``k`` (1..5) of BASELINE.json at ``scale`` times its
    source counts (scale = 1 is the full configuration)."""
    seed = BASE_SEED + k if seed is None else seed
    s = lambda n: max(1, int(round(n * scale)))
    if k == 1:
        n_a = s(100_000)
        samp = lambda rng, m: uniform_patch(rng, m, 180.0, 182.0, 0.0, 2.0)
        n_copy = int(_rng(seed, 4, 0).binomial(n_a, 0.8))
        return _build("cfg1_tiny_patch", seed, n_a, n_copy, s(20_000), samp, 0.3, 1.0,
                      ("all_pairs", "nearest"))
    if k == 2:
        return _build("cfg2_full_sky_uniform", seed, s(10_000_000), s(7_000_000), s(3_000_000),
                      uniform_sphere, 0.5, 2.0, ("all_pairs",))
    if k == 3:
        return _build("cfg3_gaia_like", seed, s(100_000_000), s(30_000_000), s(20_000_000),
                      galactic_density, 0.2, 1.0, ("all_pairs",))
    if k == 4:
        g = grid if grid is not None else default_grid()
        samp = lambda rng, m: stress_mix(rng, m, g)[:2]
        w = _build("cfg4_boundary_stress", seed, s(20_000_000), s(16_000_000), s(4_000_000),
                   samp, 0.5, 3.0, ("all_pairs",),
                   notes="stress classes placed relative to the supplied grid description")
        return w
    if k == 5:
        return _build("cfg5_streamed_large", seed, s(2_000_000_000), s(600_000_000), s(400_000_000),
                      galactic_density, 0.2, 1.0, ("nearest",))
    raise ValueError(f"unknown config {k}")


def custom(name, seed, n_a, n_copy, n_extra, sampler, sigma_arcsec, radius_arcsec, modes=("all_pairs",)) -> Workload:
    """A workload of any size with the configurations' recipe: A from ``sampler``; B = ``n_copy`` perturbed copies of
    random A sources + ``n_extra`` independent sources (used for the shapes of the paper's data sets, Table 2)."""
    return _build(name, seed, int(n_a), int(n_copy), int(n_extra), sampler, sigma_arcsec, radius_arcsec, tuple(modes))


def stress_classes(k_seed: int, n: int, grid: dict | None = None):
    """Class labels of config 4's A sources (same streams as ``config(4)``), for
    stratified subsampling.  Only valid for single-chunk sizes; larger callers
    should classify geometrically."""
    g = grid if grid is not None else default_grid()
    out = []
    for j, m in _chunks(n):
        out.append(stress_mix(_rng(k_seed, 0, j), m, g)[2])
    return np.concatenate(out)


def to_bands(cat: "Catalogue", band_edges_deg: np.ndarray):
    """Bucket a catalogue into declination bands (input preparation for the streaming entry point: band k holds
    dec in [edges[k], edges[k+1]), the last band closed above).  Returns (Catalogue in band order, int64 offsets)."""
    edges = np.asarray(band_edges_deg, np.float64)
    nb = len(edges) - 1
    k = np.clip(np.searchsorted(edges, cat.dec, side="right") - 1, 0, nb - 1)
    order = np.argsort(k, kind="stable")
    off = np.zeros(nb + 1, np.int64)
    np.cumsum(np.bincount(k, minlength=nb), out=off[1:])
    return cat.take(order), off
