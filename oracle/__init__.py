"""CPU oracle for the HLC2 cross-match path -- TEST INFRASTRUCTURE ONLY.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  It shares nothing with
``paper_2301_07331_b200`` (no code, headers, tables or helpers) and does not import it.

The arithmetic lives in ``hlc2_oracle.c`` (plain C, long double; see its header for the
passages of PAPER.md it follows).  This file only compiles that C file with gcc and
marshals numpy arrays through ctypes.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
import threading

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "hlc2_oracle.c")
_SO = os.path.join(_HERE, "libhlc2_oracle.so")
_lock = threading.Lock()
_lib = None

ALL_PAIRS, NEAREST = 0, 1
ENGINE_BRUTE_LD, ENGINE_BRUTE, ENGINE_VOXEL = 0, 1, 2


def build(force: bool = False) -> str:
    """Compile the oracle (gcc, -O2, OpenMP).  Building the checker is not using it."""
    with _lock:
        if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
            tmp = _SO + f".tmp{os.getpid()}"
            subprocess.run(["gcc", "-O2", "-std=gnu11", "-fopenmp", "-fPIC", "-shared", "-o", tmp, _SRC, "-lm"],
                           check=True)
            os.replace(tmp, _SO)
    return _SO


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        dp = ctypes.POINTER(ctypes.c_double)
        ip = ctypes.POINTER(ctypes.c_int64)
        lib.hlc2_oracle_sep_arcsec.restype = ctypes.c_double
        lib.hlc2_oracle_sep_arcsec.argtypes = [ctypes.c_double] * 4
        lib.hlc2_oracle_sep_arcsec_hilo.restype = None
        lib.hlc2_oracle_sep_arcsec_hilo.argtypes = [ctypes.c_double] * 4 + [dp, dp]
        lib.hlc2_oracle_match.restype = ctypes.c_int
        lib.hlc2_oracle_match.argtypes = [dp, dp, ip, ctypes.c_int64, dp, dp, ip, ctypes.c_int64,
                                          ctypes.c_double, ctypes.c_int, ctypes.c_int, ctypes.c_int,
                                          ip, ctypes.POINTER(ip), ctypes.POINTER(ip), ctypes.POINTER(dp),
                                          ctypes.POINTER(ctypes.c_int)]
        lib.hlc2_oracle_match_ext.restype = ctypes.c_int
        lib.hlc2_oracle_match_ext.argtypes = [dp, dp, ip, ctypes.c_int64, dp, dp, ip, ctypes.c_int64,
                                              ctypes.c_double, ctypes.c_int, ctypes.c_int, ctypes.c_int,
                                              dp, dp, ctypes.c_double, ctypes.c_int,
                                              ip, ctypes.POINTER(ip), ctypes.POINTER(ip), ctypes.POINTER(dp),
                                              ctypes.POINTER(ctypes.c_int)]
        lib.hlc2_oracle_free.restype = None
        lib.hlc2_oracle_free.argtypes = [ctypes.c_void_p]
        lib.hlc2_oracle_max_threads.restype = ctypes.c_int
        _lib = lib
    return _lib


def max_threads() -> int:
    return int(_load().hlc2_oracle_max_threads())


def sep_arcsec(ra1, dec1, ra2, dec2) -> float:
    """Great-circle separation (Eq. (1), haversine form, long double) in arcsec."""
    return float(_load().hlc2_oracle_sep_arcsec(float(ra1), float(dec1), float(ra2), float(dec2)))


def sep_arcsec_hilo(ra1, dec1, ra2, dec2):
    """The long-double separation as an unevaluated (hi, lo) pair of doubles."""
    hi, lo = ctypes.c_double(), ctypes.c_double()
    _load().hlc2_oracle_sep_arcsec_hilo(float(ra1), float(dec1), float(ra2), float(dec2),
                                        ctypes.byref(hi), ctypes.byref(lo))
    return hi.value, lo.value


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


SELF_NONE, SELF_PAIRS, SELF_PAIRS_AND_DIAGONAL, SELF_EXCLUDE_OWN = 0, 1, 2, 3


def match(ra_a, dec_a, id_a, ra_b, dec_b, id_b, radius_arcsec, mode=ALL_PAIRS, engine=ENGINE_VOXEL,
          threads=0, err_a=None, err_b=None, k_factor=3.0, self_mode=SELF_NONE):
    """Run the oracle.  Returns (idA, idB, sep_arcsec, threads_used), rows sorted by (idA, idB).

    ``id_a`` / ``id_b`` may be None (row numbers).  ``mode`` 0 = all pairs within the radius
    (inclusive), 1 = nearest B per A.  ``engine`` 0 = brute force all in long double,
    1 = brute force with fp64 pre-filter, 2 = voxel hash.

    ``err_a`` / ``err_b`` (both or neither): per-record error radii in arcsec; the criterion becomes PAPER.md
    Eq. (4) per pair, theta <= k_factor * sqrt(e1^2 + e2^2), capped by ``radius_arcsec``.  ``self_mode``: A and B
    are one catalogue (pass the same arrays): 1 = every unordered pair {i, j}, i < j, once; 2 = those and (i, i);
    3 = every ordered pair but j == i (for nearest: a source is not its own neighbour).
    """
    lib = _load()
    ra_a, dec_a, ra_b, dec_b = _f64(ra_a), _f64(dec_a), _f64(ra_b), _f64(dec_b)
    dp = ctypes.POINTER(ctypes.c_double)
    ip = ctypes.POINTER(ctypes.c_int64)

    def ids(a):
        if a is None:
            return None, ip()
        a = np.ascontiguousarray(a, dtype=np.int64)
        return a, a.ctypes.data_as(ip)

    ka, pa = ids(id_a)
    kb, pb = ids(id_b)
    n = ctypes.c_int64(0)
    oa, ob, os_ = ip(), ip(), dp()
    used = ctypes.c_int(0)
    ea = _f64(err_a) if err_a is not None else None
    eb = _f64(err_b) if err_b is not None else None
    rc = lib.hlc2_oracle_match_ext(ra_a.ctypes.data_as(dp), dec_a.ctypes.data_as(dp), pa, ra_a.shape[0],
                                   ra_b.ctypes.data_as(dp), dec_b.ctypes.data_as(dp), pb, ra_b.shape[0],
                                   float(radius_arcsec), int(mode), int(engine), int(threads),
                                   ea.ctypes.data_as(dp) if ea is not None else dp(),
                                   eb.ctypes.data_as(dp) if eb is not None else dp(), float(k_factor), int(self_mode),
                                   ctypes.byref(n), ctypes.byref(oa), ctypes.byref(ob), ctypes.byref(os_),
                                   ctypes.byref(used))
    if rc != 0:
        raise ValueError({-1: "bad coordinate (non-finite or |dec| > 90)", -2: "invalid argument",
                          -3: "out of memory"}.get(rc, f"oracle error {rc}"))
    m = n.value
    try:
        out_a = np.ctypeslib.as_array(oa, shape=(max(m, 1),))[:m].copy()
        out_b = np.ctypeslib.as_array(ob, shape=(max(m, 1),))[:m].copy()
        out_s = np.ctypeslib.as_array(os_, shape=(max(m, 1),))[:m].copy()
    finally:
        lib.hlc2_oracle_free(oa); lib.hlc2_oracle_free(ob); lib.hlc2_oracle_free(os_)
    return out_a, out_b, out_s, used.value
