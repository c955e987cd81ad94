"""paper_2301_07331_b200 -- B200-native HLC2 cross-match hot path.

Thin Python binding over ``libhlc2.so`` (the C ABI of ``include/hlc2.h``): the functions below
have the same names as the C entry points and only marshal arguments.  Every step of the path
(validation, cell keys, radix sort, gather, cell table, match, compaction) runs in the library's
hand-written sm_100a kernels.  PyTorch is used for device memory and streams only.

There is no CPU fallback: if the library has not been built (``python -m
paper_2301_07331_b200.build``) or no CUDA device is present, calls raise.
"""
from __future__ import annotations

import ctypes
import os
from dataclasses import dataclass

HLC2_ALL_PAIRS = 0
HLC2_NEAREST = 1

HLC2_KEY_MASK = (1 << 28) - 1      # low bits of hlc2_index_arrays()["cell_key"]: the cell key; top bits: window flags

HLC2_OK = 0
HLC2_ERR_INVALID_ARG = -1
HLC2_ERR_RADIUS_TOO_LARGE = -2
HLC2_ERR_BUFFER_TOO_SMALL = -3
HLC2_ERR_BAD_COORD = -4
HLC2_ERR_CUDA = -5
HLC2_ERR_GRID_MISMATCH = -6
HLC2_ERR_TOO_MANY = -7
HLC2_ERR_STATIC_LIMIT = -8
HLC2_STATIC_SCRATCH_BYTES = 8 << 20

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libhlc2.so")
_lib = None


class Hlc2Error(RuntimeError):
    def __init__(self, status: int, where: str):
        self.status = status
        msg = lib().hlc2_strerror(status).decode()
        if status == HLC2_ERR_CUDA:
            s = ctypes.c_char_p()
            code = lib().hlc2_last_cuda_error(ctypes.byref(s))
            msg += f" [cuda {code}: {s.value.decode() if s.value else '?'}]"
        super().__init__(f"{where}: {msg} ({status})")


class hlc2_opts(ctypes.Structure):
    _fields_ = [("r_max_arcsec", ctypes.c_double), ("target_occupancy", ctypes.c_double),
                ("cell_arcsec", ctypes.c_double), ("full_sky", ctypes.c_int32), ("zone_aspect", ctypes.c_int32),
                ("grid_like", ctypes.c_void_p), ("d_err_arcsec", ctypes.c_void_p),
                ("async_like", ctypes.c_int32), ("reserved", ctypes.c_int32)]


class hlc2_grid_info(ctypes.Structure):
    _fields_ = [("dec_lo_deg", ctypes.c_double), ("zone_height_deg", ctypes.c_double), ("n_zones", ctypes.c_int64),
                ("ra0_deg", ctypes.c_double), ("ra_span_deg", ctypes.c_double), ("n_cells", ctypes.c_int64),
                ("cell_arcsec", ctypes.c_double), ("n", ctypes.c_int64)]


def lib():
    """Load libhlc2.so; fail loudly if it is missing (no fallback path exists)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(f"{LIB_PATH} not built: run `python -m paper_2301_07331_b200.build` "
                              "(the CUDA library is the only implementation; there is no CPU fallback)")
        L = ctypes.CDLL(LIB_PATH)
        vp, i64, sz = ctypes.c_void_p, ctypes.c_int64, ctypes.c_size_t
        P = ctypes.POINTER
        L.hlc2_index_sizes.argtypes = [i64, P(hlc2_opts), P(sz), P(sz)]
        L.hlc2_build_index.argtypes = [vp, vp, vp, i64, P(hlc2_opts), vp, sz, vp, sz, vp, P(vp)]
        L.hlc2_index_status.argtypes = [vp, P(i64)]
        L.hlc2_grid_describe.argtypes = [vp, P(hlc2_grid_info), P(P(ctypes.c_int32))]
        L.hlc2_index_arrays.argtypes = [vp] + [P(vp)] * 6 + [P(i64), P(i64)]
        L.hlc2_crossmatch_sizes.argtypes = [vp, vp, P(sz)]
        L.hlc2_crossmatch.argtypes = [vp, vp, ctypes.c_double, ctypes.c_int, vp, vp, vp, i64, vp, vp, sz, vp]
        L.hlc2_stream_sizes.argtypes = [i64, i64, P(hlc2_opts), i64, P(sz)]
        L.hlc2_stream_crossmatch.argtypes = [vp] * 8 + [vp, i64, ctypes.c_double, ctypes.c_int, P(hlc2_opts),
                                                        vp, vp, vp, i64, vp, vp, sz, i64]
        L.hlc2_index_destroy.argtypes = [vp]
        L.hlc2_index_destroy.restype = None
        L.hlc2_strerror.argtypes = [ctypes.c_int]
        L.hlc2_strerror.restype = ctypes.c_char_p
        L.hlc2_last_cuda_error.argtypes = [P(ctypes.c_char_p)]
        L.hlc2_kernel_launches.restype = ctypes.c_ulonglong
        L.hlc2_crossmatch_events.argtypes = L.hlc2_crossmatch.argtypes + [vp, vp]
        L.hlc2_selfmatch.argtypes = [vp, ctypes.c_double, ctypes.c_int, ctypes.c_int, vp, vp, vp, i64, vp, vp, sz, vp]
        L.hlc2_crossmatch_radii.argtypes = [vp, vp, ctypes.c_double, ctypes.c_double, ctypes.c_int, vp, vp, vp, i64, vp, vp, sz, vp]
        L.hlc2_crossmatch_static.argtypes = [vp, vp, ctypes.c_double, ctypes.c_int, vp, vp, vp, i64, vp, vp]
        L.hlc2_version.restype = ctypes.c_char_p
        _lib = L
    return _lib


def _torch():
    import torch
    if not torch.cuda.is_available():
        raise RuntimeError("paper_2301_07331_b200 needs a CUDA device (B200, sm_100a); there is no CPU fallback")
    return torch


def _stream_ptr(stream):
    torch = _torch()
    s = torch.cuda.current_stream() if stream is None else stream
    return ctypes.c_void_p(s.cuda_stream)


def make_opts(r_max_arcsec=1.0, target_occupancy=0.0, cell_arcsec=0.0, full_sky=False, grid_like=None, zone_aspect=0,
              async_like=False) -> hlc2_opts:
    o = hlc2_opts()
    o.r_max_arcsec = float(r_max_arcsec); o.target_occupancy = float(target_occupancy)
    o.cell_arcsec = float(cell_arcsec); o.full_sky = int(bool(full_sky)); o.zone_aspect = int(zone_aspect)
    o.grid_like = grid_like.handle if grid_like is not None else None
    o.d_err_arcsec = None
    o.async_like = int(bool(async_like)); o.reserved = 0
    return o


@dataclass
class Index:
    """A built index: the opaque handle plus the torch buffer that owns its device memory."""
    handle: ctypes.c_void_p
    buf: object            # torch.uint8 CUDA tensor (the caller-owned d_index_buf)
    n: int
    opts: hlc2_opts
    _like: object = None   # keeps a grid_like index alive

    def __del__(self):
        try:
            if self.handle:
                lib().hlc2_index_destroy(self.handle)
                self.handle = None
        except Exception:
            pass


def hlc2_index_sizes(n: int, opts: hlc2_opts | None = None):
    ib, tb = ctypes.c_size_t(0), ctypes.c_size_t(0)
    rc = lib().hlc2_index_sizes(int(n), ctypes.byref(opts) if opts is not None else None, ctypes.byref(ib), ctypes.byref(tb))
    if rc != HLC2_OK:
        raise Hlc2Error(rc, "hlc2_index_sizes")
    return ib.value, tb.value


def hlc2_build_index(ra_deg, dec_deg, ids=None, opts: hlc2_opts | None = None, stream=None, temp=None,
                     like: Index | None = None, buf=None, err_arcsec=None) -> Index:
    """ra_deg, dec_deg: CUDA float64 tensors [n]; ids: CUDA int64 tensor [n] or None (row numbers);
    err_arcsec: optional CUDA float64 tensor [n] of per-record error radii (for hlc2_crossmatch_radii)."""
    torch = _torch()
    n = int(ra_deg.shape[0])
    # never write into the caller's options object: it may outlive `like`
    o = hlc2_opts()
    ctypes.memmove(ctypes.byref(o), ctypes.byref(opts if opts is not None else make_opts()), ctypes.sizeof(hlc2_opts))
    opts = o
    if like is not None:
        opts.grid_like = like.handle
    if err_arcsec is not None:
        assert err_arcsec.is_cuda and err_arcsec.dtype == torch.float64 and err_arcsec.is_contiguous() and err_arcsec.shape[0] == n
        opts.d_err_arcsec = err_arcsec.data_ptr()
    assert ra_deg.is_cuda and dec_deg.is_cuda and ra_deg.dtype == torch.float64 and dec_deg.dtype == torch.float64
    assert ra_deg.is_contiguous() and dec_deg.is_contiguous() and dec_deg.shape[0] == n
    if ids is not None:
        assert ids.is_cuda and ids.dtype == torch.int64 and ids.is_contiguous() and ids.shape[0] == n
    ib, tb = hlc2_index_sizes(n, opts)
    if buf is None or buf.numel() < ib:
        buf = torch.empty(ib, dtype=torch.uint8, device=ra_deg.device)
    if temp is None or temp.numel() < tb:
        temp = torch.empty(tb, dtype=torch.uint8, device=ra_deg.device)
    out = ctypes.c_void_p()
    rc = lib().hlc2_build_index(ra_deg.data_ptr(), dec_deg.data_ptr(), ids.data_ptr() if ids is not None else None,
                                n, ctypes.byref(opts), buf.data_ptr(), ib, temp.data_ptr(), temp.numel(),
                                _stream_ptr(stream), ctypes.byref(out))
    if rc != HLC2_OK:
        raise Hlc2Error(rc, "hlc2_build_index")
    # the stream still owns `temp` until the enqueued work drains
    temp.record_stream(torch.cuda.current_stream() if stream is None else stream)
    return Index(out, buf, n, opts, like)


def hlc2_index_status(idx: Index):
    row = ctypes.c_int64(-1)
    rc = lib().hlc2_index_status(idx.handle, ctypes.byref(row))
    if rc not in (HLC2_OK, HLC2_ERR_BAD_COORD, HLC2_ERR_GRID_MISMATCH):
        raise Hlc2Error(rc, "hlc2_index_status")
    return rc, row.value


def hlc2_grid_describe(idx: Index) -> dict:
    import numpy as np
    info = hlc2_grid_info()
    p = ctypes.POINTER(ctypes.c_int32)()
    rc = lib().hlc2_grid_describe(idx.handle, ctypes.byref(info), ctypes.byref(p))
    if rc != HLC2_OK:
        raise Hlc2Error(rc, "hlc2_grid_describe")
    n_ra = np.ctypeslib.as_array(p, shape=(info.n_zones,)).copy()
    return dict(dec_lo=info.dec_lo_deg, zone_h=info.zone_height_deg, n_zones=int(info.n_zones), ra0=info.ra0_deg,
                span=info.ra_span_deg, n_cells=int(info.n_cells), cell_arcsec=info.cell_arcsec, n=int(info.n), n_ra=n_ra)


def hlc2_index_arrays(idx: Index) -> dict:
    """Torch views (no copies) of the index's device arrays."""
    torch = _torch()
    ptrs = [ctypes.c_void_p() for _ in range(6)]
    n, nc = ctypes.c_int64(0), ctypes.c_int64(0)
    rc = lib().hlc2_index_arrays(idx.handle, *[ctypes.byref(p) for p in ptrs], ctypes.byref(n), ctypes.byref(nc))
    if rc != HLC2_OK:
        raise Hlc2Error(rc, "hlc2_index_arrays")
    base = idx.buf.data_ptr()

    def view(p, count, dtype, size):
        off = p.value - base
        return idx.buf[off: off + count * size].view(dtype)

    return dict(x=view(ptrs[0], n.value, torch.float64, 8), y=view(ptrs[1], n.value, torch.float64, 8),
                z=view(ptrs[2], n.value, torch.float64, 8), id=view(ptrs[3], n.value, torch.int64, 8),
                cell_start=view(ptrs[4], nc.value + 1, torch.int32, 4), cell_key=view(ptrs[5], n.value, torch.int32, 4),
                n=n.value, n_cells=nc.value)


def hlc2_crossmatch_sizes(A: Index, B: Index) -> int:
    tb = ctypes.c_size_t(0)
    rc = lib().hlc2_crossmatch_sizes(A.handle, B.handle, ctypes.byref(tb))
    if rc != HLC2_OK:
        raise Hlc2Error(rc, "hlc2_crossmatch_sizes")
    return tb.value


def hlc2_crossmatch(A: Index, B: Index, radius_arcsec: float, mode: int, out_ida, out_idb, out_sep, count,
                    stream=None, temp=None, events=None):
    """Raw call: out_* are CUDA tensors of `capacity` rows, `count` a CUDA tensor of one uint64/int64.
    Asynchronous on `stream`; read `count` after synchronising.  `events` = (start, stop) torch.cuda.Event pair
    (already created, i.e. recorded once) -> hlc2_crossmatch_events records them around the match kernel."""
    cap = int(out_ida.shape[0])
    assert out_idb.shape[0] == cap and out_sep.shape[0] == cap
    need = hlc2_crossmatch_sizes(A, B)
    if need and (temp is None or temp.numel() < need):
        torch = _torch()
        temp = torch.empty(need, dtype=torch.uint8, device=A.buf.device)
        # the stream still owns the scratch until the enqueued work drains
        temp.record_stream(torch.cuda.current_stream() if stream is None else stream)
    args = (A.handle, B.handle, float(radius_arcsec), int(mode), out_ida.data_ptr(), out_idb.data_ptr(),
            out_sep.data_ptr(), cap, count.data_ptr(), temp.data_ptr() if temp is not None else None,
            temp.numel() if temp is not None else 0, _stream_ptr(stream))
    if events is None:
        rc = lib().hlc2_crossmatch(*args)
    else:
        e0, e1 = (ctypes.c_void_p(e.cuda_event) for e in events)
        assert e0.value and e1.value, "record the events once before passing them (torch creates them lazily)"
        rc = lib().hlc2_crossmatch_events(*args, e0, e1)
    if rc != HLC2_OK:
        raise Hlc2Error(rc, "hlc2_crossmatch")


def hlc2_crossmatch_static(A: Index, B: Index, radius_arcsec: float, mode: int, out_ida, out_idb, out_sep, count, stream=None):
    """hlc2_crossmatch with the library's static scratch array (no device allocation anywhere in the call; this wrapper
    makes none either).  Raises Hlc2Error(HLC2_ERR_STATIC_LIMIT) when the match needs more than HLC2_STATIC_SCRATCH_BYTES."""
    cap = int(out_ida.shape[0])
    assert out_idb.shape[0] == cap and out_sep.shape[0] == cap
    rc = lib().hlc2_crossmatch_static(A.handle, B.handle, float(radius_arcsec), int(mode), out_ida.data_ptr(), out_idb.data_ptr(),
                                      out_sep.data_ptr(), cap, count.data_ptr(), _stream_ptr(stream))
    if rc != HLC2_OK:
        raise Hlc2Error(rc, "hlc2_crossmatch_static")


def _run_sized(call, n_hint: int, dev, capacity):
    """Allocate outputs, run `call(oa, ob, os, cnt)`, retry once with the exact size if the first buffer was too small."""
    torch = _torch()
    cap = int(capacity) if capacity is not None else max(1024, int(n_hint))
    for _ in range(2):
        oa = torch.empty(cap, dtype=torch.int64, device=dev); ob = torch.empty(cap, dtype=torch.int64, device=dev)
        os_ = torch.empty(cap, dtype=torch.float64, device=dev); cnt = torch.zeros(1, dtype=torch.int64, device=dev)
        call(oa, ob, os_, cnt, cap)
        found = int(cnt.item())
        if found <= cap:
            return oa[:found], ob[:found], os_[:found]
        cap = found
    raise RuntimeError("result count changed between runs")


def _scratch(A: Index, B: Index):
    torch = _torch()
    need = hlc2_crossmatch_sizes(A, B)
    temp = torch.empty(max(need, 1), dtype=torch.uint8, device=A.buf.device)
    temp.record_stream(torch.cuda.current_stream())
    return temp


def selfmatch(idx: Index, radius_arcsec: float, mode: int = HLC2_ALL_PAIRS, include_self: bool = False, capacity: int | None = None):
    """hlc2_selfmatch: every unordered pair of one catalogue once (all_pairs) or the nearest other source (nearest)."""
    temp = _scratch(idx, idx)

    def call(oa, ob, os_, cnt, cap):
        rc = lib().hlc2_selfmatch(idx.handle, float(radius_arcsec), int(mode), int(bool(include_self)), oa.data_ptr(), ob.data_ptr(),
                                  os_.data_ptr(), cap, cnt.data_ptr(), temp.data_ptr(), temp.numel(), _stream_ptr(None))
        if rc != HLC2_OK:
            raise Hlc2Error(rc, "hlc2_selfmatch")
    return _run_sized(call, idx.n, idx.buf.device, capacity)


def crossmatch_radii(A: Index, B: Index, radius_cap_arcsec: float, k_factor: float = 3.0, mode: int = HLC2_ALL_PAIRS,
                     capacity: int | None = None):
    """hlc2_crossmatch_radii: PAPER.md Eq. (4) per pair, from the error radii the indices were built with."""
    temp = _scratch(A, B)

    def call(oa, ob, os_, cnt, cap):
        rc = lib().hlc2_crossmatch_radii(A.handle, B.handle, float(radius_cap_arcsec), float(k_factor), int(mode), oa.data_ptr(),
                                         ob.data_ptr(), os_.data_ptr(), cap, cnt.data_ptr(), temp.data_ptr(), temp.numel(),
                                         _stream_ptr(None))
        if rc != HLC2_OK:
            raise Hlc2Error(rc, "hlc2_crossmatch_radii")
    return _run_sized(call, A.n, A.buf.device, capacity)


def crossmatch(A: Index, B: Index, radius_arcsec: float, mode: int = HLC2_ALL_PAIRS, capacity: int | None = None):
    """Convenience: allocate outputs, call hlc2_crossmatch, retry once with the exact size if the first
    buffer was too small.  Returns CUDA tensors (idA, idB, sep_arcsec) of exactly the rows found."""
    torch = _torch()
    dev = A.buf.device
    cap = int(capacity) if capacity is not None else max(1024, int(A.n))
    for _ in range(2):
        oa = torch.empty(cap, dtype=torch.int64, device=dev); ob = torch.empty(cap, dtype=torch.int64, device=dev)
        os_ = torch.empty(cap, dtype=torch.float64, device=dev); cnt = torch.zeros(1, dtype=torch.int64, device=dev)
        hlc2_crossmatch(A, B, radius_arcsec, mode, oa, ob, os_, cnt)
        found = int(cnt.item())
        if found <= cap:
            return oa[:found], ob[:found], os_[:found]
        cap = found
    raise RuntimeError("crossmatch: result count changed between runs")



def hlc2_stream_sizes(max_band_a: int, max_band_b: int, opts: hlc2_opts | None, max_band_out: int) -> int:
    ab = ctypes.c_size_t(0)
    rc = lib().hlc2_stream_sizes(int(max_band_a), int(max_band_b), ctypes.byref(opts) if opts is not None else None,
                                 int(max_band_out), ctypes.byref(ab))
    if rc != HLC2_OK:
        raise Hlc2Error(rc, "hlc2_stream_sizes")
    return ab.value


def hlc2_stream_crossmatch(a_cols, a_off, b_cols, b_off, band_edges_deg, radius_arcsec: float, mode: int,
                           opts: hlc2_opts, out_ida, out_idb, out_sep, arena, max_band_out: int) -> int:
    """Raw call.  a_cols / b_cols = (ra, dec, id-or-None) PINNED host tensors already bucketed into declination
    bands; a_off / b_off / band_edges_deg host tensors (int64 / int64 / float64, n_bands + 1 entries); out_* pinned
    host tensors; arena a CUDA uint8 tensor of hlc2_stream_sizes bytes.  Synchronous.  Returns the rows found
    (the first min(found, capacity) of them are in out_*); raises if a buffer was too small."""
    torch = _torch()
    for t in (*a_cols, *b_cols, out_ida, out_idb, out_sep):
        assert t is None or (t.device.type == "cpu" and t.is_pinned() and t.is_contiguous()), "pinned host tensors expected"
    n_bands = int(band_edges_deg.numel()) - 1
    assert a_off.numel() == n_bands + 1 and b_off.numel() == n_bands + 1
    ptr = lambda t: t.data_ptr() if t is not None else None
    cnt = ctypes.c_ulonglong(0)
    rc = lib().hlc2_stream_crossmatch(ptr(a_cols[0]), ptr(a_cols[1]), ptr(a_cols[2]), a_off.data_ptr(),
                                      ptr(b_cols[0]), ptr(b_cols[1]), ptr(b_cols[2]), b_off.data_ptr(),
                                      band_edges_deg.data_ptr(), n_bands, float(radius_arcsec), int(mode),
                                      ctypes.byref(opts), out_ida.data_ptr(), out_idb.data_ptr(), out_sep.data_ptr(),
                                      int(out_ida.shape[0]), ctypes.byref(cnt), arena.data_ptr(), arena.numel(),
                                      int(max_band_out))
    if rc != HLC2_OK:
        e = Hlc2Error(rc, "hlc2_stream_crossmatch"); e.found = cnt.value
        raise e
    return int(cnt.value)

def kernel_launches() -> int:
    return int(lib().hlc2_kernel_launches())


def version() -> str:
    return lib().hlc2_version().decode()
