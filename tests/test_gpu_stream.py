"""Partition streaming (NS (c)) through the C ABI: band-by-band matching from pinned host memory
must give exactly the resident result -- no pair lost or doubled across band edges -- in both modes."""
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


def stream_match(P, A, B, edges, radius, mode, with_ids=True, max_band_out=None, capacity=None):
    import torch
    edges = np.asarray(edges, np.float64)
    Ab, a_off = S.to_bands(A, edges)
    Bb, b_off = S.to_bands(B, edges)
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
    a_cols = (pin(Ab.ra), pin(Ab.dec), pin(Ab.id) if with_ids else None)
    b_cols = (pin(Bb.ra), pin(Bb.dec), pin(Bb.id) if with_ids else None)
    max_a = int(np.diff(a_off).max()); max_b = int(np.diff(b_off).max())
    mbo = max_band_out if max_band_out is not None else max(1024, 2 * max(max_a, max_b))
    cap = capacity if capacity is not None else max(1024, 2 * max(len(A), len(B)))
    opts = P.make_opts(radius)
    arena = torch.empty(P.hlc2_stream_sizes(max_a, max_b, opts, mbo), dtype=torch.uint8, device="cuda")
    oa = torch.empty(cap, dtype=torch.int64).pin_memory(); ob = torch.empty(cap, dtype=torch.int64).pin_memory()
    os_ = torch.empty(cap, dtype=torch.float64).pin_memory()
    n = P.hlc2_stream_crossmatch(a_cols, torch.from_numpy(a_off), b_cols, torch.from_numpy(b_off), torch.from_numpy(edges),
                                 radius, mode, opts, oa, ob, os_, arena, mbo)
    assert n <= cap
    return oa[:n].numpy().copy(), ob[:n].numpy().copy(), os_[:n].numpy().copy(), Ab, Bb, a_off, b_off


@pytest.mark.parametrize("mode", [0, 1])
def test_stream_full_sky_matches_oracle(P, mode):
    w = S.config(2, scale=0.01)                     # 1e5 x 1e5 full sky, r = 2 arcsec
    edges = np.array([-90.0, -60.0, -20.0, -19.9, 0.0, 0.001, 35.0, 89.0, 90.0])      # wide, narrow and polar bands
    ga, gb, gs, *_ = stream_match(P, w.A, w.B, edges, w.radius_arcsec, mode)
    oa, ob, os_, _ = oracle.match(w.A.ra, w.A.dec, w.A.id, w.B.ra, w.B.dec, w.B.id, w.radius_arcsec, mode)
    cmp = parity.compare_nearest if mode == 1 else parity.compare_all_pairs
    rep = cmp((ga, gb, gs), (oa, ob, os_), w.radius_arcsec, parity.make_sep_of(w.A, w.B))
    assert rep["n_gpu"] > 60_000 and len(rep["borderline"]) <= 2


def test_stream_band_edges_lose_nothing(P):
    """Sources planted within r on either side of band edges: every cross-edge pair must be reported once."""
    rng = np.random.default_rng(5)
    edges = np.linspace(-30.0, 30.0, 13)            # 5-degree bands
    n = 40_000
    e = rng.choice(edges[1:-1], n)
    ra = rng.uniform(0.0, 360.0, n)
    r = 3.0
    dec_a = e + rng.uniform(-r, r, n) / 3600.0
    A = S.Catalogue(ra, dec_a, np.arange(n, dtype=np.int64) + 10**12)
    pr, pd = S.perturb(rng, ra, dec_a, 1.0)
    B = S.Catalogue(pr, pd, np.arange(n, dtype=np.int64) * 2 + 1 + 2 * 10**12)
    ga, gb, gs, *_ = stream_match(P, A, B, edges, r, 0)
    oa, ob, os_, _ = oracle.match(A.ra, A.dec, A.id, B.ra, B.dec, B.id, r, 0)
    rep = parity.compare_all_pairs((ga, gb, gs), (oa, ob, os_), r, parity.make_sep_of(A, B))
    assert rep["n_gpu"] > 20_000
    # a good share of the pairs really straddles an edge
    a_band = np.searchsorted(edges, A.dec[np.searchsorted(A.id, ga)], side="right")
    b_pos = {int(i): k for k, i in enumerate(B.id)}
    b_band = np.searchsorted(edges, B.dec[[b_pos[int(i)] for i in gb]], side="right")
    assert (a_band != b_band).sum() > 2_000


def test_stream_row_number_ids_and_small_buffers(P):
    w = S.config(1, scale=0.5)                      # the 2 x 2 degree patch
    edges = np.array([0.0, 0.5, 1.0, 1.5, 2.0])
    ga, gb, gs, Ab, Bb, a_off, b_off = stream_match(P, w.A, w.B, edges, w.radius_arcsec, 0, with_ids=False)
    # ids are global row numbers of the banded arrays
    A2 = S.Catalogue(Ab.ra, Ab.dec, np.arange(len(Ab), dtype=np.int64)); B2 = S.Catalogue(Bb.ra, Bb.dec, np.arange(len(Bb), dtype=np.int64))
    oa, ob, os_, _ = oracle.match(A2.ra, A2.dec, A2.id, B2.ra, B2.dec, B2.id, w.radius_arcsec, 0)
    rep = parity.compare_all_pairs((ga, gb, gs), (oa, ob, os_), w.radius_arcsec, parity.make_sep_of(A2, B2))
    assert rep["n_gpu"] > 30_000
    # too small a per-band slot or total capacity is reported, with the full count
    with pytest.raises(P.Hlc2Error) as ei:
        stream_match(P, w.A, w.B, edges, w.radius_arcsec, 0, max_band_out=100)
    assert ei.value.status == P.HLC2_ERR_BUFFER_TOO_SMALL and ei.value.found == rep["n_gpu"]
    with pytest.raises(P.Hlc2Error) as ei:
        stream_match(P, w.A, w.B, edges, w.radius_arcsec, 0, capacity=1000)
    assert ei.value.status == P.HLC2_ERR_BUFFER_TOO_SMALL and ei.value.found == rep["n_gpu"]


def test_stream_argument_checks(P):
    import ctypes
    L = P.lib()
    cnt = ctypes.c_ulonglong(7)
    assert L.hlc2_stream_crossmatch(*([None] * 9), 0, 1.0, 0, None, None, None, None, 0, ctypes.byref(cnt), None, 0, 0) == P.HLC2_OK
    assert cnt.value == 0
    assert L.hlc2_stream_crossmatch(*([None] * 9), 2, 1.0, 0, None, None, None, None, 0, ctypes.byref(cnt), None, 0, 0) == P.HLC2_ERR_INVALID_ARG
    assert L.hlc2_stream_crossmatch(*([None] * 9), 0, -1.0, 0, None, None, None, None, 0, ctypes.byref(cnt), None, 0, 0) == P.HLC2_ERR_INVALID_ARG


def test_cfg5_streamed_nearest_scaled(P):
    """Config 5 (streamed large, nearest) at a scale the oracle finishes in seconds: 2e5 x 1e5, 1-degree .. 30-degree bands."""
    w = S.config(5, scale=1e-4)
    assert w.modes == ("nearest",)
    edges = np.array([-90.0, -45.0, -30.0, -29.0, -10.0, 0.0, 10.0, 30.0, 60.0, 90.0])
    ga, gb, gs, *_ = stream_match(P, w.A, w.B, edges, w.radius_arcsec, 1)
    oa, ob, os_, _ = oracle.match(w.A.ra, w.A.dec, w.A.id, w.B.ra, w.B.dec, w.B.id, w.radius_arcsec, 1)
    rep = parity.compare_nearest((ga, gb, gs), (oa, ob, os_), w.radius_arcsec, parity.make_sep_of(w.A, w.B))
    assert rep["n_gpu"] > 50_000


def test_bench_streamed_legs_emit_the_contract_line():
    """bench.py --config 5 (at a stated small scale) and --shape D2: one JSON line each with the contract's keys, the PCIe
    roofline, the oracle check of the sampled bands and the fitted cost model."""
    import json
    import os
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    for extra in (["--config", "5", "--scale", "0.002", "--bands", "16"], ["--shape", "D2"]):
        out = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--steps", "1", "--warmup", "1"] + extra,
                             capture_output=True, text=True, timeout=600, cwd=root)
        assert out.returncode == 0, out.stderr[-2000:]
        line = json.loads(out.stdout.strip().splitlines()[-1])
        for key in ("metric", "value", "unit", "n_gpus", "ms_per_step", "config", "e2e", "roofline", "cpu_baseline", "verify", "model", "gpu_launches"):
            assert key in line, key
        assert line["roofline"]["bound"] == "pcie" and 0.0 < line["roofline"]["frac"] < 1.2
        assert line["verify"]["rows_gpu"] == line["verify"]["rows_oracle"] > 1000 and line["gpu_launches"] > 0
        assert line["model"]["eq6_sum_ms"] >= line["model"]["overlapped_max_ms"] > 0.0
