#!/usr/bin/env python
"""bench.py -- the measurement contract of the HLC2 cross-match hot path.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config C] [--scale S]

A "step" is one pass of the whole hot path over one batch of synthetic input already resident in
HBM: hlc2_build_index(B) + hlc2_build_index(A, on B's grid: opts.grid_like) + hlc2_crossmatch(A, B) (all
SURVEY 8(a) rows except streaming; --grid own gives A a grid of its own).  Workload at N = 1: configuration 3 of BASELINE.json ("Gaia-like density", A = 100M,
B = 50M, r = 1 arcsec, all_pairs) -- the configuration north_star's target is quoted on.

One JSON line is printed (rank 0).  `value` = A sources cross-matched per second over the whole step,
all GPUs together.  north_star allows one GPU only (no sharding, no collectives): with --gpus N > 1
every rank runs an independent replica on its own GPU ("replicas only", weak scaling).

--impl reference times the CPU oracle (oracle/, as it stands) on the host cores over a bounded sample
of the same workload; it is a deliberately slow program, reported as a baseline, not a target.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "A-sources cross-matched/sec"
UNIT = "A-sources/s"
FALLBACK_HBM_GBS = 6650.0       # /opt/skills/guides/B200_PROFILING.md fallback if MEASURED_PEAKS.json is absent


def dist_env():
    return int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))


def peak_hbm():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md)"


def ncu_traffic():
    """DRAM bytes per launch of the match kernel from this round's committed `ncu --set full` capture
    (profiles/match_traffic.txt).  The record names the sha256 of the kernel source it was taken on: a capture of an
    older kernel is reported as stale and its number is NOT used."""
    import hashlib
    p = os.path.join(ROOT, "profiles", "match_traffic.txt")
    try:
        rec = json.load(open(p))
    except Exception:
        return None, "no capture committed"
    src = os.path.join(ROOT, "paper_2301_07331_b200", "csrc", "hlc2_match_same.cu")
    sha = hashlib.sha256(open(src, "rb").read()).hexdigest()
    if rec.get("hlc2_match_same_cu_sha256") != sha:
        return None, f"stale: {p} was captured on another version of hlc2_match_same.cu"
    return rec, rec.get("source", "")


def pcie_rates(gib=1):
    """Pinned host <-> device copy rates, one plain cudaMemcpyAsync of `gib` GiB per direction (best of 3): the roofline
    of every number that includes host copies (e2e, streamed config 5)."""
    import torch
    n = gib << 30
    h = torch.empty(n, dtype=torch.uint8).pin_memory(); d = torch.empty(n, dtype=torch.uint8, device="cuda")
    out = {}
    for name, src, dst in (("h2d_gbs", h, d), ("d2h_gbs", d, h)):
        best = 0.0
        for _ in range(3):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(); dst.copy_(src, non_blocking=True); e1.record(); e1.synchronize()
            best = max(best, n / (e0.elapsed_time(e1) * 1e-3) / 1e9)
        out[name] = best
    out["how"] = f"one cudaMemcpyAsync of {gib} GiB pinned<->device per direction, best of 3, CUDA events"
    return out


class ClockSampler:
    """Samples nvidia-smi clocks / throttle reasons during the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.rows = []; self.proc = None; self.index = index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "50"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True); self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            if len(r) < 7:
                continue
            try:
                sm.append(float(r[0])); mx.append(float(r[1]))
            except ValueError:
                continue
            for nme, v in zip(names, r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nme)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


def sample_patch(w, ra_lo=0.0, ra_hi=3.6):
    """Bounded sample of a workload for the CPU legs: both catalogues restricted to an RA slice
    (same sky density, so per-source work is representative; edge effects ~ r / slice width)."""
    import hlc2_synth as S
    ma = (w.A.ra >= ra_lo) & (w.A.ra < ra_hi); mb = (w.B.ra >= ra_lo) & (w.B.ra < ra_hi)
    return S.Catalogue(w.A.ra[ma], w.A.dec[ma], w.A.id[ma]), S.Catalogue(w.B.ra[mb], w.B.dec[mb], w.B.id[mb])


def time_oracle(A, B, radius, mode, keep=False, threads=0):
    import oracle
    t = time.perf_counter()
    a, b, s, used = oracle.match(A.ra, A.dec, A.id, B.ra, B.dec, B.id, radius, mode, threads=threads)
    dt = time.perf_counter() - t
    return (dt, len(a), used, (a, b, s)) if keep else (dt, len(a), used)


def run_reference(args, w, mode):
    """--impl reference: the oracle, as it stands, on the host cores; each step = the bounded sample."""
    rank, _, world = dist_env()
    if rank != 0:
        return
    # size the sample so that the whole --steps/--warmup run takes about two minutes on this box's cores
    # and is the WHOLE workload whenever that fits (config 3: ~45 s per pass on 16 cores -> up to 3 passes)
    pa, pb = sample_patch(w, 0.0, 3.6)
    dt_probe, _, _ = time_oracle(pa, pb, w.radius_arcsec, mode)
    budget = 150.0 / max(1, args.steps + args.warmup)
    args.sample_ra_deg = float(min(360.0, max(1.0, 3.6 * budget / max(dt_probe, 1e-3))))
    whole = args.sample_ra_deg >= 360.0
    A, B = (w.A, w.B) if whole else sample_patch(w, 0.0, args.sample_ra_deg)
    for _ in range(args.warmup):
        time_oracle(A, B, w.radius_arcsec, mode)
    t_tot, used = 0.0, 0
    for _ in range(args.steps):
        dt, npairs, used = time_oracle(A, B, w.radius_arcsec, mode)
        t_tot += dt
    val = len(A) * args.steps / t_tot
    sample = (f"the whole workload: {len(A)} x {len(B)} sources, {npairs} rows" if whole else
              f"both catalogues restricted to RA in [0,{args.sample_ra_deg:.2f}) deg: {len(A)} x {len(B)} sources, {npairs} rows")
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * t_tot / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f80 (x87 long double)", "data": "synthetic",
            "config": {"workload": w.name, "n_a": len(w.A), "n_b": len(w.B), "radius_arcsec": w.radius_arcsec,
                       "mode": "nearest" if mode else "all_pairs", "sample": sample},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": used, "kind": "oracle", "sample": sample},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def host_register(arr):
    """Pin a numpy array in place (cudaHostRegister): no second copy of a multi-GB catalogue."""
    import torch
    rt = torch.cuda.cudart()
    err = rt.cudaHostRegister(arr.ctypes.data, arr.nbytes, 0)
    assert int(err) == 0, f"cudaHostRegister failed: {err}"
    return torch.from_numpy(arr)


def transfer_model(gib=1):
    """alpha and beta of PAPER.md Eq. (5), T(d) = alpha + beta d, measured as the paper prescribes (L204-208): alpha = the
    time of a one-byte transfer, beta = (t_s - alpha) / s for one large transfer (here 1 GiB), pinned memory, per direction."""
    import torch
    big = gib << 30
    h1 = torch.empty(1, dtype=torch.uint8).pin_memory(); d1 = torch.empty(1, dtype=torch.uint8, device="cuda")
    hb = torch.empty(big, dtype=torch.uint8).pin_memory(); db = torch.empty(big, dtype=torch.uint8, device="cuda")
    ev = lambda: torch.cuda.Event(enable_timing=True)
    out = {}
    for name, (s1, t1, sb, tb) in {"h2d": (h1, d1, hb, db), "d2h": (d1, h1, db, hb)}.items():
        for _ in range(20): t1.copy_(s1, non_blocking=True)
        torch.cuda.synchronize()
        e0, e1 = ev(), ev(); e0.record()
        for _ in range(200): t1.copy_(s1, non_blocking=True)
        e1.record(); e1.synchronize()
        alpha = e0.elapsed_time(e1) * 1e-3 / 200
        best = 1e9
        for _ in range(3):
            e0, e1 = ev(), ev(); e0.record(); tb.copy_(sb, non_blocking=True); e1.record(); e1.synchronize()
            best = min(best, e0.elapsed_time(e1) * 1e-3)
        out[name] = {"alpha_s": alpha, "beta_s_per_byte": (best - alpha) / big, "gbs": big / best / 1e9}
    return out


def run_streamed(args, w, label, mode, nb, clocks_index=0, extra=None, paper=None):
    """One step = one call of hlc2_stream_crossmatch over all declination bands from pinned host memory (H2D of the next
    bands, index build + match of the current one and D2H of the previous one's rows overlap on three streams): the
    catalogues never sit in HBM as a whole.  Bound by the PCIe link, so the roofline is the measured pinned copy rate.
    Also fits the paper's cost model (Eq. (5)-(6), L204-214) on this machine and compares its prediction."""
    import gc
    import torch
    import hlc2_synth as S
    import paper_2301_07331_b200 as P
    import oracle
    from tests import parity
    n_a, n_b, r = len(w.A), len(w.B), w.radius_arcsec
    lo_d, hi_d = float(w.A.dec.min()), float(w.A.dec.max())
    edges = np.quantile(w.A.dec[:: max(1, n_a // 2_000_000)], np.linspace(0.0, 1.0, nb + 1))
    edges[0], edges[-1] = -90.0, 90.0
    edges = np.maximum.accumulate(edges)
    for k in range(1, nb + 1):                              # bands at least 2 r high (a narrow strip: fewer, equal bands)
        if edges[k] - edges[k - 1] < 2.0 * r / 3600.0:
            edges = np.concatenate([[-90.0], np.linspace(lo_d, hi_d, nb + 1)[1:-1], [90.0]]); break
    t0 = time.perf_counter()
    def bands_of(cat):         # band order without the id columns (ids are implicit: the global row numbers of the banded arrays)
        k = np.clip(np.searchsorted(edges, cat.dec, side="right") - 1, 0, nb - 1).astype(np.int16)
        off = np.zeros(nb + 1, np.int64); np.cumsum(np.bincount(k, minlength=nb), out=off[1:])
        order = np.argsort(k, kind="stable"); del k
        ra = cat.ra[order]; dec = cat.dec[order]
        return ra, dec, off
    w.planted_a = None; w.planted_b = None                 # multi-GB bookkeeping of the generator, not needed here
    a_ra, a_dec, a_off = bands_of(w.A); w.A = None          # free each original as soon as its banded copy exists
    b_ra, b_dec, b_off = bands_of(w.B); w.B = None
    del w; gc.collect()
    t_band = time.perf_counter() - t0
    sA = [host_register(a_ra), host_register(a_dec), None]; sB = [host_register(b_ra), host_register(b_dec), None]
    max_a, max_b = int(np.diff(a_off).max()), int(np.diff(b_off).max())
    cap = int(0.45 * n_a) + 1024 if mode == 1 else int(1.1 * min(n_a, n_b)) + 1_000_000
    mbo = max(max_a, max_b)
    opts = P.make_opts(r, target_occupancy=args.occupancy)
    arena = torch.empty(P.hlc2_stream_sizes(max_a, max_b, opts, mbo), dtype=torch.uint8, device="cuda")
    h_out = [torch.empty(cap, dtype=torch.int64).pin_memory(), torch.empty(cap, dtype=torch.int64).pin_memory(),
             torch.empty(cap, dtype=torch.float64).pin_memory()]
    t_off = [torch.from_numpy(a_off), torch.from_numpy(b_off), torch.from_numpy(np.ascontiguousarray(edges))]
    def step():
        return P.hlc2_stream_crossmatch(sA, t_off[0], sB, t_off[1], t_off[2], r, mode, opts, h_out[0], h_out[1], h_out[2], arena, mbo)
    ev = lambda: torch.cuda.Event(enable_timing=True)
    for _ in range(max(1, min(args.warmup, 2))):
        found = step()
    clocks = ClockSampler(clocks_index); clocks.start()
    n0 = P.kernel_launches()
    torch.cuda.synchronize()
    t_wall = time.perf_counter()
    e0, e1 = ev(), ev(); e0.record()
    for _ in range(args.steps):
        found = step()
    e1.record(); torch.cuda.synchronize()
    t_wall = (time.perf_counter() - t_wall) / args.steps
    launches = P.kernel_launches() - n0
    clk = clocks.stop()
    t_ms = e0.elapsed_time(e1) / args.steps
    h2d, d2h = 16 * (n_a + n_b), 24 * found
    # ---- parity on a stated sample of bands: every 16th, both end bands, and the bands next to them
    ga = h_out[0][:found].numpy(); gb_ = h_out[1][:found].numpy(); gs = h_out[2][:found].numpy()
    sample = sorted(set(list(range(0, nb, 16)) + [0, 1, nb - 2, nb - 1]) & set(range(nb)))
    ver = {"bands_checked": sample, "rows_gpu": 0, "rows_oracle": 0, "borderline": 0, "swaps": 0, "max_sep_err": 0.0}
    t_or = 0.0; used = 0
    cmp = parity.compare_nearest if mode == 1 else parity.compare_all_pairs
    for k in sample:
        a0, a1 = int(a_off[k]), int(a_off[k + 1]); lo, hi = max(k - 1, 0), min(k + 1, nb - 1)
        b0, b1 = int(b_off[lo]), int(b_off[hi + 1])
        if a1 == a0: continue
        A = S.Catalogue(a_ra[a0:a1], a_dec[a0:a1], np.arange(a0, a1, dtype=np.int64)); B = S.Catalogue(b_ra[b0:b1], b_dec[b0:b1], np.arange(b0, b1, dtype=np.int64))
        t1 = time.perf_counter()
        oa, ob, os_, used = oracle.match(A.ra, A.dec, A.id, B.ra, B.dec, B.id, r, mode)
        t_or += time.perf_counter() - t1
        m = (ga >= a0) & (ga < a1)
        rep = cmp((ga[m], gb_[m], gs[m]), (oa, ob, os_), r, parity.make_sep_of(A, B))     # raises on any lost / invented pair
        ver["rows_gpu"] += int(m.sum()); ver["rows_oracle"] += len(oa)
        ver["borderline"] += len(rep["borderline"]); ver["swaps"] += len(rep.get("swaps", []))
        ver["max_sep_err"] = max(ver["max_sep_err"], float(rep["max_sep_err"]))
    a_checked = int(sum(a_off[k + 1] - a_off[k] for k in sample))
    # ---- the paper's cost model on this machine (Eq. (5)-(6)): transfer alpha / beta, device term sigma + c n fitted on
    # resident runs of 1, 2 and 4 merged bands from the middle of the sky
    tm = transfer_model()
    pts = []
    mid = nb // 2
    for g in (1, 2, 4):
        k0, k1 = max(0, mid - g // 2), min(nb, max(0, mid - g // 2) + g)
        a0, a1, b0, b1 = int(a_off[k0]), int(a_off[k1]), int(b_off[k0]), int(b_off[k1])
        if a1 - a0 < 1000 or b1 - b0 < 1000: continue
        da = [torch.from_numpy(a_ra[a0:a1]).cuda(), torch.from_numpy(a_dec[a0:a1]).cuda()]
        db = [torch.from_numpy(b_ra[b0:b1]).cuda(), torch.from_numpy(b_dec[b0:b1]).cuda()]
        oc = torch.empty(a1 - a0 + b1 - b0, dtype=torch.int64, device="cuda"); od = torch.empty_like(oc); os2 = torch.empty(oc.shape[0], dtype=torch.float64, device="cuda")
        cnt = torch.zeros(1, dtype=torch.int64, device="cuda")
        ts = []
        for rep_ in range(4):
            f0, f1 = ev(), ev(); f0.record()
            ib = P.hlc2_build_index(db[0], db[1], None, opts=opts); ia = P.hlc2_build_index(da[0], da[1], None, opts=opts, like=ib)
            P.hlc2_crossmatch(ia, ib, r, mode, oc, od, os2, cnt)
            f1.record(); f1.synchronize()
            if rep_: ts.append(f0.elapsed_time(f1) * 1e-3)
        pts.append((a1 - a0 + b1 - b0, float(np.median(ts))))
        del da, db, oc, od, os2
    model = {"transfer": tm}
    if len(pts) >= 2:
        xs, ys = np.array([p_[0] for p_ in pts], float), np.array([p_[1] for p_ in pts], float)
        c_dev, sigma = np.polyfit(xs, ys, 1)
        na_k, nb_k = np.diff(a_off).astype(float), np.diff(b_off).astype(float)
        win_k = nb_k.copy()          # (the window also holds a thin halo of its neighbours: negligible for the model)
        t_in = tm["h2d"]["alpha_s"] * 2 * nb + tm["h2d"]["beta_s_per_byte"] * 16.0 * (na_k + nb_k).sum()
        t_dev = float((sigma + c_dev * (na_k + win_k)).sum())
        t_out = tm["d2h"]["alpha_s"] * 3 * nb + tm["d2h"]["beta_s_per_byte"] * 24.0 * found
        model.update({"device_fit": {"points_n_seconds": pts, "sigma_s": float(sigma), "seconds_per_source": float(c_dev)},
                      "eq6_sum_ms": 1e3 * (t_in + t_dev + t_out), "overlapped_max_ms": 1e3 * max(t_in, t_dev, t_out),
                      "terms_ms": {"transfer_in": 1e3 * t_in, "device": 1e3 * t_dev, "transfer_out": 1e3 * t_out},
                      "measured_ms": t_ms,
                      "note": "Eq. (6) adds the terms of every round (the paper's upper limit, no overlap); with the three streams overlapped the step should take about the largest term"})
    t_pcie = max(tm["h2d"]["beta_s_per_byte"] * h2d, tm["d2h"]["beta_s_per_byte"] * d2h)
    cfg = {"workload": label, "n_a": n_a, "n_b": n_b, "radius_arcsec": r, "mode": "nearest" if mode else "all_pairs",
           "rows_found": int(found), "bands": nb, "max_band_a": max_a, "max_band_b": max_b, "arena_bytes": int(arena.numel()),
           "ids": "implicit (global row numbers of the banded arrays)", "band_seconds": t_band}
    cfg.update(extra or {})
    line = {"metric": METRIC, "value": n_a / (t_ms * 1e-3), "unit": UNIT, "n_gpus": 1, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": t_ms, "wall_s_per_step": t_wall, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": cfg,
            "e2e": {"value": n_a / (t_ms * 1e-3), "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                    "path": "pinned host bands -> hlc2_stream_crossmatch (H2D, build, match, D2H overlapped on 3 streams)"},
            "roofline": {"bound": "pcie", "achieved": h2d / (t_ms * 1e-3) / 1e9, "peak": tm["h2d"]["gbs"], "unit": "GB/s",
                         "frac": (h2d / (t_ms * 1e-3) / 1e9) / tm["h2d"]["gbs"], "traffic": None, "ms_at_peak": 1e3 * t_pcie},
            "cpu_baseline": {"value": a_checked / t_or if t_or else None, "unit": UNIT, "cores": used, "kind": "oracle",
                             "sample": f"the {len(sample)} checked bands: {a_checked} A sources against their three-band B windows"},
            "verify": ver, "model": model, "paper_context": paper, "gpu_launches": int(launches), "clocks": clk}
    print(json.dumps(line), flush=True)
    return 0


def run_config5(args, clocks_index=0):
    """Configuration 5 ("Streamed large", nearest).  At scale 1 the pinned inputs are 48 GB (ids implicit) and generation
    takes minutes on the box's 16 cores; --scale states the fraction actually run."""
    import hlc2_synth as S
    t0 = time.perf_counter()
    w = S.config(5, scale=args.scale)
    t_gen = time.perf_counter() - t0
    return run_streamed(args, w, "cfg5_streamed_large", 1, args.bands, clocks_index,
                        extra={"scale": args.scale, "gen_seconds": t_gen, "note": "scale 1 = 2e9 x 1e9; the fraction run is stated here"})


def run_shape(args, clocks_index=0):
    """End to end from host arrays at the shapes of the paper's data sets (Table 2), beside its own times
    (Table 5: P100 / V100, file I/O included, radius not stated) -- context, not a target.  Synthetic stand-ins:
    D2 = two 1 105 627-source catalogues in the strip RA [340, 360], Dec [1, 1.2]; D4 = 61 734 000 sources of a
    galactic-plane-concentrated full sky matched with themselves; D6 = 467 555 800 x 102 890 000 sources of the same sky."""
    import torch
    import hlc2_synth as S
    import paper_2301_07331_b200 as P
    import oracle
    from tests import parity
    shape = args.shape
    t0 = time.perf_counter()
    if shape == "D2":
        n = 1_105_627
        samp = lambda rng, m: S.uniform_patch(rng, m, 340.0, 360.0, 1.0, 1.2)
        w = S.custom("shape_D2_1105627x1105627_strip", S.BASE_SEED + 12, n, int(0.7 * n), n - int(0.7 * n), samp, 0.3, 1.0, ("all_pairs",))
        return run_streamed(args, w, w.name, 0, 4, clocks_index, extra={"gen_seconds": time.perf_counter() - t0},
                            paper={"table5": "HLC2 5 s (1105627 x 1105627), P100 / V100, files included", "line": "P:L368"})
    if shape == "D6":
        na, nb_ = 467_555_800, 102_890_000
        w = S.custom("shape_D6_467555800x102890000_fullsky", S.BASE_SEED + 16, na, int(0.6 * nb_), nb_ - int(0.6 * nb_), S.galactic_density, 0.2, 1.0, ("all_pairs",))
        return run_streamed(args, w, w.name, 0, 128, clocks_index, extra={"gen_seconds": time.perf_counter() - t0},
                            paper={"table5": "HLC2 260 s (467555800 x 102890000), P100 / V100, files included", "line": "P:L368"})
    assert shape == "D4"
    n, r = 61_734_000, 1.0
    w = S.custom("shape_D4_61734000_self", S.BASE_SEED + 14, n, 0, 1, S.galactic_density, 0.2, r, ("all_pairs",))
    t_gen = time.perf_counter() - t0
    h = [torch.from_numpy(w.A.ra).pin_memory(), torch.from_numpy(w.A.dec).pin_memory()]
    opts = P.make_opts(r)
    ib, tb = P.hlc2_index_sizes(n, opts)
    buf = torch.empty(ib, dtype=torch.uint8, device="cuda"); temp = torch.empty(tb, dtype=torch.uint8, device="cuda")
    cap = n // 8 + 1024
    oa = torch.empty(cap, dtype=torch.int64, device="cuda"); ob = torch.empty_like(oa); os_ = torch.empty(cap, dtype=torch.float64, device="cuda")
    cnt = torch.zeros(1, dtype=torch.int64, device="cuda")
    ho = [torch.empty(cap, dtype=torch.int64).pin_memory(), torch.empty(cap, dtype=torch.int64).pin_memory(), torch.empty(cap, dtype=torch.float64).pin_memory()]
    idx = P.hlc2_build_index(h[0].cuda(), h[1].cuda(), None, opts=opts, temp=temp, buf=buf)
    mtemp = torch.empty(max(1, P.hlc2_crossmatch_sizes(idx, idx)), dtype=torch.uint8, device="cuda")
    ev = lambda: torch.cuda.Event(enable_timing=True)
    def step(marks=None):
        d = [t.cuda(non_blocking=True) for t in h]
        if marks: marks[0].record()
        ix = P.hlc2_build_index(d[0], d[1], None, opts=opts, temp=temp, buf=buf)
        if marks: marks[1].record()
        rc = P.lib().hlc2_selfmatch(ix.handle, r, 0, 0, oa.data_ptr(), ob.data_ptr(), os_.data_ptr(), cap, cnt.data_ptr(), mtemp.data_ptr(), mtemp.numel(), None)
        assert rc == 0
        if marks: marks[2].record()
        nf = int(cnt.item())
        for src, dst in zip((oa, ob, os_), ho): dst[:nf].copy_(src[:nf], non_blocking=True)
        return nf
    for _ in range(3): nf = step()
    torch.cuda.synchronize()
    marks = [ev(), ev(), ev()]
    e0, e1 = ev(), ev(); e0.record()
    for k in range(args.steps): nf = step(marks if k == args.steps - 1 else None)
    e1.record(); torch.cuda.synchronize()
    t_ms = e0.elapsed_time(e1) / args.steps
    # parity on a 6-degree RA slice: the slice's pairs from the oracle's self-match against the GPU rows of those sources
    m = (w.A.ra >= 100.0) & (w.A.ra < 106.0); rows = np.flatnonzero(m)
    A = S.Catalogue(w.A.ra[rows], w.A.dec[rows], rows.astype(np.int64))
    o_a, o_b, o_s, used = oracle.match(A.ra, A.dec, A.id, A.ra, A.dec, A.id, r, 0, self_mode=oracle.SELF_PAIRS)
    ga, gb_, gs = ho[0][:nf].numpy(), ho[1][:nf].numpy(), ho[2][:nf].numpy()
    inside = m[ga] & m[gb_]
    lo = lambda x, y: (np.minimum(x, y), np.maximum(x, y))
    g = lo(ga[inside], gb_[inside]); o = lo(o_a, o_b)
    rep = parity.compare_all_pairs((g[0], g[1], gs[inside]), (o[0], o[1], o_s), r, parity.make_sep_of(A, A))
    line = {"metric": METRIC, "value": n / (t_ms * 1e-3), "unit": UNIT, "n_gpus": 1, "steps": args.steps, "warmup": 3, "ms_per_step": t_ms,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": w.name, "n_a": n, "n_b": n, "radius_arcsec": r, "mode": "self-match, every unordered pair once", "rows_found": int(nf),
                       "gen_seconds": t_gen, "path": "pinned host -> H2D -> hlc2_build_index -> hlc2_selfmatch -> D2H of count and rows"},
            "phases_ms": {"build_index": marks[0].elapsed_time(marks[1]), "selfmatch": marks[1].elapsed_time(marks[2])},
            "e2e": {"value": n / (t_ms * 1e-3), "unit": UNIT, "h2d_bytes_per_step": 16 * n, "d2h_bytes_per_step": 24 * nf + 8},
            "verify": {"against": "oracle self-match on the RA slice [100, 106) deg", "n_gpu": rep["n_gpu"], "n_oracle": rep["n_oracle"],
                       "borderline": len(rep["borderline"]), "max_sep_err": float(rep["max_sep_err"])},
            "paper_context": {"table5": "HLC2 150 s (61734000 x 61734000), P100 / V100, files included", "line": "P:L368"}}
    print(json.dumps(line), flush=True)
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=3)
    ap.add_argument("--scale", type=float, default=1.0, help="scale the source counts (1.0 = the named configuration)")
    ap.add_argument("--sample-ra-deg", type=float, default=360.0, help="RA slice of the CPU-baseline sample (360 = the whole workload)")
    ap.add_argument("--grid", default="shared", choices=["shared", "own"], help="shared: A is filed on B's grid (opts.grid_like); own: each index plans its own grid")
    ap.add_argument("--no-verify", action="store_true", help="do not compare the CUDA rows with the oracle's (needs the cpu_baseline leg on the whole workload)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--occupancy", type=float, default=0.0)
    ap.add_argument("--occupancy-b", type=float, default=None, help="target occupancy of B's index (default: same as --occupancy)")
    ap.add_argument("--bands", type=int, default=0, help="declination bands of the streamed legs (0: 32 for the e2e leg of a resident configuration -- measured best of 16 / 32 / 64 on config 3 -- and 64 for --config 5)")
    ap.add_argument("--no-stream", action="store_true", help="skip the streamed e2e leg")
    ap.add_argument("--shape", default=None, choices=["D2", "D4", "D6"], help="end to end at the shape of one of the paper's data sets (Table 2) instead of a configuration")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    rank, local_rank, world = dist_env()

    import hlc2_synth as S
    if args.impl == "reference" and rank != 0:
        return 0
    if (args.config == 5 or args.shape) and args.impl == "ours":
        import torch
        from paper_2301_07331_b200 import build as hb
        hb.build()
        torch.cuda.set_device(local_rank)
        if args.shape:
            return run_shape(args, local_rank)
        if args.bands <= 0: args.bands = 64
        return run_config5(args, local_rank)
    t0 = time.perf_counter()
    # replicas: every rank generates its own catalogue (different seed) of the same shape
    w = S.config(args.config, scale=args.scale, seed=S.BASE_SEED + args.config + 1000 * rank)
    t_gen = time.perf_counter() - t0
    mode = 1 if w.modes == ("nearest",) else 0
    if args.impl == "reference":
        run_reference(args, w, mode)
        return 0

    import torch
    import paper_2301_07331_b200 as P
    from paper_2301_07331_b200 import build as hb
    hb.build()
    assert torch.cuda.is_available(), "bench.py needs a CUDA device; there is no CPU fallback"
    torch.cuda.set_device(local_rank)
    use_dist = world > 1
    if use_dist:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))

    n_a, n_b, r = len(w.A), len(w.B), w.radius_arcsec
    # pinned host copies (the e2e leg copies from these inside its timed region)
    pin = lambda a: torch.from_numpy(a).pin_memory()
    hA = [pin(w.A.ra), pin(w.A.dec), pin(w.A.id)]; hB = [pin(w.B.ra), pin(w.B.dec), pin(w.B.id)]
    dA = [t.cuda(non_blocking=True) for t in hA]; dB = [t.cuda(non_blocking=True) for t in hB]
    torch.cuda.synchronize()

    # shared grid: A is filed on B's grid, which needs no extent pass and no host synchronisation (opts.async_like)
    opts_a = P.make_opts(r, target_occupancy=args.occupancy, async_like=args.grid == "shared"); opts_b = P.make_opts(r, target_occupancy=args.occupancy if args.occupancy_b is None else args.occupancy_b)
    ib_b, tb_b = P.hlc2_index_sizes(n_b, opts_b)
    buf_b = torch.empty(ib_b, dtype=torch.uint8, device="cuda")
    temp = torch.empty(tb_b, dtype=torch.uint8, device="cuda")
    if args.grid == "shared":             # A's buffers are sized for B's grid: build B once to learn it
        ib0 = P.hlc2_build_index(dB[0], dB[1], dB[2], opts=opts_b, temp=temp, buf=buf_b)
        ib_a, tb_a = P.hlc2_index_sizes(n_a, P.make_opts(r, target_occupancy=args.occupancy, grid_like=ib0))
        del ib0
    else:
        ib_a, tb_a = P.hlc2_index_sizes(n_a, opts_a)
    buf_a = torch.empty(ib_a, dtype=torch.uint8, device="cuda")
    if tb_a > tb_b:
        temp = torch.empty(tb_a, dtype=torch.uint8, device="cuda")
    # output rows: config 3 finds 0.3 per A source; the others up to 2.2 per source (config 4's dense strips and caps)
    cap = (int(max(n_a, n_b) * (0.5 if args.config == 3 else 2.5)) + 1024) if mode == 0 else n_a
    out_a = torch.empty(cap, dtype=torch.int64, device="cuda"); out_b = torch.empty(cap, dtype=torch.int64, device="cuda")
    out_s = torch.empty(cap, dtype=torch.float64, device="cuda"); cnt = torch.zeros(1, dtype=torch.int64, device="cuda")
    h_out = [torch.empty(cap, dtype=torch.int64).pin_memory(), torch.empty(cap, dtype=torch.int64).pin_memory(),
             torch.empty(cap, dtype=torch.float64).pin_memory()]

    ev = lambda: torch.cuda.Event(enable_timing=True)

    shared = args.grid == "shared"

    def step(devA, devB, marks=None):
        if marks is not None: marks[0].record()
        ib = P.hlc2_build_index(devB[0], devB[1], devB[2], opts=opts_b, temp=temp, buf=buf_b)
        if marks is not None: marks[1].record()
        ia = P.hlc2_build_index(devA[0], devA[1], devA[2], opts=opts_a, temp=temp, buf=buf_a, like=ib if shared else None)
        if marks is not None: marks[2].record()
        P.hlc2_crossmatch(ia, ib, r, mode, out_a, out_b, out_s, cnt, temp=temp)
        if marks is not None: marks[3].record()
        return ia, ib

    def barrier():
        if use_dist:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(args.warmup):
        ia, ib = step(dA, dB)
    torch.cuda.synchronize()
    found = int(cnt.item())
    assert found <= cap, f"output capacity {cap} too small for {found} rows"
    assert P.hlc2_index_status(ia)[0] == 0 and P.hlc2_index_status(ib)[0] == 0, "index status"
    grid_a, grid_b = P.hlc2_grid_describe(ia), P.hlc2_grid_describe(ib)

    # ---- timed region 1: inputs resident in HBM (inputs 3.6 GB >> 126 MB L2, so every step starts cold) ----
    marks = [[ev() for _ in range(4)] for _ in range(args.steps)]
    clocks = ClockSampler(local_rank); clocks.start()
    n0 = P.kernel_launches()
    barrier()
    e0, e1 = ev(), ev()
    e0.record()
    for k in range(args.steps):
        step(dA, dB, marks[k])
    e1.record()
    barrier()
    launches = P.kernel_launches() - n0
    t_ms = e0.elapsed_time(e1)
    ph = np.array([[m[0].elapsed_time(m[1]), m[1].elapsed_time(m[2]), m[2].elapsed_time(m[3])] for m in marks])
    t_build_b, t_build_a, t_match = ph.mean(axis=0)

    # ---- the dominant kernel alone: CUDA events recorded by the library around k_match on this stream (the planner and
    # the count memset of the hlc2_crossmatch call are left out), one launch at a time on the indices of the last step ----
    kms = []
    k0, k1 = ev(), ev()
    k0.record(); k1.record()                       # torch creates the CUDA events lazily: record once so that they exist
    for _ in range(max(5, args.steps)):
        P.hlc2_crossmatch(ia, ib, r, mode, out_a, out_b, out_s, cnt, temp=temp, events=(k0, k1))
        k1.synchronize()
        kms.append(k0.elapsed_time(k1))
    t_kernel = float(np.mean(kms))

    # ---- timed region 2 (e2e): host buffers, H2D of the inputs and D2H of the results inside the region ----
    def e2e_step():
        da = [t.cuda(non_blocking=True) for t in hA]; db = [t.cuda(non_blocking=True) for t in hB]
        step(da, db)
        nf = int(cnt.item())                       # D2H of the count (sync), then of the rows found
        for src, dst in zip((out_a, out_b, out_s), h_out):
            dst[:nf].copy_(src[:nf], non_blocking=True)
        return nf
    e2e_step(); torch.cuda.synchronize()
    barrier()
    g0, g1 = ev(), ev()
    g0.record()
    for _ in range(args.steps):
        nf = e2e_step()
    g1.record()
    barrier()
    t_e2e_ms = g0.elapsed_time(g1)

    # ---- timed region 3 (e2e, streamed): the same host buffers bucketed into declination bands beforehand, one call of
    # hlc2_stream_crossmatch per step: H2D of band k+1, build + match of band k and D2H of band k-1 overlap ----
    t_stream_ms, stream_info = None, None
    if not args.no_stream:
        nb = args.bands if args.bands > 0 else 32
        edges = np.quantile(w.A.dec[:: max(1, n_a // 2_000_000)], np.linspace(0.0, 1.0, nb + 1))
        edges[0], edges[-1] = -90.0, 90.0
        Ab, a_off = S.to_bands(w.A, edges); Bb, b_off = S.to_bands(w.B, edges)
        sA = [pin(Ab.ra), pin(Ab.dec), pin(Ab.id)]; sB = [pin(Bb.ra), pin(Bb.dec), pin(Bb.id)]
        del Ab, Bb
        max_a, max_b = int(np.diff(a_off).max()), int(np.diff(b_off).max())
        mbo = max(1024, (3 * found) // nb) if mode == 0 else max_a
        opts_s = P.make_opts(r, target_occupancy=args.occupancy)
        arena = torch.empty(P.hlc2_stream_sizes(max_a, max_b, opts_s, mbo), dtype=torch.uint8, device="cuda")
        t_off = [torch.from_numpy(a_off), torch.from_numpy(b_off), torch.from_numpy(np.ascontiguousarray(edges))]
        def stream_step():
            return P.hlc2_stream_crossmatch(sA, t_off[0], sB, t_off[1], t_off[2], r, mode, opts_s, h_out[0], h_out[1], h_out[2], arena, mbo)
        nfs = stream_step()
        assert nfs == found, f"streamed path found {nfs} rows, resident path {found}"
        barrier()
        s0, s1 = ev(), ev()
        s0.record()
        for _ in range(args.steps):
            stream_step()                          # synchronous call: returns when the pinned outputs are complete
        s1.record()
        barrier()
        t_stream_ms = s0.elapsed_time(s1)
        stream_info = {"bands": nb, "max_band_a": max_a, "max_band_b": max_b, "arena_bytes": int(arena.numel())}
    clk = clocks.stop()                            # sampled across the timed regions
    h2d = 24 * (n_a + n_b); d2h = 24 * nf + 8

    if use_dist:
        tt = torch.tensor([t_ms, t_e2e_ms, t_match, t_stream_ms or 0.0], dtype=torch.float64, device="cuda")
        dist.all_reduce(tt, op=dist.ReduceOp.MAX)
        t_ms, t_e2e_ms, t_match_max, ts_ = tt.tolist()
        t_stream_ms = ts_ if t_stream_ms is not None else None
        tot = torch.tensor([n_a, found], dtype=torch.float64, device="cuda")
        dist.all_reduce(tot, op=dist.ReduceOp.SUM)
        units, pairs_all = tot.tolist()
    else:
        units, pairs_all = float(n_a), float(found)

    if rank == 0:
        peak, peak_src = peak_hbm()
        alg_bytes = 32.0 * n_a + 32.0 * n_b + 24.0 * found          # catalogue (sorted SoA) + output bytes
        achieved = alg_bytes / (t_kernel * 1e-3) / 1e9
        tr, tr_note = ncu_traffic()
        roof = {"bound": "hbm", "kernel": "k_match_same (+ k_match_general_rows)" if shared else "k_match", "achieved": achieved, "peak": peak, "unit": "GB/s",
                "frac": achieved / peak, "frac_of_nominal_8TBs": achieved / 8000.0, "peak_source": peak_src,
                "traffic": tr["dram_bytes_per_launch"] if tr else None, "traffic_source": tr_note, "algorithmic_bytes": alg_bytes,
                "ms_per_launch": t_kernel, "launches_timed": len(kms),
                "timing": "the caller's CUDA events recorded by the library around the match kernel(s) on the caller's stream (hlc2_crossmatch_events)",
                "whole_call": {"ms": float(t_match), "frac": alg_bytes / (t_match * 1e-3) / 1e9 / peak,
                               "what": "hlc2_crossmatch inside the timed steps: memsets + every kernel of the call"}}
        cpu, verify = None, None
        if not args.no_cpu_baseline:
            whole = args.sample_ra_deg >= 360.0
            sa, sb = (w.A, w.B) if whole else sample_patch(w, 0.0, args.sample_ra_deg)
            dt, npairs, used, rows = time_oracle(sa, sb, r, mode, keep=True)
            cpu = {"value": len(sa) / dt, "unit": UNIT, "cores": used, "kind": "oracle", "seconds": dt,
                   "sample": (f"the whole workload: {len(sa)} x {len(sb)} sources, {npairs} rows" if whole else
                              f"both catalogues restricted to RA in [0,{args.sample_ra_deg}) deg: {len(sa)} x {len(sb)} sources, {npairs} rows")}
            if whole and not args.no_verify:
                # the oracle's rows are the expected result of the very arrays the GPU just matched: compare them
                # element by element (tests/fullsize.py: the comparison procedure of SURVEY 8(c))
                from tests import fullsize
                gk, gs = fullsize.gpu_rows_sorted(out_a[:found], out_b[:found], out_s[:found])
                rep = fullsize.compare_packed(gk, gs, fullsize.pack(rows[0], rows[1]), rows[2], r, w.A, w.B, nearest=mode == 1)
                verify = {"against": "oracle, whole workload, element by element", **rep}
            del rows
        resident = {"value": units * args.steps / (t_e2e_ms * 1e-3), "ms_per_step": t_e2e_ms / args.steps,
                    "path": "pinned host -> H2D -> hlc2_build_index x2 -> hlc2_crossmatch -> D2H of count and rows"}
        pcie = pcie_rates()
        e2e = {"unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h, "resident_path": resident, "pcie": pcie}
        if t_stream_ms is not None:
            streamed = {"value": units * args.steps / (t_stream_ms * 1e-3), "ms_per_step": t_stream_ms / args.steps,
                        "path": "pinned host bands -> hlc2_stream_crossmatch (H2D, build, match, D2H overlapped on 3 streams)",
                        "timing": "CUDA events on the caller's stream around the synchronous calls (the library runs on 3 streams of its own)", **stream_info}
            e2e["streamed_path"] = streamed
        best = e2e.get("streamed_path", resident) if e2e.get("streamed_path", resident)["value"] > resident["value"] else resident
        e2e.update({"value": best["value"], "ms_per_step": best["ms_per_step"], "path": best["path"]})
        # roofline of the end-to-end number: the step's H2D and D2H bytes at the measured pinned copy rates (the two
        # directions overlap on the PCIe link, so the bound is the slower of the two, not their sum)
        t_pcie = max(h2d / (pcie["h2d_gbs"] * 1e9), d2h / (pcie["d2h_gbs"] * 1e9))
        e2e["roofline"] = {"bound": "pcie", "ms_at_peak": 1e3 * t_pcie, "frac": 1e3 * t_pcie / best["ms_per_step"]}
        line = {"metric": METRIC, "value": units * args.steps / (t_ms * 1e-3), "unit": UNIT, "n_gpus": world,
                "steps": args.steps, "warmup": args.warmup, "ms_per_step": t_ms / args.steps, "higher_is_better": True,
                "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
                "config": {"workload": w.name, "n_a": n_a, "n_b": n_b, "radius_arcsec": r,
                           "mode": "nearest" if mode else "all_pairs", "rows_found": found,
                           "parallelism": "replicas only (north_star: one GPU, no collectives)" if world > 1 else "1 gpu",
                           "l2": "inputs (3.6 GB at scale 1) larger than L2; no explicit flush", "grid": args.grid,
                           "cells_a": grid_a["n_cells"], "cells_b": grid_b["n_cells"], "cell_arcsec_b": grid_b["cell_arcsec"],
                           "gen_seconds": t_gen},
                "pairs_per_s": pairs_all * args.steps / (t_ms * 1e-3),
                "match_phase": {"ms": float(t_match), "a_sources_per_s": n_a / (t_match * 1e-3), "pairs_per_s": found / (t_match * 1e-3)},
                "phases_ms": {"build_index_A": float(t_build_a), "build_index_B": float(t_build_b), "crossmatch": float(t_match)},
                "roofline": roof, "cpu_baseline": cpu, "verify": verify,
                "e2e": e2e,
                "gpu_launches": int(launches), "clocks": clk}
        print(json.dumps(line), flush=True)
    if use_dist:
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
