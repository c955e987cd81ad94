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
    src = os.path.join(ROOT, "paper_2301_07331_b200", "csrc", "hlc2_match.cu")
    sha = hashlib.sha256(open(src, "rb").read()).hexdigest()
    if rec.get("hlc2_match_cu_sha256") != sha:
        return None, f"stale: {p} was captured on another version of hlc2_match.cu"
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


def run_config5(args, clocks_index=0):
    """Configuration 5 ("Streamed large", nearest): the catalogues never sit in HBM as a whole; one step = one call of
    hlc2_stream_crossmatch over all declination bands from pinned host memory (H2D of the next bands, index build + match
    of the current one and D2H of the previous one's rows overlap on three streams).  Bound by the PCIe link, so the
    roofline is the measured pinned copy rate.  At scale 1 the pinned inputs are 48 GB (ids implicit) and generation
    takes a quarter of an hour on the box's 16 cores; --scale states the fraction actually run."""
    import torch
    import hlc2_synth as S
    import paper_2301_07331_b200 as P
    import oracle
    from tests import parity
    scale = args.scale
    t0 = time.perf_counter()
    w = S.config(5, scale=scale)
    t_gen = time.perf_counter() - t0
    n_a, n_b, r, mode = len(w.A), len(w.B), w.radius_arcsec, 1
    nb = args.bands
    edges = np.quantile(w.A.dec[:: max(1, n_a // 2_000_000)], np.linspace(0.0, 1.0, nb + 1))
    edges[0], edges[-1] = -90.0, 90.0
    t0 = time.perf_counter()
    # band order without the id columns (ids are implicit: the global row numbers of the banded arrays)
    def bands_of(cat):
        k = np.clip(np.searchsorted(edges, cat.dec, side="right") - 1, 0, nb - 1).astype(np.int16)
        off = np.zeros(nb + 1, np.int64); np.cumsum(np.bincount(k, minlength=nb), out=off[1:])
        order = np.argsort(k, kind="stable"); del k
        ra = cat.ra[order]; dec = cat.dec[order]
        return ra, dec, off
    w.planted_a = None; w.planted_b = None               # multi-GB bookkeeping of the generator, not needed here
    a_ra, a_dec, a_off = bands_of(w.A); w.A = None      # free each original as soon as its banded copy exists
    b_ra, b_dec, b_off = bands_of(w.B); w.B = None
    del w
    import gc; gc.collect()
    t_band = time.perf_counter() - t0
    sA = [host_register(a_ra), host_register(a_dec), None]; sB = [host_register(b_ra), host_register(b_dec), None]
    max_a, max_b = int(np.diff(a_off).max()), int(np.diff(b_off).max())
    cap = int(0.45 * n_a) + 1024
    mbo = max_a
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
    e0, e1 = ev(), ev(); e0.record()
    for _ in range(args.steps):
        found = step()
    e1.record(); torch.cuda.synchronize()
    launches = P.kernel_launches() - n0
    clk = clocks.stop()
    t_ms = e0.elapsed_time(e1) / args.steps
    pcie = pcie_rates()
    h2d, d2h = 16 * (n_a + n_b), 24 * found
    t_pcie = max(h2d / (pcie["h2d_gbs"] * 1e9), d2h / (pcie["d2h_gbs"] * 1e9))
    # ---- parity on a stated sample of bands: every 16th, both polar bands, and the bands next to them
    ga = h_out[0][:found].numpy(); gb_ = h_out[1][:found].numpy(); gs = h_out[2][:found].numpy()
    sample = sorted(set(list(range(0, nb, 16)) + [0, 1, nb - 2, nb - 1]) & set(range(nb)))
    ver = {"bands_checked": sample, "rows_gpu": 0, "rows_oracle": 0, "only_gpu": 0, "only_oracle": 0, "borderline": 0, "swaps": 0, "max_sep_err": 0.0}
    t_or = 0.0; used = 0
    for k in sample:
        a0, a1 = int(a_off[k]), int(a_off[k + 1]); lo, hi = max(k - 1, 0), min(k + 1, nb - 1)
        b0, b1 = int(b_off[lo]), int(b_off[hi + 1])
        A = S.Catalogue(a_ra[a0:a1], a_dec[a0:a1], np.arange(a0, a1, dtype=np.int64)); B = S.Catalogue(b_ra[b0:b1], b_dec[b0:b1], np.arange(b0, b1, dtype=np.int64))
        t1 = time.perf_counter()
        oa, ob, os_, used = oracle.match(A.ra, A.dec, A.id, B.ra, B.dec, B.id, r, mode)
        t_or += time.perf_counter() - t1
        m = (ga >= a0) & (ga < a1)
        rep = parity.compare_nearest((ga[m], gb_[m], gs[m]), (oa, ob, os_), r, parity.make_sep_of(A, B))
        ver["rows_gpu"] += int(m.sum()); ver["rows_oracle"] += len(oa)
        ver["borderline"] += len(rep["borderline"]); ver["swaps"] += len(rep.get("swaps", []))
        ver["max_sep_err"] = max(ver["max_sep_err"], float(rep["max_sep_err"]))
    a_checked = int(sum(a_off[k + 1] - a_off[k] for k in sample))
    line = {"metric": METRIC, "value": n_a / (t_ms * 1e-3), "unit": UNIT, "n_gpus": 1, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": t_ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": "cfg5_streamed_large", "scale": scale, "n_a": n_a, "n_b": n_b, "radius_arcsec": r, "mode": "nearest",
                       "rows_found": int(found), "bands": nb, "max_band_a": max_a, "max_band_b": max_b, "arena_bytes": int(arena.numel()),
                       "ids": "implicit (global row numbers of the banded arrays)", "gen_seconds": t_gen, "band_seconds": t_band,
                       "note": "scale 1 = 2e9 x 1e9; the fraction run is stated here"},
            "e2e": {"value": n_a / (t_ms * 1e-3), "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                    "path": "pinned host bands -> hlc2_stream_crossmatch (H2D, build, match, D2H overlapped on 3 streams)"},
            "roofline": {"bound": "pcie", "achieved": h2d / (t_ms * 1e-3) / 1e9, "peak": pcie["h2d_gbs"], "unit": "GB/s",
                         "frac": (h2d / (t_ms * 1e-3) / 1e9) / pcie["h2d_gbs"], "traffic": None, "pcie": pcie, "ms_at_peak": 1e3 * t_pcie},
            "cpu_baseline": {"value": a_checked / t_or if t_or else None, "unit": UNIT, "cores": used, "kind": "oracle",
                             "sample": f"the {len(sample)} checked bands: {a_checked} A sources against their three-band B windows"},
            "verify": ver, "gpu_launches": int(launches), "clocks": clk}
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
    ap.add_argument("--bands", type=int, default=16, help="declination bands of the streamed e2e leg")
    ap.add_argument("--no-stream", action="store_true", help="skip the streamed e2e leg")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    rank, local_rank, world = dist_env()

    import hlc2_synth as S
    if args.impl == "reference" and rank != 0:
        return 0
    if args.config == 5 and args.impl == "ours":
        import torch
        from paper_2301_07331_b200 import build as hb
        hb.build()
        torch.cuda.set_device(local_rank)
        if args.bands == 16: args.bands = 64
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

    opts_a = P.make_opts(r, target_occupancy=args.occupancy); opts_b = P.make_opts(r, target_occupancy=args.occupancy if args.occupancy_b is None else args.occupancy_b)
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
    cap = int(max(n_a, n_b) * 0.5) + 1024 if mode == 0 else n_a
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
        nb = args.bands
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
        roof = {"bound": "hbm", "kernel": "k_match", "achieved": achieved, "peak": peak, "unit": "GB/s",
                "frac": achieved / peak, "frac_of_nominal_8TBs": achieved / 8000.0, "peak_source": peak_src,
                "traffic": tr["dram_bytes_per_launch"] if tr else None, "traffic_source": tr_note, "algorithmic_bytes": alg_bytes,
                "ms_per_launch": t_kernel, "launches_timed": len(kms),
                "timing": "the caller's CUDA events recorded by the library around k_match on the caller's stream (hlc2_crossmatch_events)",
                "whole_call": {"ms": float(t_match), "frac": alg_bytes / (t_match * 1e-3) / 1e9 / peak,
                               "what": "hlc2_crossmatch inside the timed steps: count memset + k_plan + k_match"}}
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
