// hlc2_match.cu -- the match kernels (NS (b)).
//
// Work unit = one A tile: up to kTile consecutive cell-sorted A rows of one A zone.  Two kernels:
//
//   k_plan   one thread per A tile.  From the tile's own cell bounds (exact: zone edges and RA-cell edges of
//            A's grid) it derives the window on B's grid that any row of the tile can reach:
//              dec  [dec_lo - r, dec_hi + r]                           -> consecutive zones of B's grid
//              RA   [ra_lo - W, ra_hi + W], W >= asin(sin r / cos dec*) -> one cell range per zone, a second one
//                   when the window passes RA = 0/360, the whole ring at the poles
//            (the cells the quad-direction strategy probes, plus the diagonal neighbours and
//            the 1/cos(dec) widening it omits, so no pair is lost: the "No Index" result, L344).  The window is
//            cut into pieces (zone, cell range, B row range) and the pieces are packed into jobs that fit one
//            shared-memory stage -- the role of the paper's calculation blocks, L253-257, which were cut to fit
//            device memory.  jobs[t] is the first job of tile t; further jobs hang off it through `next`.
//            Only a tile that reaches more than kMaxZones zones of B's grid (B far denser than A) or that finds
//            the job pool full is marked DIRECT.
//   k_match  persistent CTAs of kCW consumer warps + 1 producer warp around a kStages-deep mbarrier ring.  The
//            producer warp turns each job into 1-D bulk copies (cp.async.bulk, the TMA engine): the A tile (x, y,
//            z, pos) and, per piece, B's x, y, z rows and the cell_start slice -- all contiguous because
//            keys are zone-major / RA-minor.  Consumers: one lane per A row (the paper's thread-per-A-record
//            hierarchy, L271-276).  A lane locates its own cells from the fp32 (ra, dec) estimate padded by a
//            rigorous error bound, clips them to the piece (the jobs of a tile cover every cell a row of the tile
//            needs, so clipping never loses one), reads its row range from the staged cell_start slice and tests
//            the staged rows: chord^2 <= 4 sin^2(r/2), all fp64 from shared memory, two candidates per step
//            without branches.  Hits (the role of d_out_dis, L282) are compacted by ballot + popcount into a
//            per-warp queue of (A row, B row, chord^2) and flushed 32 at a time: one global atomic, the id
//            look-ups, coalesced stores, sep computed on full warps.  DIRECT tiles run the general per-lane path
//            from global memory.
//
// Decisions are fp64; the fp32 estimate only ever selects a superset of cells.
#include <math.h>

#include <algorithm>

#include "hlc2_match_common.cuh"

namespace hlc2 {

#ifndef HLC2_STAGES
#define HLC2_STAGES 2
#endif
#ifndef HLC2_BCAP
#define HLC2_BCAP 320
#endif
#ifndef HLC2_CSCAP
#define HLC2_CSCAP 1024
#endif
#ifndef HLC2_CTAS
#define HLC2_CTAS 6
#endif
constexpr int kStages = HLC2_STAGES;
constexpr int kSegs = 3;                     // window pieces per job
constexpr int kBCap = HLC2_BCAP;             // staged B rows per job, all pieces, after 16-byte alignment
constexpr int kCsCap = HLC2_CSCAP;           // staged cell_start entries per job, after alignment
constexpr int kAPad = kTile + 2;             // A tile rows after alignment to 16 bytes
constexpr int kMaxZones = 8;                 // tiles whose window spans more zones of B's grid take the general path

// job flags (bits 0-3: number of pieces)
constexpr uint32_t kJobDirect = 1u << 8;     // general per-lane path from global memory
constexpr uint32_t kJobRing = 1u << 9;       // every row takes all cells of every piece (polar tiles)
constexpr uint32_t kJobWrap = 1u << 10;      // window touches u = 0 / 360: rows re-centre their RA on each piece
constexpr uint32_t kJobFirst = 1u << 11;     // first / last job of its A tile (nearest mode carries the best across jobs)
constexpr uint32_t kJobLast = 1u << 12;
constexpr uint32_t kJobEnd = 1u << 13;       // producer -> consumers: no more work

// 128-byte job record (32 words).  jobs[t] is the first job of A tile t; further jobs of a tile (windows that do
// not fit one stage: the paper's calculation blocks, L253-257, cut to fit shared memory) are chained by `next`.
// A piece = cells [k_lo, k_lo + nk) of one zone of B's grid restricted to B rows [row_lo, row_lo + n_rows).
struct JobSeg { int32_t zone, k_lo; uint32_t nk, row_lo, n_rows; int32_t n_ra; uint32_t cs_lo; float centre; };
struct Job { uint32_t a_first, a_count, flags, next; JobSeg seg[kSegs]; uint32_t pad[4]; };
static_assert(sizeof(JobSeg) == 32 && sizeof(Job) == 128, "the producer reads a job as 32 words");

struct SegDesc { double n_d; double centre; int32_t zone, k_lo, k_hi, cdelta; uint32_t rdelta, row_lo, row_hi; int32_t pad; };
struct StageDesc { uint32_t a_first, a_count, a_off, flags; int32_t nseg; uint32_t pad; SegDesc seg[kSegs]; };

struct __align__(16) Stage {
    double ax[kAPad], ay[kAPad], az[kAPad];
    float2 apos[kAPad];
    double bx[kBCap + 2], by[kBCap + 2], bz[kBCap + 2];     // slot kBCap: a point no chord test can reach
    uint32_t cs[kCsCap];
    StageDesc d;
};
struct __align__(16) MatchSmem {
    Stage st[kStages];
    WarpQueue q[kCW];
    unsigned long long full[kStages], empty[kStages];
};
static_assert((kAPad * 8) % 16 == 0 && (kBCap * 8) % 16 == 0 && (kCsCap * 4) % 16 == 0, "bulk copies need 16-byte pieces");
static_assert(sizeof(Stage) % 16 == 0, "stages stay 16-byte aligned");

// ------------------------------------------------------------------------------------------------------
// k_plan: the jobs of every A tile
// ------------------------------------------------------------------------------------------------------
struct PlanState {
    uint32_t w[32];            // the job being assembled
    uint32_t slot;             // where it will be written
    uint32_t rows_used, cs_used;
    int nseg;
    bool first, overflow;
};

__device__ __forceinline__ void plan_store(Job* jobs, uint32_t slot, const uint32_t* w) {
    uint4* o = reinterpret_cast<uint4*>(jobs + slot);
#pragma unroll
    for (int i = 0; i < 8; ++i) o[i] = make_uint4(w[4 * i], w[4 * i + 1], w[4 * i + 2], w[4 * i + 3]);
}

// write the assembled job; unless it is the tile's last one, take a pool slot for its successor
__device__ __noinline__ void plan_close(PlanState& st, const MatchArgs& p, uint32_t common, bool last) {
    uint32_t next = 0;
    if (!last) {
        const uint32_t idx = atomicAdd(p.pool_count, 1u);
        if (idx >= p.pool_cap) { st.overflow = true; return; }
        next = p.tile_cap + idx;
    }
    st.w[2] = (uint32_t)st.nseg | common | (st.first ? kJobFirst : 0u) | (last ? kJobLast : 0u);
    st.w[3] = next;
    plan_store(p.jobs, st.slot, st.w);
    st.slot = next; st.first = false; st.nseg = 0; st.rows_used = 0; st.cs_used = 0;
#pragma unroll
    for (int i = 4; i < 32; ++i) st.w[i] = 0;
}

// cells [ka, kb] of zone z: cut into pieces that fit what is left of the current job, opening new jobs as needed
__device__ __noinline__ void plan_piece(PlanState& st, const MatchArgs& p, const uint32_t* __restrict__ cs, uint32_t common,
                                        int z, int n, uint32_t cb, int ka, int kb, float centre) {
    uint32_t ra = __ldg(cs + cb + (uint32_t)ka);
    const uint32_t rb = __ldg(cs + cb + (uint32_t)kb + 1u);
    while (ra < rb && !st.overflow) {
        if (st.nseg == kSegs || st.rows_used + 4u > (uint32_t)kBCap || st.cs_used + 12u > (uint32_t)kCsCap) {
            plan_close(st, p, common, false);
            if (st.overflow) return;
        }
        const uint32_t max_rows = (uint32_t)kBCap - st.rows_used - 2u, max_cells = (uint32_t)kCsCap - st.cs_used - 8u;
        int ke = (int)min((long long)kb, (long long)ka + (long long)max_cells - 1);
        uint32_t re = ke == kb ? rb : __ldg(cs + cb + (uint32_t)ke + 1u);
        if (re - ra > max_rows) {
            re = ra + max_rows;
            int lo = ka, hi = ke;                           // largest k with cs[k] < re: the cell holding row re - 1
            while (lo < hi) {
                const int mid = (int)(((long long)lo + hi + 1) >> 1);
                if (__ldg(cs + cb + (uint32_t)mid) < re) lo = mid; else hi = mid - 1;
            }
            ke = lo;
        }
        if (re == ra) { ka = ke + 1; continue; }             // a run of empty cells (ke < kb here): nothing to stage
        uint32_t* s = st.w + 4 + 8 * st.nseg;
        s[0] = (uint32_t)z; s[1] = (uint32_t)ka; s[2] = (uint32_t)(ke - ka + 1); s[3] = ra; s[4] = re - ra;
        s[5] = (uint32_t)n; s[6] = cb + (uint32_t)ka; s[7] = __float_as_uint(centre);
        st.rows_used += ((re + 1u) & ~1u) - (ra & ~1u);
        st.cs_used += ((cb + (uint32_t)ke + 2u + 3u) & ~3u) - ((cb + (uint32_t)ka) & ~3u);
        ++st.nseg;
        if (re >= rb) break;
        ra = re;
        ka = (ke < kb && __ldg(cs + cb + (uint32_t)ke + 1u) <= re) ? ke + 1 : ke;     // the cell holding row `re`
    }
}

__global__ void __launch_bounds__(128)
k_plan(const __grid_constant__ IndexView A, const __grid_constant__ IndexView B, const __grid_constant__ MatchArgs p) {
    const uint32_t nt = __ldg(A.n_tiles);
    const GridView& ga = A.g;
    const GridView& gb = B.g;
    for (uint32_t t = blockIdx.x * 128 + threadIdx.x; t < nt; t += gridDim.x * 128) {
        const uint4 t0 = __ldg(reinterpret_cast<const uint4*>(A.tiles + t));        // first, count, zone, k_first
        const uint4 t1 = __ldg(reinterpret_cast<const uint4*>(A.tiles + t) + 1);    // k_last, flags, n, cb
        PlanState st;
#pragma unroll
        for (int i = 0; i < 32; ++i) st.w[i] = 0;
        st.w[0] = t0.x; st.w[1] = t0.y;
        st.slot = t; st.rows_used = 0; st.cs_used = 0; st.nseg = 0; st.first = true; st.overflow = false;
        const int za = (int)t0.z;
        // declination and RA bounds of the tile's rows: the edges of its zone and of its first / last cell in
        // A's grid (rows were filed by the same floor expressions; kTinyDeg covers their rounding)
        const double dlo = za == 0 ? ga.dec_min : fmax(ga.dec_min, ga.dec_lo + (double)za * ga.h - kTinyDeg);
        const double dhi = za == ga.n_zones - 1 ? ga.dec_max : fmin(ga.dec_max, ga.dec_lo + (double)(za + 1) * ga.h + kTinyDeg);
        const double qlo = dlo - p.r_deg - kTinyDeg, qhi = dhi + p.r_deg + kTinyDeg;
        const bool empty = qhi < gb.dec_min || qlo > gb.dec_max || t0.y == 0;
        bool direct = false;
        uint32_t common = 0;
        if (!empty) {
            const int zb0 = zone_of(gb, qlo), zb1 = zone_of(gb, qhi);
            if (zb1 - zb0 + 1 > kMaxZones) direct = true;
            const double cw = ga.span / (double)__ldg(ga.n_ra + za);
            const double ua_lo = (double)t0.w * cw - kTinyDeg, ua_hi = (double)(t1.x + 1u) * cw + kTinyDeg;
            // RA half-window of the most poleward row: sin(dRA) = sin r / cos dec; the rows bound asin(s) by
            // 1.011 s (s < 0.25) from their own fp32 cos dec; the extra 1.001 and kEpsRaDeg keep W above all of them
            const double dabs = fmin(90.0, fmax(fabs(dlo), fabs(dhi)));
            const double s = (double)p.sin_r_up / fmax(cos(dabs * 0.017453292519943295), 1e-300);
            const double W = s * (1.011 * 57.29577951308232 * 1.001) + 2.0 * kEpsRaDeg;
            double ub = (ga.ra0 + ua_lo) - gb.ra0;
            ub -= 360.0 * floor(ub * (1.0 / 360.0));
            if (!(ub >= 0.0 && ub < 360.0)) ub = 0.0;
            const double L = ub - W, H = ub + (ua_hi - ua_lo) + W;           // the tile's RA window in B's box frame
            const bool ring = !(s < 0.2) || !(H - L < 300.0);
            // up to two RA intervals inside [0, span]: the window itself and its image through u = 0 / 360
            double ilo[2], ihi[2]; float ctr[2]; int ni = 0;
            if (ring) { common |= kJobRing; ilo[0] = 0.0; ihi[0] = gb.span; ctr[0] = 0.0f; ni = 1; }
            else {
                if (!(L >= 2.0 * kEpsRaDeg) || !(H + 2.0 * kEpsRaDeg < 360.0)) common |= kJobWrap;
                const float c = (float)(0.5 * (L + H));
                if (H >= 0.0 && L <= gb.span) { ilo[ni] = fmax(L, 0.0); ihi[ni] = fmin(H, gb.span); ctr[ni] = c; ++ni; }
                if (L < 0.0 && L + 360.0 <= gb.span) { ilo[ni] = L + 360.0; ihi[ni] = fmin(H + 360.0, gb.span); ctr[ni] = c + 360.0f; ++ni; }
                else if (H >= 360.0) { ilo[ni] = fmax(L - 360.0, 0.0); ihi[ni] = fmin(H - 360.0, gb.span); ctr[ni] = c - 360.0f; ++ni; }
            }
            // two RA intervals whose cell ranges meet in some zone (few cells per zone: polar zones next to the seam)
            // would stage those cells twice and report their pairs twice: such tiles take the general path, whose
            // per-row ranges are merged before they are scanned
            if (!direct && ni == 2)
                for (int z = zb0; z <= zb1; ++z) {
                    const int n = __ldg(gb.n_ra + z);
                    const int a0 = cell_of_u(gb, ilo[0], n), a1 = cell_of_u(gb, ihi[0], n);
                    const int b0 = cell_of_u(gb, ilo[1], n), b1 = cell_of_u(gb, ihi[1], n);
                    if (!(a1 < b0 || b1 < a0)) { direct = true; break; }
                }
            if (!direct) {
                for (int i = 0; i < ni && !st.overflow; ++i)
                    for (int z = zb0; z <= zb1 && !st.overflow; ++z) {
                        const int n = __ldg(gb.n_ra + z);
                        const uint32_t cb = __ldg(gb.cell_base + z);
                        const int k0 = ring ? 0 : cell_of_u(gb, ilo[i], n), k1 = ring ? n - 1 : cell_of_u(gb, ihi[i], n);
                        plan_piece(st, p, B.cell_start, common, z, n, cb, k0, k1, ctr[i]);
                    }
                if (st.overflow) direct = true;
            }
        }
        if (direct) {                       // general path: one job, no pieces (rewrites the tile's first job)
#pragma unroll
            for (int i = 4; i < 32; ++i) st.w[i] = 0;
            st.w[2] = kJobDirect | kJobFirst | kJobLast; st.w[3] = 0;
            plan_store(p.jobs, t, st.w);
        } else {
            plan_close(st, p, common, true);        // a tile without pieces ends up as one empty job
        }
    }
}

// ------------------------------------------------------------------------------------------------------
// staged scan: every lane tests its rows [p0, p1) of the stage's B arrays (stage slot j holds B row j - delta); the
// trip count is the warp's maximum so that hits can be compacted with one ballot per step
// ------------------------------------------------------------------------------------------------------
template <int MODE>
__device__ __forceinline__ void scan_staged(const IndexView& A, const IndexView& B, const Stage& st, const MatchArgs& p,
                                            WarpQueue& q, unsigned& qn, uint32_t a_row, double ax, double ay, double az,
                                            unsigned p0, unsigned p1, uint32_t delta, Best& best, int lane) {
    const unsigned len = p1 - p0;
    const unsigned mx = __reduce_max_sync(kFull, len);
    // two candidates per step, no branches: a lane past its range reads the sentinel slot, which never matches
    for (unsigned i = 0; i < mx; i += 2) {
        const unsigned j0 = i < len ? p0 + i : (unsigned)kBCap;
        const unsigned j1 = i + 1 < len ? p0 + i + 1 : (unsigned)kBCap;
        const double dx0 = ax - st.bx[j0], dy0 = ay - st.by[j0], dz0 = az - st.bz[j0];
        const double dx1 = ax - st.bx[j1], dy1 = ay - st.by[j1], dz1 = az - st.bz[j1];
        const double c20 = fma(dx0, dx0, fma(dy0, dy0, dz0 * dz0));
        const double c21 = fma(dx1, dx1, fma(dy1, dy1, dz1 * dz1));
        const bool h0 = c20 <= p.thr2, h1 = c21 <= p.thr2;
        if (MODE == HLC2_ALL_PAIRS) {
            push_hits(A, B, p, q, qn, h0, a_row, j0 - delta, c20, lane);
            push_hits(A, B, p, q, qn, h1, a_row, j1 - delta, c21, lane);
        } else {
            // ties -> smaller idB: the ids are only fetched when two candidates are exactly equidistant
            if (h0) {
                const uint32_t r = j0 - delta;
                if (!best.has || c20 < best.c2 || (c20 == best.c2 && __ldg(B.id + r) < __ldg(B.id + best.row))) { best.has = true; best.row = r; best.c2 = c20; }
            }
            if (h1) {
                const uint32_t r = j1 - delta;
                if (!best.has || c21 < best.c2 || (c21 == best.c2 && __ldg(B.id + r) < __ldg(B.id + best.row))) { best.has = true; best.row = r; best.c2 = c21; }
            }
        }
    }
}

// a lane's up to two row ranges (rows whose Dec window spans two zones) with the slot -> row offsets of their pieces
struct Ranges { unsigned p0, p1, s0, s1; uint32_t pd, sd; };

// a lane's row ranges in the pieces of a job.  GENERAL: ring and wrap jobs (polar tiles, windows through u = 0 / 360).
template <int MODE, bool GENERAL>
__device__ __forceinline__ void seg_ranges(const IndexView& A, const IndexView& B, const Stage& st, const MatchArgs& p,
                                           WarpQueue& q, unsigned& qn, const GridView& g,
                                           uint32_t flags, int nseg, bool act, int zlo, int zhi, double u, double w,
                                           double vlo0, double vhi0, uint32_t a_row, double ax, double ay, double az,
                                           Best& best, int lane, Ranges& R) {
    const StageDesc& d = st.d;
    for (int sg = 0; sg < nseg; ++sg) {
        const SegDesc& e = d.seg[sg];
        bool has = act && e.zone >= zlo && e.zone <= zhi;
        int k0, k1;
        if (GENERAL && (flags & kJobRing)) { k0 = e.k_lo; k1 = e.k_hi; }
        else {
            double vlo = vlo0, vhi = vhi0;
            if (GENERAL && (flags & kJobWrap)) {           // re-centre this row's RA on the piece, then clip to the box
                double dd = u - e.centre;
                dd = dd > 180.0 ? dd - 360.0 : (dd < -180.0 ? dd + 360.0 : dd);
                const double lo = e.centre + dd - w, hi = e.centre + dd + w;
                has = has && hi >= 0.0 && lo <= g.span;
                vlo = fmax(lo, 0.0) * g.inv_span; vhi = fmin(hi, g.span) * g.inv_span;
            }
            k0 = __double2int_rd(vlo * e.n_d); k1 = __double2int_rd(vhi * e.n_d);
            has = has && k1 >= e.k_lo && k0 <= e.k_hi;
            k0 = min(max(k0, e.k_lo), e.k_hi); k1 = min(max(k1, e.k_lo), e.k_hi);
        }
        unsigned q0 = st.cs[k0 + e.cdelta], q1 = st.cs[k1 + 1 + e.cdelta];
        q0 = min(max(q0, e.row_lo), e.row_hi) + e.rdelta; q1 = min(max(q1, e.row_lo), e.row_hi) + e.rdelta;
        has = has && q1 > q0;
        if (sg >= 2 && __any_sync(kFull, has && R.p1 > R.p0 && R.s1 > R.s0)) {      // a third range: drain first
            scan_staged<MODE>(A, B, st, p, q, qn, a_row, ax, ay, az, R.p0, R.p1, R.pd, best, lane);
            scan_staged<MODE>(A, B, st, p, q, qn, a_row, ax, ay, az, R.s0, R.s1, R.sd, best, lane);
            R.p0 = R.p1 = R.s0 = R.s1 = 0;
        }
        if (has) { if (R.p1 == R.p0) { R.p0 = q0; R.p1 = q1; R.pd = e.rdelta; } else { R.s0 = q0; R.s1 = q1; R.sd = e.rdelta; } }
    }
}

// ------------------------------------------------------------------------------------------------------
// k_match
// ------------------------------------------------------------------------------------------------------
template <int MODE>
__global__ void __launch_bounds__(kMatchThreads, HLC2_CTAS)
k_match(const __grid_constant__ IndexView A, const __grid_constant__ IndexView B, const __grid_constant__ MatchArgs p) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    MatchSmem& sm = *reinterpret_cast<MatchSmem*>(smem_raw);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    if (threadIdx.x == 0) {
        for (int s = 0; s < kStages; ++s) { mbar_init(&sm.full[s], 1); mbar_init(&sm.empty[s], kCW); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (threadIdx.x < kStages) { Stage& st = sm.st[threadIdx.x]; st.bx[kBCap] = 0.0; st.by[kBCap] = 0.0; st.bz[kBCap] = 2.0; }
    __syncthreads();

    if (warp == kCW) {
        // ---------------- producer warp: job -> bulk copies ----------------
        const uint32_t nt = __ldg(A.n_tiles);
        const uint32_t* jw = reinterpret_cast<const uint32_t*>(p.jobs);
        // first jobs of this CTA's tiles are fetched two tiles ahead (one word per lane), so the producer never waits
        // on them; only a chained job (a tile whose window did not fit one stage) is fetched on demand
        uint32_t t = blockIdx.x;
        const uint32_t G = gridDim.x;
        bool have = t < nt;
        uint32_t wcur = have ? __ldg(jw + (size_t)t * 32 + lane) : 0u;
        uint32_t w1 = (t + G < nt) ? __ldg(jw + (size_t)(t + G) * 32 + lane) : 0u;
        uint32_t w2 = (t + 2 * G < nt) ? __ldg(jw + (size_t)(t + 2 * G) * 32 + lane) : 0u;
        uint32_t it = 0;
        for (; have; ++it) {
            const uint32_t next = __shfl_sync(kFull, wcur, 3);
            uint32_t wnext;
            bool nhave = true;
            if (next != 0) wnext = __ldg(jw + (size_t)next * 32 + lane);
            else {
                t += G; nhave = t < nt;
                wnext = w1; w1 = w2;
                w2 = (t + 2 * G < nt) ? __ldg(jw + (size_t)(t + 2 * G) * 32 + lane) : 0u;
            }

            const int s = (int)(it % kStages);
            const unsigned ph = (it / kStages) & 1u;
            Stage& st = sm.st[s];
            const uint32_t a_first = __shfl_sync(kFull, wcur, 0), a_count = __shfl_sync(kFull, wcur, 1);
            const uint32_t flags = __shfl_sync(kFull, wcur, 2);
            const int nseg = (int)(flags & 0xFu);
            const int sb = 4 + 8 * min(lane, kSegs - 1);
            const uint32_t zone = __shfl_sync(kFull, wcur, sb), k_lo = __shfl_sync(kFull, wcur, sb + 1);
            const uint32_t nk = __shfl_sync(kFull, wcur, sb + 2), row_lo = __shfl_sync(kFull, wcur, sb + 3);
            const uint32_t nr = __shfl_sync(kFull, wcur, sb + 4), n_ra = __shfl_sync(kFull, wcur, sb + 5);
            const uint32_t cs_lo = __shfl_sync(kFull, wcur, sb + 6), ctr = __shfl_sync(kFull, wcur, sb + 7);
            const bool segact = lane < nseg;
            const uint32_t row_al = row_lo & ~1u, cs_al = cs_lo & ~3u;
            const uint32_t n_ld = segact ? (((row_lo + nr + 1u) & ~1u) - row_al) : 0u;
            const uint32_t c_ld = segact ? (((cs_lo + nk + 1u + 3u) & ~3u) - cs_al) : 0u;
            uint32_t roff = 0, coff = 0, rtot = 0, ctot = 0;
#pragma unroll
            for (int l = 0; l < kSegs; ++l) {
                const uint32_t a = __shfl_sync(kFull, n_ld, l), c = __shfl_sync(kFull, c_ld, l);
                if (l < lane) { roff += a; coff += c; }
                rtot += a; ctot += c;
            }
            const bool any = nseg != 0 || (flags & kJobDirect);
            const uint32_t a_al = a_first & ~1u;
            const uint32_t a_ld = any ? (((a_first + a_count + 1u) & ~1u) - a_al) : 0u;
            const uint32_t bytes = a_ld * 32u + rtot * 24u + ctot * 4u;

            mbar_wait(&sm.empty[s], ph ^ 1u);
            if (lane == 0) { st.d.a_first = a_first; st.d.a_count = a_count; st.d.a_off = a_first - a_al; st.d.flags = flags; st.d.nseg = nseg; }
            if (segact) {
                SegDesc& e = st.d.seg[lane];
                e.n_d = (double)(int32_t)n_ra; e.centre = (double)__uint_as_float(ctr);
                e.zone = (int32_t)zone; e.k_lo = (int32_t)k_lo; e.k_hi = (int32_t)(k_lo + nk) - 1;
                e.cdelta = (int32_t)((cs_lo - k_lo) - cs_al + coff); e.rdelta = roff - row_al;
                e.row_lo = row_lo; e.row_hi = row_lo + nr;
            }
            __syncwarp();
            if (lane == 0) { if (bytes) mbar_arrive_expect_tx(&sm.full[s], bytes); else mbar_arrive(&sm.full[s]); }
            if (segact) {
                bulk_g2s(st.bx + roff, B.x + row_al, n_ld * 8u, &sm.full[s]);
                bulk_g2s(st.by + roff, B.y + row_al, n_ld * 8u, &sm.full[s]);
                bulk_g2s(st.bz + roff, B.z + row_al, n_ld * 8u, &sm.full[s]);
                bulk_g2s(st.cs + coff, B.cell_start + cs_al, c_ld * 4u, &sm.full[s]);
            }
            if (a_ld && lane >= 8 && lane < 12) {
                const int k = lane - 8;
                const void* src = k == 0 ? (const void*)(A.x + a_al) : k == 1 ? (const void*)(A.y + a_al) : k == 2 ? (const void*)(A.z + a_al)
                                : (const void*)(A.pos + a_al);
                void* dst = k == 0 ? (void*)st.ax : k == 1 ? (void*)st.ay : k == 2 ? (void*)st.az : (void*)st.apos;
                bulk_g2s(dst, src, a_ld * 8u, &sm.full[s]);
            }
            wcur = wnext; have = nhave;
        }
        // tell the consumers that nothing follows
        const int s = (int)(it % kStages);
        mbar_wait(&sm.empty[s], ((it / kStages) & 1u) ^ 1u);
        if (lane == 0) { sm.st[s].d.flags = kJobEnd; sm.st[s].d.nseg = 0; sm.st[s].d.a_count = 0; mbar_arrive(&sm.full[s]); }
        return;
    }

    // ---------------- consumer warps: one lane per A row of the tile ----------------
    const GridView& g = B.g;
    WarpQueue& q = sm.q[warp];
    unsigned qn = 0;
    Best best; best.has = false; best.c2 = 0.0; best.row = 0;
    for (uint32_t it = 0;; ++it) {
        const int s = (int)(it % kStages);
        const unsigned ph = (it / kStages) & 1u;
        mbar_wait(&sm.full[s], ph);
        const Stage& st = sm.st[s];
        const StageDesc& d = st.d;
        const uint32_t flags = d.flags, a_count = d.a_count;
        if (flags & kJobEnd) break;
        const int nseg = d.nseg;
        if ((uint32_t)(warp * 32) < a_count) {
            const bool act = threadIdx.x < a_count;
            if (MODE == HLC2_NEAREST && (flags & kJobFirst)) best.has = false;
            const uint32_t a_row = d.a_first + threadIdx.x;
            if (nseg != 0 || (flags & kJobDirect)) {
                const unsigned ra = act ? threadIdx.x + d.a_off : d.a_off;
                const double ax = st.ax[ra], ay = st.ay[ra], az = st.az[ra];
                const float2 pf = st.apos[ra];
                if (flags & kJobDirect) {
                    if (act) scan_general<MODE>(A, B, p, a_row, ax, ay, az, pf, best);
                    __syncwarp();
                } else {
                    const double dlo = (double)pf.y - p.pad_dec, dhi = (double)pf.y + p.pad_dec;
                    const int zlo = zone_of(g, dlo), zhi = zone_of(g, dhi);
                    const float fx = (float)ax, fy = (float)ay;
                    const float sn = p.sin_r_up * rsqrtf(fx * fx + fy * fy);
                    const double w = (double)(sn * (1.011f * 57.29577951f)) + kEpsRaDeg;
                    const double u = box_u(g, (double)pf.x);
                    const double vlo0 = (u - w) * g.inv_span, vhi0 = (u + w) * g.inv_span;
                    Ranges R; R.p0 = R.p1 = R.s0 = R.s1 = 0; R.pd = R.sd = 0;
                    if (flags & (kJobRing | kJobWrap))
                        seg_ranges<MODE, true>(A, B, st, p, q, qn, g, flags, nseg, act, zlo, zhi, u, w, vlo0, vhi0, a_row, ax, ay, az, best, lane, R);
                    else
                        seg_ranges<MODE, false>(A, B, st, p, q, qn, g, flags, nseg, act, zlo, zhi, u, w, vlo0, vhi0, a_row, ax, ay, az, best, lane, R);
                    scan_staged<MODE>(A, B, st, p, q, qn, a_row, ax, ay, az, R.p0, R.p1, R.pd, best, lane);
                    if (__any_sync(kFull, R.s1 > R.s0)) scan_staged<MODE>(A, B, st, p, q, qn, a_row, ax, ay, az, R.s0, R.s1, R.sd, best, lane);
                }
            }
            if (MODE == HLC2_NEAREST && (flags & kJobLast)) push_hits(A, B, p, q, qn, act && best.has, a_row, best.row, best.c2, lane);
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(&sm.empty[s]);
    }
    __syncwarp();
    if (qn) flush_rows(A, B, p, q, 0, qn, lane);
}

static inline size_t pool_cap_of(size_t tile_cap) { return 3 * tile_cap + 4096; }

size_t match_temp_for_tiles(size_t tile_cap) { return (tile_cap + pool_cap_of(tile_cap)) * sizeof(Job) + 256; }
size_t match_temp_bytes(const IndexView& A, const IndexView& B) {
    return std::max(match_temp_for_tiles(std::max(A.tile_cap, B.tile_cap)), match_same_temp_bytes(A));
}

void launch_match(const IndexView& A_in, const IndexView& B_in, double radius_arcsec, int mode,
                  int64_t* out_ida, int64_t* out_idb, double* out_sep, unsigned long long capacity,
                  unsigned long long* d_count, void* d_temp, cudaStream_t s, uint32_t match_flags,
                  cudaEvent_t ev_start, cudaEvent_t ev_stop, const MatchExtra* ex) {
    if (A_in.n == 0 || B_in.n == 0) {
        if (ev_start) cudaEventRecord(ev_start, s);
        if (ev_stop) cudaEventRecord(ev_stop, s);
        return;
    }
    // all_pairs is symmetric: the pair set of (A, B) is that of (B, A) with the id columns exchanged.  The per-row
    // work (window, cell look-ups) is paid by the catalogue whose rows drive the lanes, while staging grows with the
    // scanned rows per driving row; measured on config 3 (ratio 2) the two directions tie, so the roles are
    // exchanged only when B is much the smaller catalogue.
    const bool same = (match_flags & kMatchSameGrid) != 0;
    const bool swap = !same && !ex && mode == HLC2_ALL_PAIRS && (size_t)B_in.n * 3 < (size_t)A_in.n;
    const IndexView& A = swap ? B_in : A_in;
    const IndexView& B = swap ? A_in : B_in;
    if (swap) std::swap(out_ida, out_idb);
    MatchArgs p;
    long double r_rad = (long double)radius_arcsec * (3.141592653589793238462643383279502884L / 648000.0L);
    long double hs = sinl(0.5L * r_rad);
    p.thr2 = (double)(4.0L * hs * hs);
    p.r_deg = radius_arcsec / 3600.0;
    p.pad_dec = p.r_deg + kEpsDecDeg;
    p.sin_r_up = (float)((double)sinl(r_rad) * (1.0 + 1e-5));
    p.out_ida = out_ida; p.out_idb = out_idb; p.out_sep = out_sep; p.capacity = capacity; p.count = d_count;
    p.jobs = nullptr; p.pool_count = nullptr; p.tile_cap = 0; p.pool_cap = 0;
    p.self_mode = ex ? ex->self_mode : 0;
    p.ea2 = nullptr; p.eb2 = nullptr; p.kfac2rad = 0.0;
    if (ex && ex->k_factor > 0.0) {
        p.ea2 = A.err2; p.eb2 = B.err2;
        const long double f = (long double)ex->k_factor * (3.141592653589793238462643383279502884L / 648000.0L);
        p.kfac2rad = (double)(f * f);
    }
    if (p.eb2 || (p.self_mode && !same)) {     // per-record radii, or a self-match off the same-grid kernel: the general per-lane path
        launch_match_all_general(A, B, p, mode, s, ev_start, ev_stop);
        return;
    }
    if (same) {         // both indices on one grid: no planner, no job records (hlc2_match_same.cu)
        launch_match_same(A, B, p, mode, d_temp, s, ev_start, ev_stop);
        return;
    }
    const size_t tiles = A.tile_cap;
    // scratch: 256-byte header (pool counter), then the tiles' first jobs, then the pool of chained jobs
    p.pool_count = reinterpret_cast<uint32_t*>(d_temp);
    p.jobs = reinterpret_cast<Job*>(reinterpret_cast<char*>(d_temp) + 256);
    p.tile_cap = (uint32_t)tiles; p.pool_cap = (uint32_t)pool_cap_of(tiles);
    cudaMemsetAsync(p.pool_count, 0, sizeof(uint32_t), s);
    const int m = mode == HLC2_NEAREST ? 1 : 0;
    const void* kern = m == 0 ? (const void*)k_match<HLC2_ALL_PAIRS> : (const void*)k_match<HLC2_NEAREST>;
    static int per_sm_dev[kMaxDevices][2] = {};        // resident CTAs per SM; the smem opt-in is per device
    int* per_sm = per_sm_dev[current_device()];
    const size_t smem = sizeof(MatchSmem);
    if (!per_sm[m]) {
        int v = 0;
        cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        cudaOccupancyMaxActiveBlocksPerMultiprocessor(&v, kern, kMatchThreads, smem);
        per_sm[m] = v > 0 ? v : 1;
    }
    const unsigned pblocks = (unsigned)std::min<size_t>((tiles + 127) / 128, (size_t)sm_count() * 8);
    k_plan<<<pblocks, 128, 0, s>>>(A, B, p);
    count_launch();
    // persistent grid: SM count x resident CTAs, never more CTAs than tiles
    const unsigned blocks = (unsigned)std::max<size_t>(1, std::min<size_t>(tiles, (size_t)sm_count() * per_sm[m]));
    if (ev_start) cudaEventRecord(ev_start, s);          // the caller's events bracket k_match alone (hlc2_crossmatch_events)
    void* kargs[3] = {(void*)&A, (void*)&B, (void*)&p};
    cudaLaunchKernel(kern, dim3(blocks), dim3(kMatchThreads), kargs, smem, s);
    count_launch();
    if (ev_stop) cudaEventRecord(ev_stop, s);
}

}  // namespace hlc2
