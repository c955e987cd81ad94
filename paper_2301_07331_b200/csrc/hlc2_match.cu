// hlc2_match.cu -- the match kernels (NS (b)).
//
// Work unit = one A tile: up to kTile consecutive cell-sorted A rows of one A zone (the role of the paper's
// calculation blocks).  Two kernels:
//
//   k_plan   one thread per A tile.  From the tile's own cell bounds (exact: zone edges and RA-cell edges of
//            A's grid) it derives the window on B's grid that any row of the tile can reach:
//              dec  [dec_lo - r, dec_hi + r]                          -> <= kSegs consecutive zones of B's grid
//              RA   [ra_lo - W, ra_hi + W], W = asin(sin r / cos dec*) -> ONE contiguous cell range per zone
//            (the cells the quad-direction strategy probes, L122-169, plus the diagonal neighbours and the
//            1/cos(dec) widening it omits, so no pair is lost: the "No Index" result, L344) and writes a job:
//            per zone the B row range and the slice of cell_start that covers it.  Tiles whose window wraps
//            through RA = 0/360, touches a polar ring, needs more zones or more rows than a stage holds are
//            marked DIRECT.
//   k_match  persistent CTAs of kCW consumer warps + 1 producer warp, kStages-deep mbarrier ring.  The producer
//            warp turns each job into 1-D bulk copies (cp.async.bulk, the TMA engine): the A tile (x, y, z,
//            pos, id) and, per zone segment, B's x, y, z, id rows and the cell_start slice -- all contiguous
//            because keys are zone-major / RA-minor.  Consumers: one lane per A row (the paper's
//            thread-per-A-record hierarchy, L271-276).  A lane locates its own cells from the fp32 (ra, dec)
//            estimate padded by a rigorous error bound, clips them to the job's range (the job covers every
//            cell a row of the tile needs, so clipping never loses one), reads its row range from the staged
//            cell_start slice and tests the staged rows: chord^2 <= 4 sin^2(r/2), all fp64 from shared memory.
//            Hits (the role of d_out_dis, L282) are compacted by ballot + popcount into a per-warp queue of
//            (idA, idB, chord^2) and flushed 64 at a time: one global atomic, coalesced stores, sep computed
//            on full warps.  DIRECT tiles run the general per-lane path from global memory (any number of
//            zones, RA wrap, polar rings).
//
// Decisions are fp64; the fp32 estimate only ever selects a superset of cells.
#include <math.h>

#include "hlc2_grid.cuh"

namespace hlc2 {

constexpr int kCW = kTile / 32;              // consumer warps (one lane per A row of the tile)
constexpr int kMatchThreads = kTile + 32;    // + the producer warp
constexpr int kStages = 3;
constexpr int kSegs = 4;                     // zone segments per job
constexpr int kBCap = 448;                   // staged B rows per job, all segments, after 16-byte alignment
constexpr int kCsCap = 512;                  // staged cell_start entries per job, after alignment
constexpr int kQCap = 96;                    // rows in a warp's hit queue
constexpr int kQFlush = 64;                  // flushed as soon as this many are queued (<= 63 + 32 < kQCap)
constexpr int kAPad = kTile + 2;             // A tile rows after alignment to 16 bytes
constexpr double kRad2Arcsec = 206264.80624709636;   // 648000 / pi
constexpr unsigned kFull = 0xffffffffu;

// padding of the fp32 position estimate (degrees); derivation in DESIGN.md section 5 (~3x the worst case)
constexpr double kEpsRaDeg = 2.5e-4;
constexpr double kEpsDecDeg = 1.5e-4;
constexpr double kTinyDeg = 1e-9;            // fp64 slop on cell / zone edges in the planner

constexpr uint32_t kJobDirect = 1u << 8;

// 96-byte job record (24 words), one per A tile, written by k_plan
struct JobSeg { uint32_t row_lo, cs_lo; int32_t k_lo, n_ra; uint32_t nk_nrows; };   // n_k | n_rows << 16
struct Job { uint32_t a_first, a_count; int32_t z_lo; uint32_t flags; JobSeg seg[kSegs]; };
static_assert(sizeof(Job) == 96, "the producer reads a job as 24 words");

struct MatchArgs {
    double thr2;          // 4 sin^2(r/2)
    double pad_dec;       // r in degrees + kEpsDecDeg
    double r_deg;
    float sin_r_up;       // sin(r) * (1 + 1e-5)
    int64_t* out_ida; int64_t* out_idb; double* out_sep;
    unsigned long long capacity;
    unsigned long long* count;
    const Job* jobs;
};

struct SegDesc { double n_d; int32_t k_lo, k_hi, cdelta; uint32_t rdelta, n_rows, pad; };
struct StageDesc { uint32_t a_first, a_count, a_off, flags; int32_t nseg, z_lo; uint32_t pad[2]; SegDesc seg[kSegs]; };

struct __align__(16) Stage {
    double ax[kAPad], ay[kAPad], az[kAPad];
    float2 apos[kAPad];
    long long aid[kAPad];
    double bx[kBCap + 2], by[kBCap + 2], bz[kBCap + 2];     // slot kBCap: a point no chord test can reach
    long long bid[kBCap];
    uint32_t cs[kCsCap];
    StageDesc d;
};
struct WarpQueue { long long ida[kQCap], idb[kQCap]; double c2[kQCap]; };
struct __align__(16) MatchSmem {
    Stage st[kStages];
    WarpQueue q[kCW];
    unsigned long long full[kStages], empty[kStages];
};
static_assert((kAPad * 8) % 16 == 0 && (kBCap * 8) % 16 == 0 && (kCsCap * 4) % 16 == 0, "bulk copies need 16-byte pieces");
static_assert(sizeof(Stage) % 16 == 0, "stages stay 16-byte aligned");

// ---- mbarrier / bulk-copy primitives (sm_90+ PTX) ----------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned long long* b, unsigned count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(b)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(unsigned long long* b) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(b)) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(unsigned long long* b, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(b)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long* b, unsigned parity) {
    const uint32_t a = smem_u32(b);
    unsigned done;
    do {
        asm volatile("{\n .reg .pred p;\n mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n selp.u32 %0, 1, 0, p;\n}"
                     : "=r"(done) : "r"(a), "r"(parity) : "memory");
    } while (!done);
}
// global -> shared bulk copy, completion counted in bytes on an mbarrier; 16-byte aligned src, dst and size
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, unsigned bytes, unsigned long long* b) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(b)) : "memory");
}

// sep = 2 asin(chord / 2) in arcsec.  Below 2^-10 rad (403 arcsec) the series h + h^3/6 + 3 h^5/40 is exact to
// 4e-20 relative; above it the library asin.
__device__ __forceinline__ double sep_from_chord2(double c2) {
    const double h = 0.5 * sqrt(c2);
    double a;
    if (h < 0.0009765625) { const double t = h * h; a = fma(h * t, fma(t, 0.075, 1.0 / 6.0), h); }
    else a = asin(fmin(1.0, h));
    return a * (2.0 * kRad2Arcsec);
}

// ------------------------------------------------------------------------------------------------------
// k_plan: one job per A tile
// ------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(128)
k_plan(const __grid_constant__ IndexView A, const __grid_constant__ IndexView B, const __grid_constant__ MatchArgs p,
       Job* __restrict__ jobs) {
    const uint32_t nt = __ldg(A.n_tiles);
    const GridView& ga = A.g;
    const GridView& gb = B.g;
    for (uint32_t t = blockIdx.x * 128 + threadIdx.x; t < nt; t += gridDim.x * 128) {
        const uint4 t0 = __ldg(reinterpret_cast<const uint4*>(A.tiles + t));        // first, count, zone, k_first
        const uint4 t1 = __ldg(reinterpret_cast<const uint4*>(A.tiles + t) + 1);    // k_last
        uint32_t w[24];
#pragma unroll
        for (int i = 0; i < 24; ++i) w[i] = 0;
        w[0] = t0.x; w[1] = t0.y;
        const int za = (int)t0.z;
        // declination and RA bounds of the tile's rows: the edges of its zone and of its first / last cell in
        // A's grid (rows were filed by the same floor expressions; kTinyDeg covers their rounding)
        const double dlo = za == 0 ? ga.dec_min : fmax(ga.dec_min, ga.dec_lo + (double)za * ga.h - kTinyDeg);
        const double dhi = za == ga.n_zones - 1 ? ga.dec_max : fmin(ga.dec_max, ga.dec_lo + (double)(za + 1) * ga.h + kTinyDeg);
        const double qlo = dlo - p.r_deg - kTinyDeg, qhi = dhi + p.r_deg + kTinyDeg;
        bool empty = qhi < gb.dec_min || qlo > gb.dec_max || t0.y == 0;
        bool direct = false;
        if (!empty) {
            const int zb0 = zone_of(gb, qlo), zb1 = zone_of(gb, qhi);
            const int nseg = zb1 - zb0 + 1;
            if (nseg > kSegs) direct = true;
            const double cw = ga.span / (double)__ldg(ga.n_ra + za);
            const double ua_lo = (double)t0.w * cw - kTinyDeg, ua_hi = (double)(t1.x + 1u) * cw + kTinyDeg;
            // RA half-window of the most poleward row: sin(dRA) = sin r / cos dec; the rows bound asin(s) by
            // 1.011 s (s < 0.25) from their own fp32 cos dec; the extra 1.001 and kEpsRaDeg keep W above all of them
            const double dabs = fmin(90.0, fmax(fabs(dlo), fabs(dhi)));
            const double s = (double)p.sin_r_up / fmax(cos(dabs * 0.017453292519943295), 1e-300);
            if (!(s < 0.2)) direct = true;
            const double W = s * (1.011 * 57.29577951308232 * 1.001) + 2.0 * kEpsRaDeg;
            double ub = (ga.ra0 + ua_lo) - gb.ra0;
            ub -= 360.0 * floor(ub * (1.0 / 360.0));
            if (!(ub >= 0.0 && ub < 360.0)) ub = 0.0;
            const double lo = ub - W, hi = ub + (ua_hi - ua_lo) + W;
            // a window that comes within the estimate's error of u = 0 / 360 could see a row's estimate wrap
            if (!(lo >= 2.0 * kEpsRaDeg) || !(hi + 2.0 * kEpsRaDeg < 360.0)) direct = true;
            if (!direct && lo > gb.span + 2.0 * kEpsRaDeg) empty = true;      // beyond B's RA box
            if (!direct && !empty) {
                uint32_t rows_tot = 0, cs_tot = 0;
                w[2] = (uint32_t)zb0;
#pragma unroll
                for (int sg = 0; sg < kSegs; ++sg) {
                    if (sg < nseg) {
                        const int z = zb0 + sg, n = __ldg(gb.n_ra + z);
                        const uint32_t cb = __ldg(gb.cell_base + z);
                        const int k0 = cell_of_u(gb, lo, n), k1 = cell_of_u(gb, hi, n);
                        const uint32_t r0 = __ldg(B.cell_start + cb + (uint32_t)k0), r1 = __ldg(B.cell_start + cb + (uint32_t)k1 + 1u);
                        const uint32_t nk = (uint32_t)(k1 - k0 + 1), nr = r1 - r0, c0 = cb + (uint32_t)k0;
                        if (nr) {
                            rows_tot += ((r1 + 1u) & ~1u) - (r0 & ~1u);
                            cs_tot += ((c0 + nk + 1u + 3u) & ~3u) - (c0 & ~3u);
                        }
                        if (nk > 0xFFFFu || nr > 0xFFFFu) direct = true;
                        w[4 + 5 * sg] = r0; w[5 + 5 * sg] = c0; w[6 + 5 * sg] = (uint32_t)k0; w[7 + 5 * sg] = (uint32_t)n;
                        w[8 + 5 * sg] = (nk & 0xFFFFu) | (nr << 16);
                    }
                }
                if (rows_tot > (uint32_t)kBCap || cs_tot > (uint32_t)kCsCap) direct = true;
                if (rows_tot == 0) empty = true;
                w[3] = (uint32_t)nseg;
            }
        }
        if (direct || empty) {
#pragma unroll
            for (int i = 2; i < 24; ++i) w[i] = 0;
            if (direct && !empty) w[3] = kJobDirect;
        }
        uint4* o = reinterpret_cast<uint4*>(jobs + t);
#pragma unroll
        for (int i = 0; i < 6; ++i) o[i] = make_uint4(w[4 * i], w[4 * i + 1], w[4 * i + 2], w[4 * i + 3]);
    }
}

// ------------------------------------------------------------------------------------------------------
// the general per-lane path (DIRECT tiles): any number of zones, RA wrap, polar ring, window partly outside
// B's box.  Reads B through global memory / L2.
// ------------------------------------------------------------------------------------------------------
struct Best { double c2; long long idb; bool has; };

// one row straight to the output; lanes that arrive together share one global atomic
__device__ __forceinline__ void emit_direct(const MatchArgs& p, long long ida, long long idb, double c2) {
    const unsigned m = __activemask();
    const int lane = threadIdx.x & 31, leader = __ffs(m) - 1;
    unsigned long long base = 0;
    if (lane == leader) base = atomicAdd(p.count, (unsigned long long)__popc(m));
    base = __shfl_sync(m, base, leader);
    const unsigned long long o = base + __popc(m & ((1u << lane) - 1u));
    if (o < p.capacity) { p.out_ida[o] = ida; p.out_idb[o] = idb; p.out_sep[o] = sep_from_chord2(c2); }
}

template <int MODE>
__device__ __forceinline__ void scan_global(const IndexView& B, const MatchArgs& p, long long ida,
                                            double ax, double ay, double az, uint32_t j0, uint32_t j1, Best& h) {
    for (uint32_t j = j0; j < j1; ++j) {
        const double dx = ax - __ldg(B.x + j), dy = ay - __ldg(B.y + j), dz = az - __ldg(B.z + j);
        const double c2 = fma(dx, dx, fma(dy, dy, dz * dz));
        if (c2 <= p.thr2) {
            const long long idb = __ldg(B.id + j);
            if (MODE == HLC2_ALL_PAIRS) emit_direct(p, ida, idb, c2);
            else if (!h.has || c2 < h.c2 || (c2 == h.c2 && idb < h.idb)) { h.has = true; h.idb = idb; h.c2 = c2; }
        }
    }
}

template <int MODE>
__device__ __noinline__ void scan_general(const IndexView& B, const MatchArgs& p, long long ida,
                                          double ax, double ay, double az, float2 pf, Best& h) {
    const GridView& g = B.g;
    const double dlo = (double)pf.y - p.pad_dec, dhi = (double)pf.y + p.pad_dec;
    if (dhi < g.dec_min || dlo > g.dec_max) return;
    const float fx = (float)ax, fy = (float)ay;
    const float s = p.sin_r_up * rsqrtf(fx * fx + fy * fy);               // sin(dRA_max) = sin r / cos dec
    const bool ring = !(s < 0.25f);
    const double w = ring ? 360.0 : (double)(s * (1.011f * 57.29577951f)) + kEpsRaDeg;   // asin(s) <= 1.011 s below 0.25
    const double u = box_u(g, (double)pf.x);
    const double ulo = u - w, uhi = u + w;
    const int z0 = zone_of(g, dlo), z1 = zone_of(g, dhi);
    for (int z = z0; z <= z1; ++z) {
        const int n = __ldg(g.n_ra + z);
        const uint32_t base = __ldg(g.cell_base + z);
        int k0 = 0, k1 = n - 1, k2 = 0, k3 = -1;      // [k0,k1] and optional [k2,k3]
        if (!(ring || w >= 180.0)) {
            const bool va = ulo <= g.span;
            k0 = cell_of_u(g, fmax(ulo, 0.0), n); k1 = cell_of_u(g, fmin(uhi, g.span), n);
            bool vx = false;
            if (ulo < 0.0) { if (ulo + 360.0 <= g.span) { vx = true; k2 = cell_of_u(g, ulo + 360.0, n); k3 = n - 1; } }
            else if (uhi >= 360.0) { vx = true; k2 = 0; k3 = cell_of_u(g, fmin(uhi - 360.0, g.span), n); }
            if (va && vx && !(k3 < k0 || k2 > k1)) { k0 = 0; k1 = n - 1; vx = false; }
            if (!va) { if (!vx) continue; k0 = k2; k1 = k3; vx = false; }
            if (!vx) k3 = k2 - 1;
        }
        scan_global<MODE>(B, p, ida, ax, ay, az, __ldg(B.cell_start + base + k0), __ldg(B.cell_start + base + k1 + 1), h);
        if (k3 >= k2)
            scan_global<MODE>(B, p, ida, ax, ay, az, __ldg(B.cell_start + base + k2), __ldg(B.cell_start + base + k3 + 1), h);
    }
}

// ------------------------------------------------------------------------------------------------------
// hit queue of one consumer warp
// ------------------------------------------------------------------------------------------------------
// write queue rows [first, first + cnt) to the output: one global atomic, coalesced stores
__device__ __forceinline__ void flush_rows(const MatchArgs& p, const WarpQueue& q, unsigned first, unsigned cnt, int lane) {
    unsigned long long base = 0;
    if (lane == 0) base = atomicAdd(p.count, (unsigned long long)cnt);
    base = __shfl_sync(kFull, base, 0);
    for (unsigned k = lane; k < cnt; k += 32) {
        const unsigned long long o = base + k;
        if (o < p.capacity) {
            p.out_ida[o] = q.ida[first + k]; p.out_idb[o] = q.idb[first + k];
            p.out_sep[o] = sep_from_chord2(q.c2[first + k]);
        }
    }
}

// append the lanes with `hit`; flush the top kQFlush rows once that many are queued.  qn is warp-uniform.
__device__ __forceinline__ void push_hits(const MatchArgs& p, WarpQueue& q, unsigned& qn, bool hit,
                                          long long ida, long long idb, double c2, int lane) {
    const unsigned m = __ballot_sync(kFull, hit);
    if (m == 0) return;
    if (hit) {
        const unsigned k = qn + __popc(m & ((1u << lane) - 1u));
        q.ida[k] = ida; q.idb[k] = idb; q.c2[k] = c2;
    }
    qn += __popc(m);
    if (qn >= (unsigned)kQFlush) {
        __syncwarp();
        qn -= kQFlush;
        flush_rows(p, q, qn, kQFlush, lane);
        __syncwarp();
    }
}

// ------------------------------------------------------------------------------------------------------
// staged scan: every lane tests its rows [p0, p1) of the stage's B arrays; the trip count is the warp's
// maximum so that hits can be compacted with one ballot per step
// ------------------------------------------------------------------------------------------------------
template <int MODE>
__device__ __forceinline__ void scan_staged(const Stage& st, const MatchArgs& p, WarpQueue& q, unsigned& qn,
                                            long long ida, double ax, double ay, double az,
                                            unsigned p0, unsigned p1, Best& best, int lane) {
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
            push_hits(p, q, qn, h0, ida, h0 ? st.bid[j0] : 0ll, c20, lane);
            push_hits(p, q, qn, h1, ida, h1 ? st.bid[j1] : 0ll, c21, lane);
        } else {
            if (h0) {
                const long long idb = st.bid[j0];
                if (!best.has || c20 < best.c2 || (c20 == best.c2 && idb < best.idb)) { best.has = true; best.idb = idb; best.c2 = c20; }
            }
            if (h1) {
                const long long idb = st.bid[j1];
                if (!best.has || c21 < best.c2 || (c21 == best.c2 && idb < best.idb)) { best.has = true; best.idb = idb; best.c2 = c21; }
            }
        }
    }
}

// ------------------------------------------------------------------------------------------------------
// k_match
// ------------------------------------------------------------------------------------------------------
template <int MODE>
__global__ void __launch_bounds__(kMatchThreads, 3)
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
    const uint32_t nt = __ldg(A.n_tiles);

    if (warp == kCW) {
        // ---------------- producer warp: job -> bulk copies ----------------
        const uint32_t* jw = reinterpret_cast<const uint32_t*>(p.jobs);
        uint32_t t = blockIdx.x;
        uint32_t wcur = (t < nt && lane < 24) ? __ldg(jw + (size_t)t * 24 + lane) : 0u;
        for (uint32_t it = 0; t < nt; ++it, t += gridDim.x) {
            const uint32_t tn = t + gridDim.x;
            const uint32_t wnext = (tn < nt && lane < 24) ? __ldg(jw + (size_t)tn * 24 + lane) : 0u;
            const int s = (int)(it % kStages);
            const unsigned ph = (it / kStages) & 1u;
            Stage& st = sm.st[s];
            const uint32_t a_first = __shfl_sync(kFull, wcur, 0), a_count = __shfl_sync(kFull, wcur, 1);
            const uint32_t z_lo = __shfl_sync(kFull, wcur, 2), flags = __shfl_sync(kFull, wcur, 3);
            const int nseg = (int)(flags & 0xFFu);
            const int sb = 4 + 5 * min(lane, kSegs - 1);
            const uint32_t row_lo = __shfl_sync(kFull, wcur, sb), cs_lo = __shfl_sync(kFull, wcur, sb + 1);
            const uint32_t k_lo = __shfl_sync(kFull, wcur, sb + 2), n_ra = __shfl_sync(kFull, wcur, sb + 3);
            const uint32_t nkr = __shfl_sync(kFull, wcur, sb + 4);
            const uint32_t nk = nkr & 0xFFFFu, nr = nkr >> 16;
            const bool segact = lane < nseg && nr != 0;
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
            const uint32_t bytes = a_ld * 40u + rtot * 32u + ctot * 4u;

            mbar_wait(&sm.empty[s], ph ^ 1u);
            if (lane == 0) {
                st.d.a_first = a_first; st.d.a_count = a_count; st.d.a_off = a_first - a_al; st.d.flags = flags;
                st.d.nseg = nseg; st.d.z_lo = (int32_t)z_lo;
            }
            if (lane < kSegs) {
                SegDesc& e = st.d.seg[lane];
                e.n_d = (double)(int32_t)n_ra; e.k_lo = (int32_t)k_lo; e.k_hi = (int32_t)(k_lo + nk) - 1;
                e.cdelta = (int32_t)((cs_lo - k_lo) - cs_al + coff); e.rdelta = roff - row_al; e.n_rows = segact ? nr : 0u;
            }
            __syncwarp();
            if (lane == 0) { if (bytes) mbar_arrive_expect_tx(&sm.full[s], bytes); else mbar_arrive(&sm.full[s]); }
            if (segact) {
                bulk_g2s(st.bx + roff, B.x + row_al, n_ld * 8u, &sm.full[s]);
                bulk_g2s(st.by + roff, B.y + row_al, n_ld * 8u, &sm.full[s]);
                bulk_g2s(st.bz + roff, B.z + row_al, n_ld * 8u, &sm.full[s]);
                bulk_g2s(st.bid + roff, B.id + row_al, n_ld * 8u, &sm.full[s]);
                bulk_g2s(st.cs + coff, B.cell_start + cs_al, c_ld * 4u, &sm.full[s]);
            }
            if (a_ld && lane >= 8 && lane < 13) {
                const int k = lane - 8;
                const void* src = k == 0 ? (const void*)(A.x + a_al) : k == 1 ? (const void*)(A.y + a_al) : k == 2 ? (const void*)(A.z + a_al)
                                : k == 3 ? (const void*)(A.pos + a_al) : (const void*)(A.id + a_al);
                void* dst = k == 0 ? (void*)st.ax : k == 1 ? (void*)st.ay : k == 2 ? (void*)st.az : k == 3 ? (void*)st.apos : (void*)st.aid;
                bulk_g2s(dst, src, a_ld * 8u, &sm.full[s]);
            }
            wcur = wnext;
        }
        return;
    }

    // ---------------- consumer warps: one lane per A row of the tile ----------------
    const GridView& g = B.g;
    WarpQueue& q = sm.q[warp];
    unsigned qn = 0;
    uint32_t it = 0;
    for (uint32_t t = blockIdx.x; t < nt; t += gridDim.x, ++it) {
        const int s = (int)(it % kStages);
        const unsigned ph = (it / kStages) & 1u;
        mbar_wait(&sm.full[s], ph);
        const Stage& st = sm.st[s];
        const StageDesc& d = st.d;
        const uint32_t flags = d.flags, a_count = d.a_count;
        const int nseg = d.nseg;
        if ((nseg != 0 || (flags & kJobDirect)) && (uint32_t)(warp * 32) < a_count) {
            const bool act = threadIdx.x < a_count;
            const unsigned ra = act ? threadIdx.x + d.a_off : d.a_off;
            const double ax = st.ax[ra], ay = st.ay[ra], az = st.az[ra];
            const float2 pf = st.apos[ra];
            const long long ida = st.aid[ra];
            Best best; best.has = false; best.c2 = 0.0; best.idb = 0;
            if (flags & kJobDirect) {
                if (act) scan_general<MODE>(B, p, ida, ax, ay, az, pf, best);
                __syncwarp();
            } else {
                const double dlo = (double)pf.y - p.pad_dec, dhi = (double)pf.y + p.pad_dec;
                const int zlo = zone_of(g, dlo) - d.z_lo, zhi = zone_of(g, dhi) - d.z_lo;
                const float fx = (float)ax, fy = (float)ay;
                const float sn = p.sin_r_up * rsqrtf(fx * fx + fy * fy);
                const double w = (double)(sn * (1.011f * 57.29577951f)) + kEpsRaDeg;
                const double u = box_u(g, (double)pf.x);
                const double vlo = (u - w) * g.inv_span, vhi = (u + w) * g.inv_span;
                unsigned p0 = 0, p1 = 0, s0 = 0, s1 = 0;      // a lane's first and (zone-spanning rows) second range
                for (int sg = 0; sg < nseg; ++sg) {
                    const SegDesc& e = d.seg[sg];
                    if (e.n_rows == 0) continue;
                    int k0 = __double2int_rd(vlo * e.n_d), k1 = __double2int_rd(vhi * e.n_d);
                    k0 = min(max(k0, e.k_lo), e.k_hi); k1 = min(max(k1, e.k_lo), e.k_hi);
                    const unsigned q0 = st.cs[k0 + e.cdelta] + e.rdelta, q1 = st.cs[k1 + 1 + e.cdelta] + e.rdelta;
                    const bool has = act && sg >= zlo && sg <= zhi && q1 > q0;
                    if (sg >= 2 && __any_sync(kFull, has && p1 > p0 && s1 > s0)) {      // a third range: drain first
                        scan_staged<MODE>(st, p, q, qn, ida, ax, ay, az, p0, p1, best, lane);
                        scan_staged<MODE>(st, p, q, qn, ida, ax, ay, az, s0, s1, best, lane);
                        p0 = p1 = s0 = s1 = 0;
                    }
                    if (has) { if (p1 == p0) { p0 = q0; p1 = q1; } else { s0 = q0; s1 = q1; } }
                }
                scan_staged<MODE>(st, p, q, qn, ida, ax, ay, az, p0, p1, best, lane);
                if (__any_sync(kFull, s1 > s0)) scan_staged<MODE>(st, p, q, qn, ida, ax, ay, az, s0, s1, best, lane);
            }
            if (MODE == HLC2_NEAREST) push_hits(p, q, qn, best.has, ida, best.idb, best.c2, lane);
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(&sm.empty[s]);
    }
    __syncwarp();
    if (qn) flush_rows(p, q, 0, qn, lane);
}

size_t match_temp_bytes(const IndexView& A, const IndexView&) { return ((size_t)A.tile_cap + 1) * sizeof(Job); }

void launch_match(const IndexView& A, const IndexView& B, double radius_arcsec, int mode,
                  int64_t* out_ida, int64_t* out_idb, double* out_sep, unsigned long long capacity,
                  unsigned long long* d_count, void* d_temp, cudaStream_t s) {
    if (A.n == 0 || B.n == 0) return;
    MatchArgs p;
    long double r_rad = (long double)radius_arcsec * (3.141592653589793238462643383279502884L / 648000.0L);
    long double hs = sinl(0.5L * r_rad);
    p.thr2 = (double)(4.0L * hs * hs);
    p.r_deg = radius_arcsec / 3600.0;
    p.pad_dec = p.r_deg + kEpsDecDeg;
    p.sin_r_up = (float)((double)sinl(r_rad) * (1.0 + 1e-5));
    p.out_ida = out_ida; p.out_idb = out_idb; p.out_sep = out_sep; p.capacity = capacity; p.count = d_count;
    Job* jobs = reinterpret_cast<Job*>(d_temp);
    p.jobs = jobs;
    const int m = mode == HLC2_NEAREST ? 1 : 0;
    static int per_sm[2] = {0, 0};
    const size_t smem = sizeof(MatchSmem);
    if (!per_sm[m]) {
        int v = 0;
        if (m) {
            cudaFuncSetAttribute(k_match<HLC2_NEAREST>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
            cudaOccupancyMaxActiveBlocksPerMultiprocessor(&v, k_match<HLC2_NEAREST>, kMatchThreads, smem);
        } else {
            cudaFuncSetAttribute(k_match<HLC2_ALL_PAIRS>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
            cudaOccupancyMaxActiveBlocksPerMultiprocessor(&v, k_match<HLC2_ALL_PAIRS>, kMatchThreads, smem);
        }
        per_sm[m] = v > 0 ? v : 1;
    }
    const size_t tiles = A.tile_cap;
    const unsigned pblocks = (unsigned)std::min<size_t>((tiles + 127) / 128, (size_t)sm_count() * 8);
    k_plan<<<pblocks, 128, 0, s>>>(A, B, p, jobs);
    count_launch();
    // persistent grid: SM count x resident CTAs, never more CTAs than tiles
    const unsigned blocks = (unsigned)std::max<size_t>(1, std::min<size_t>(tiles, (size_t)sm_count() * per_sm[m]));
    if (m) k_match<HLC2_NEAREST><<<blocks, kMatchThreads, smem, s>>>(A, B, p);
    else   k_match<HLC2_ALL_PAIRS><<<blocks, kMatchThreads, smem, s>>>(A, B, p);
    count_launch();
}

}  // namespace hlc2
