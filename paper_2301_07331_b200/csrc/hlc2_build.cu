// hlc2_build.cu -- index-build kernels (NS (a)).
//
//   k_stats        (a1) validity, dec extent, coarse RA occupancy            16 B/source read
//   k_keys_pack    (a1) cell key + window flags; packs a 32-byte AoS record {ra, dec, -, id} in input order and
//                       accumulates the digit histograms of every radix pass  24 B read, 36 B written
//   k_digit_scan   (a2) exclusive scan of the per-pass digit histograms (one CTA)
//   k_onesweep     (a2) one LSD radix pass over (key, row): chained-scan ("decoupled look-back") of tile digit
//                       counts, ranks by owner tags and votes, smem reorder so that every digit run is written
//                       coalesced                                              8 B read, 8 B written per pass
//   k_gather       (a3) one 32-byte sector per source (the packed record) -> unit vector -> cell-sorted SoA x,y,z,id
//   k_cell_fill    (a4) run boundaries of the sorted keys -> cell_start[] (also for empty cells), long empty
//                       runs handed to k_cell_fill_big
//   k_zone_tiles, k_tile_desc (a4) tile descriptors: runs of <= kTile consecutive sources inside one zone
//
// All of them are streaming passes; persistent grids are multiples of the SM count, the gather runs one row per thread.
#include <string.h>
#include <algorithm>

#include "hlc2_grid.cuh"

namespace hlc2 {

// per-device caches (a process may drive several devices); benign race: every thread computes the same value
int current_device() {
    int dev = 0; cudaGetDevice(&dev);
    return dev >= 0 && dev < kMaxDevices ? dev : 0;
}
int sm_count() {
    static int cache[kMaxDevices] = {};
    const int dev = current_device();
    if (!cache[dev]) {
        int v = 0;
        cudaDeviceGetAttribute(&v, cudaDevAttrMultiProcessorCount, dev);
        cache[dev] = v > 0 ? v : 148;
    }
    return cache[dev];
}

// ------------------------------------------------------------------------------------------
// (a1) extent statistics: validity, dec range, coarse RA occupancy
// ------------------------------------------------------------------------------------------
constexpr int kStatsThreads = 512;

__global__ void __launch_bounds__(kStatsThreads)
k_stats(const double* __restrict__ ra, const double* __restrict__ dec, uint32_t n, Stats* __restrict__ st) {
    __shared__ uint32_t hist[kRaBins];
    __shared__ unsigned long long s_min[kStatsThreads / 32], s_max[kStatsThreads / 32];
    for (int i = threadIdx.x; i < kRaBins; i += kStatsThreads) hist[i] = 0;
    __syncthreads();
    unsigned long long dmin = ~0ull, dmax = 0ull, bad_row = ~0ull; unsigned nbad = 0;
    for (size_t i = (size_t)blockIdx.x * kStatsThreads + threadIdx.x; i < n; i += (size_t)gridDim.x * kStatsThreads) {
        double a = __ldg(ra + i), d = __ldg(dec + i);
        if (coord_ok(a, d)) {
            unsigned long long b = f64_order_bits(d);
            dmin = min(dmin, b); dmax = max(dmax, b);
            int bin = min(kRaBins - 1, (int)(norm_ra(a) * (1.0 / kRaBinDeg)));
            atomicAdd(&hist[bin], 1u);
        } else {
            ++nbad; bad_row = min(bad_row, (unsigned long long)i);
        }
    }
    for (int o = 16; o; o >>= 1) {
        dmin = min(dmin, __shfl_xor_sync(0xffffffffu, dmin, o));
        dmax = max(dmax, __shfl_xor_sync(0xffffffffu, dmax, o));
    }
    if ((threadIdx.x & 31) == 0) { s_min[threadIdx.x >> 5] = dmin; s_max[threadIdx.x >> 5] = dmax; }
    if (nbad) { atomicAdd(&st->n_bad, (unsigned long long)nbad); atomicMin(&st->first_bad_row, bad_row); }
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int w = 1; w < kStatsThreads / 32; ++w) { dmin = min(dmin, s_min[w]); dmax = max(dmax, s_max[w]); }
        if (dmin != ~0ull) { atomicMin(&st->dec_min_bits, dmin); atomicMax(&st->dec_max_bits, dmax); }
    }
    for (int i = threadIdx.x; i < kRaBins; i += kStatsThreads)
        if (hist[i]) atomicAdd(&st->ra_hist[i], hist[i]);
}

__global__ void k_stats_init(Stats* st) {
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < kRaBins) st->ra_hist[i] = 0;
    if (i == 0) { st->dec_min_bits = ~0ull; st->dec_max_bits = 0ull; st->first_bad_row = ~0ull; st->n_bad = 0; }
}

void launch_stats_init(Stats* d_stats, cudaStream_t s) { k_stats_init<<<(kRaBins + 255) / 256, 256, 0, s>>>(d_stats); count_launch(); }

void launch_stats(const double* ra, const double* dec, uint32_t n, Stats* d_stats, cudaStream_t s) {
    launch_stats_init(d_stats, s);
    if (n == 0) return;
    int blocks = (int)std::min<size_t>(((size_t)n + kStatsThreads - 1) / kStatsThreads, (size_t)sm_count() * 4);
    k_stats<<<blocks, kStatsThreads, 0, s>>>(ra, dec, n, d_stats); count_launch();
}

// ------------------------------------------------------------------------------------------
// (a1) cell key + unit vector + packed record + digit histograms
// Accuracy of the unit vector: RA is reduced to |t| <= 45 deg in the degree domain (t = ra - 90 rint(ra/90) is
// exact), Dec uses the colatitude 90 - |dec| (exact) beyond 45 deg, so the radian conversion never rounds an
// angle larger than pi/4; unit-vector chords are then good to ~5e-11 arcsec.
// ------------------------------------------------------------------------------------------
// sin and cos of |x| <= pi/4 without range reduction: the classic minimax polynomials of that interval (Cephes
// sin.c / cos.c coefficients; |error| < 1.2e-16, sin keeps full relative accuracy for tiny x).  The arguments here are
// already reduced in the degree domain, so the library sincos' reduction and special cases are dead weight.
// The fp64 literals of this kernel live in constant memory on purpose: as immediates every one of them costs two 32-bit
// moves per use (74 of the key pass's 330 instructions per source were such moves), as c[bank][offset] operands none.
__constant__ double kSinPoly[6] = {1.58962301576546568060e-10, -2.50507477628578072866e-8, 2.75573136213857245213e-6,
                                   -1.98412698295895385996e-4, 8.33333333332211858878e-3, -1.66666666666666307295e-1};
__constant__ double kCosPoly[6] = {-1.13585365213876817300e-11, 2.08757008419747316778e-9, -2.75573141792967388112e-7,
                                   2.48015872888517045348e-5, -1.38888888888730564116e-3, 4.16666666666665929218e-2};
__constant__ double kTrig[4] = {0.017453292519943295 /* pi / 180 */, 1.0 / 90.0, -90.0, 57.29577951308232};

__device__ __forceinline__ void sincos_quarter(double x, double& s, double& c) {
    const double z = x * x;
    double ps = kSinPoly[0];
#pragma unroll
    for (int i = 1; i < 6; ++i) ps = fma(ps, z, kSinPoly[i]);
    s = fma(x * z, ps, x);
    double pc = kCosPoly[0];
#pragma unroll
    for (int i = 1; i < 6; ++i) pc = fma(pc, z, kCosPoly[i]);
    c = fma(z * z, pc, fma(-0.5, z, 1.0));
}

// also returns cos(dec) (>= 0), which the window flags need
__device__ __forceinline__ double unit_vector(double ra_norm, double dec, double& x, double& y, double& z) {
    const double D2R = kTrig[0];
    double q = rint(ra_norm * kTrig[1]);
    double t = fma(kTrig[2], q, ra_norm);
    double st, ct; sincos_quarter(t * D2R, st, ct);
    int iq = ((int)q) & 3;
    double ca = (iq == 0) ? ct : (iq == 1) ? -st : (iq == 2) ? -ct : st;
    double sa = (iq == 0) ? st : (iq == 1) ? ct : (iq == 2) ? -st : -ct;
    const double ad = fabs(dec);
    const bool polar = ad > 45.0;
    double s, c; sincos_quarter((polar ? 90.0 - ad : ad) * D2R, s, c);
    const double sd = copysign(polar ? c : s, dec), cd = polar ? s : c;
    x = cd * ca; y = cd * sa; z = sd;
    return cd;
}

constexpr int kKeyThreads = 256;

// Window flags of a valid source on its own grid (see kKeyExtLo ... kKeyGeneral).  Any source within r_max of
// this one has a declination in [dec - r, dec + r] and an RA within asin(sin r / cos dec) of it, and zone_of / cell_of_u
// are monotone, so its zone and cell lie between those of the window's ends evaluated with the SAME expressions that
// file sources: flags computed from the padded window are a superset of what any query radius <= r_max needs.
__device__ __forceinline__ uint32_t window_flags(const GridView& g, double dec, float cd_lo, double u, int z, int nra, int k,
                                                 double rpad_deg, double sin_r) {
    const int zl = zone_of(g, dec - rpad_deg), zh = zone_of(g, dec + rpad_deg);
    if (zl < z - 1 || zh > z + 1) return kKeyGeneral;
    // sin of the RA half-window, in fp32 rounded up (conversions and the approximate division stay below 1e-6 relative;
    // flags only have to be a superset): an fp64 division costs as much as one of this kernel's sincos
    const float sf = __fdividef((float)sin_r, cd_lo) * 1.000002f;        // cd_lo = 0 (near a pole): inf, the general path
    if (!(sf < 0.2f)) return kKeyGeneral;                             // polar rows: wide windows, rings
    const double s = (double)sf;
    const double w = fma(0.2 * s * s, s, s) * kTrig[3] + 1e-9;         // asin(s) <= s + s^3 / 5 below 0.2
    const double ulo = u - w, uhi = u + w;
    if (ulo < 0.0 ? ulo + 360.0 <= g.span : uhi >= 360.0) return kKeyGeneral;  // the window's image through RA = 0/360 lies inside the box
    const int klo = cell_of_u(g, fmax(ulo, 0.0), nra), khi = cell_of_u(g, fmin(uhi, g.span), nra);
    if (klo < k - 1 || khi > k + 1) return kKeyGeneral;
    return (klo < k ? kKeyExtLo : 0u) | (khi > k ? kKeyExtHi : 0u) | (zl < z ? kKeyDecLo : 0u) | (zh > z ? kKeyDecHi : 0u);
}

__global__ void __launch_bounds__(kKeyThreads)
k_keys_pack(const double* __restrict__ ra, const double* __restrict__ dec, const int64_t* __restrict__ id, uint32_t n,
            GridView g, int passes, double rpad_deg, double sin_r, int flagged,
            uint32_t* __restrict__ keys, Rec* __restrict__ rec, uint32_t* __restrict__ digit_hist, Stats* __restrict__ st) {
    // st != null (a build on a given grid without the extent pass): this kernel also gathers what hlc2_index_status
    // reports -- bad rows, the declination extent, and in ra_hist[0] the sources that lie outside the grid's RA box
    unsigned long long dmin = ~0ull, dmax = 0ull, bad_row = ~0ull; unsigned nbad = 0, nout = 0;
    __shared__ uint32_t hist[kMaxPasses * kRadix];
    for (int i = threadIdx.x; i < kMaxPasses * kRadix; i += kKeyThreads) hist[i] = 0;
    __syncthreads();
    // the loads of the next source are issued before the ~300 instructions of this one: without that a warp has nothing
    // in flight while it computes, and the pass waits on memory latency at half occupancy
    const size_t step = (size_t)gridDim.x * kKeyThreads;
    size_t i = (size_t)blockIdx.x * kKeyThreads + threadIdx.x;
    double a_next = 0.0, d_next = 0.0; long long v_next = 0;
    if (i < n) { a_next = __ldg(ra + i); d_next = __ldg(dec + i); v_next = id ? (long long)__ldg(id + i) : (long long)i; }
    for (; i < n; i += step) {
        const double a = a_next, d = d_next;
        const long long v = v_next;
        if (i + step < n) { a_next = __ldg(ra + i + step); d_next = __ldg(dec + i + step); v_next = id ? (long long)__ldg(id + i + step) : (long long)(i + step); }
        uint32_t key = 0, flags = 0;
        // bad coordinate: the record carries NaNs, which the gather turns into a NaN unit vector, so that no chord test
        // against anything (another bad row, the match's sentinel slot) can pass; such rows are filed under cell 0 and
        // never appear in a result
        double an = __longlong_as_double(0x7ff8000000000000ll), dd = an;
        if (coord_ok(a, d)) {
            an = norm_ra(a); dd = d;
            int z = zone_of(g, d);
            int nra = __ldg(g.n_ra + z);
            const double u = box_u(g, an);
            const int k = cell_of_u(g, u, nra);
            key = __ldg(g.cell_base + z) + (uint32_t)k;
            if (st) {
                const unsigned long long b = f64_order_bits(d);
                dmin = min(dmin, b); dmax = max(dmax, b);
                if (u > g.span) ++nout;
            }
            if (flagged) {
                // cos(dec) from below in fp32 (|error| of the conversion and of __cosf < 1e-6): the flags only have to be a
                // superset; the unit vector itself (fp64) is computed by the gather, which waits on DRAM and has the issue
                // slots this pass lacks
                const float cd_lo = fmaxf(__cosf((float)d * 0.017453292f) - 1.5e-6f, 0.0f);
                flags = window_flags(g, d, cd_lo, u, z, nra, k, rpad_deg, sin_r);
            }
        }
        else if (st) { ++nbad; bad_row = min(bad_row, (unsigned long long)i); }
        keys[i] = key | flags;          // the sort looks at the key bits only; the flags ride along
        double2* o = reinterpret_cast<double2*>(rec + i);
        o[0] = make_double2(an, dd);
        o[1] = make_double2(0.0, __longlong_as_double(v));
        for (int p = 0; p < passes; ++p) atomicAdd(&hist[p * kRadix + ((key >> (p * kRadixBits)) & (kRadix - 1))], 1u);
    }
    __syncthreads();
    for (int i = threadIdx.x; i < passes * kRadix; i += kKeyThreads)
        if (hist[i]) atomicAdd(&digit_hist[i], hist[i]);
    if (st) {
        for (int o = 16; o; o >>= 1) {
            dmin = min(dmin, __shfl_xor_sync(0xffffffffu, dmin, o)); dmax = max(dmax, __shfl_xor_sync(0xffffffffu, dmax, o));
            nout += __shfl_xor_sync(0xffffffffu, nout, o);
        }
        if ((threadIdx.x & 31) == 0) {
            if (dmin != ~0ull) { atomicMin(&st->dec_min_bits, dmin); atomicMax(&st->dec_max_bits, dmax); }
            if (nout) atomicAdd(&st->ra_hist[0], nout);
        }
        if (nbad) { atomicAdd(&st->n_bad, (unsigned long long)nbad); atomicMin(&st->first_bad_row, bad_row); }
    }
}

void launch_keys_pack(const double* ra, const double* dec, const int64_t* id, uint32_t n, GridView g, int passes,
                      double r_max_arcsec, bool flagged, uint32_t* keys, Rec* rec, uint32_t* digit_hist, cudaStream_t s, Stats* collect) {
    if (n == 0) return;
#ifndef HLC2_KEYS_CTAS
#define HLC2_KEYS_CTAS 32
#endif
    int blocks = (int)std::min<size_t>(((size_t)n + kKeyThreads - 1) / kKeyThreads, (size_t)sm_count() * HLC2_KEYS_CTAS);
    const double rpad_deg = r_max_arcsec / 3600.0 + 1e-9;
    const double sin_r = sin(r_max_arcsec * (M_PI / 648000.0)) * (1.0 + 1e-9);
    k_keys_pack<<<blocks, kKeyThreads, 0, s>>>(ra, dec, id, n, g, passes, rpad_deg, sin_r, flagged ? 1 : 0, keys, rec, digit_hist, collect);
    count_launch();
}

// ------------------------------------------------------------------------------------------
// block-wide inclusive scan of one value per thread (any multiple of 32 threads up to 1024)
// ------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t block_scan_incl(uint32_t v, uint32_t* total, uint32_t* sm /*[33]*/) {
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    for (int o = 1; o < 32; o <<= 1) { uint32_t t = __shfl_up_sync(0xffffffffu, v, o); if (lane >= o) v += t; }
    if (lane == 31) sm[w] = v;
    __syncthreads();
    if (w == 0) {
        uint32_t t = lane < (int)(blockDim.x >> 5) ? sm[lane] : 0u;
        for (int o = 1; o < 32; o <<= 1) { uint32_t u = __shfl_up_sync(0xffffffffu, t, o); if (lane >= o) t += u; }
        sm[lane] = t;
        if (lane == 31) sm[32] = t;
    }
    __syncthreads();
    if (w > 0) v += sm[w - 1];
    *total = sm[32];
    __syncthreads();
    return v;
}

// ------------------------------------------------------------------------------------------
// (a2) LSD radix sort of (key, row): 9-bit digits, one kernel per pass.
// ------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(kRadix)
k_digit_scan(const uint32_t* __restrict__ digit_hist, uint32_t* __restrict__ digit_base, int passes) {
    __shared__ uint32_t sm[33];
    for (int p = 0; p < passes; ++p) {
        uint32_t c = digit_hist[p * kRadix + threadIdx.x], tot;
        uint32_t inc = block_scan_incl(c, &tot, sm);
        digit_base[p * kRadix + threadIdx.x] = inc - c;
    }
}

#ifndef HLC2_OS_THREADS
#define HLC2_OS_THREADS 512
#endif
constexpr int kOsThreads = HLC2_OS_THREADS;     // thread t owns digits t * kOsDig .. in the tile-level scans
constexpr int kOsDig = kRadix / kOsThreads;
constexpr int kOsCtas = 1024 / kOsThreads;      // CTAs per SM the kernel is sized for
#ifndef HLC2_OS_LOOK
#define HLC2_OS_LOOK 4
#endif
constexpr int kLook = HLC2_OS_LOOK;       // predecessor records read per look-back step
#ifndef HLC2_OS_PREFETCH
#define HLC2_OS_PREFETCH 1
#endif
#ifndef HLC2_OS_ITEMS
#define HLC2_OS_ITEMS 18
#endif
constexpr int kOsItems = HLC2_OS_ITEMS;         // even
constexpr int kOsTile = kOsThreads * kOsItems;  // 9216 keys per tile
constexpr int kOsWarps = kOsThreads / 32;
constexpr uint32_t kFlagAgg = 1u << 30, kFlagIncl = 2u << 30, kFlagMask = 3u << 30;
constexpr size_t kOsSmem = (size_t)(kOsWarps * kRadix + 2 * kOsTile) * 4;
static_assert(kOsThreads * kOsDig == kRadix && kOsDig >= 1, "whole digits per thread");

size_t sort_tiles(uint32_t n) { return ((size_t)n + kOsTile - 1) / kOsTile; }

// lanes of the (converged) warp that hold the same value d < 2^(kRadixBits + 1), one ballot per bit.  Out of line: it is the
// rare path of the ranking and must not cost the common one registers.
__device__ __noinline__ unsigned match_by_votes(uint32_t d) {
    unsigned p = 0xffffffffu;
#pragma unroll 1
    for (int b = 0; b <= kRadixBits; ++b) {                           // bit kRadixBits tells empty slots (all ones) apart
        const bool bit = (d >> b) & 1u;
        const unsigned vote = __ballot_sync(0xffffffffu, bit);
        p &= bit ? vote : ~vote;
    }
    return p;
}

template <bool FirstPass>
__global__ void __launch_bounds__(kOsThreads, kOsCtas)
k_onesweep(const uint32_t* __restrict__ keys, const uint32_t* __restrict__ vals, uint32_t n, int shift, uint32_t mask,
           const uint32_t* __restrict__ digit_base, volatile uint32_t* __restrict__ status, uint32_t* __restrict__ ticket,
           uint32_t* __restrict__ out_keys, uint32_t* __restrict__ out_vals) {
    extern __shared__ uint32_t dsm[];
    uint32_t* wh = dsm;                            // [kOsWarps][kRadix] per-warp digit counters -> offsets
    uint32_t* s_keys = dsm + kOsWarps * kRadix;    // [kOsTile]
    uint32_t* s_vals = s_keys + kOsTile;           // [kOsTile]
    __shared__ uint32_t s_tile, s_scan[33];
    __shared__ uint32_t s_gbase[kRadix];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;

    // tiles are taken in ticket order, so every predecessor of a running tile has itself started: the
    // look-back below can only wait on CTAs that are resident or finished
    if (threadIdx.x == 0) s_tile = atomicAdd(ticket, 1u);
    for (int i = threadIdx.x; i < kOsWarps * kRadix; i += kOsThreads) wh[i] = 0;
    __syncthreads();
    const uint32_t tile = s_tile;
    const size_t tile_base = (size_t)tile * kOsTile;
    const uint32_t cnt = (uint32_t)min((size_t)kOsTile, (size_t)n - tile_base);

    // warp w owns kOsItems*32 consecutive keys; item r of lane l is key (w*kOsItems + r)*32 + l of the tile
    const uint32_t t0 = (uint32_t)w * (kOsItems * 32) + lane;         // slot of item r in the tile: t0 + 32 r
    const uint32_t* tkeys = keys + tile_base;
    // the rows (vals) are not held across the ranking: they are read when the reorder needs them, which keeps the
    // kernel inside 64 registers without spills
    uint32_t k[kOsItems], rk[kOsItems / 2];                   // ranks (< kOsTile) packed two per register
#pragma unroll
    for (int r = 0; r < kOsItems; ++r) {
        const uint32_t t = t0 + r * 32;
        k[r] = t < cnt ? __ldg(tkeys + t) : 0xFFFFFFFFu;
#if HLC2_OS_PREFETCH
        // the rows are read after the ranking (three groups, each a DRAM latency if cold): ask L2 for their lines now
        if (!FirstPass && lane == 0 && t < cnt) asm volatile("prefetch.global.L2 [%0];" :: "l"(vals + tile_base + t));
#endif
    }
    const unsigned lt = (1u << lane) - 1;
    uint32_t* mywh = wh + w * kRadix;
    // ranks, kG items at a time in phases (tags, matches, counter bumps, broadcasts), so that the latencies of the
    // shared-memory accesses, of the atomics and of the shuffles overlap instead of adding up item by item.
    // No MATCH.ANY: it measures 48 cycles per warp instruction per SM on sm_100a and alone was half of this kernel's time
    // (profiles/r2_build_experiments.md); nine ballots (one per digit bit) measure 20, the owner tags below about half of that.
#ifndef HLC2_OS_GROUP
#define HLC2_OS_GROUP 3
#endif
    constexpr int kG = HLC2_OS_GROUP;
    static_assert(kOsItems % kG == 0, "items are ranked in groups");
#pragma unroll
    for (int g = 0; g < kOsItems; g += kG) {
        uint32_t d[kG]; unsigned peers[kG]; uint32_t old[kG];
        // owner tags: every lane writes its number under its digit in a table of the warp's own and reads it back; a lane
        // that reads another lane's number shares its digit with it.  Only those digits (one per item on average with 32
        // keys over 512 digits) are then settled by a vote each; everybody else is alone and needs no vote at all.
        uint8_t* own = reinterpret_cast<uint8_t*>(s_keys) + (size_t)(w * kG) * kRadix;     // the staging area is free until the reorder
#pragma unroll
        for (int j = 0; j < kG; ++j) {
            const bool ok = t0 + (g + j) * 32 < cnt;
            d[j] = ok ? ((k[g + j] >> shift) & mask) : 0xFFFFFFFFu;
            if (ok) own[j * kRadix + d[j]] = (uint8_t)lane;
        }
        __syncwarp();
#pragma unroll
        for (int j = 0; j < kG; ++j) {
            const bool lost = d[j] != 0xFFFFFFFFu && own[j * kRadix + d[j]] != (uint8_t)lane;
            unsigned open = __ballot_sync(0xffffffffu, lost);
            peers[j] = 1u << lane;
            // many shared digits (a dense cell, sorted input): one vote per digit bit settles them all at once
            if (__popc(open) > 8) { peers[j] = match_by_votes(d[j]); open = 0; }
            while (open) {
                const uint32_t dl = __shfl_sync(0xffffffffu, d[j], __ffs(open) - 1);
                const unsigned grp = __ballot_sync(0xffffffffu, d[j] == dl);
                if (d[j] == dl) peers[j] = grp;
                open &= ~grp;
            }
        }
        __syncwarp();                                                 // the next group reuses the tables
        // lanes with the same digit: the lowest of them bumps the warp's counter once for all and hands the old value
        // round; the groups of one step are disjoint digits or the same counter in program order: atomics keep it exact
#pragma unroll
        for (int j = 0; j < kG; ++j) {
            old[j] = 0;
            if (d[j] != 0xFFFFFFFFu && lane == __ffs(peers[j]) - 1) old[j] = atomicAdd(&mywh[d[j]], (uint32_t)__popc(peers[j]));
        }
#pragma unroll
        for (int j = 0; j < kG; ++j) {
            const int r = g + j;
            const uint32_t rank = __shfl_sync(0xffffffffu, old[j], __ffs(peers[j]) - 1) + (uint32_t)__popc(peers[j] & lt);
            if (r & 1) rk[r >> 1] |= rank << 16; else rk[r >> 1] = rank;
        }
    }
    __syncthreads();

    // digits threadIdx.x * kOsDig ..: exclusive scan over the warps, tile count, chained scan over the tiles
    const int dgt0 = threadIdx.x * kOsDig;
    uint32_t c[kOsDig], loc[kOsDig], csum = 0;
#pragma unroll
    for (int q = 0; q < kOsDig; ++q) {
        const int dgt = dgt0 + q;
        uint32_t cc = 0;
#pragma unroll
        for (int ww = 0; ww < kOsWarps; ++ww) { uint32_t t = wh[ww * kRadix + dgt]; wh[ww * kRadix + dgt] = cc; cc += t; }
        c[q] = cc; csum += cc;
        status[(size_t)tile * kRadix + dgt] = cc | (tile == 0 ? kFlagIncl : kFlagAgg);
    }
    uint32_t tot;
    uint32_t run = block_scan_incl(csum, &tot, s_scan) - csum;      // first position of the thread's first digit in the sorted tile
#pragma unroll
    for (int q = 0; q < kOsDig; ++q) {
        loc[q] = run; run += c[q];
#pragma unroll
        for (int ww = 0; ww < kOsWarps; ++ww) wh[ww * kRadix + dgt0 + q] += loc[q];
    }
    __syncthreads();

    // the reorder in shared memory needs tile-local offsets only: it runs BEFORE the look-back, so that the tiles ahead
    // (which started earlier) have had that much longer to publish their inclusive prefixes and the walk stays short
    constexpr int kV = 6;
#pragma unroll
    for (int g = 0; g < kOsItems; g += kV) {
        uint32_t v[kV];
#pragma unroll
        for (int j = 0; j < kV; ++j) {
            const uint32_t t = t0 + (g + j) * 32;
            v[j] = FirstPass ? (uint32_t)tile_base + t : (t < cnt ? __ldg(vals + tile_base + t) : 0u);
        }
#pragma unroll
        for (int j = 0; j < kV; ++j) {
            const int r = g + j;
            if (t0 + r * 32 < cnt) {
                const uint32_t d = (k[r] >> shift) & mask;
                const uint32_t pos = mywh[d] + ((rk[r >> 1] >> (16 * (r & 1))) & 0xFFFFu);
                s_keys[pos] = k[r]; s_vals[pos] = v[j];
            }
        }
    }

    uint32_t excl[kOsDig];
#pragma unroll
    for (int q = 0; q < kOsDig; ++q) excl[q] = 0;
    if (tile > 0) {
        // look back over the predecessors' records, kLook at a time (independent loads: one memory latency per kLook
        // tiles instead of one per tile); stop at the first inclusive prefix, re-poll from the first record not yet there
        long long at[kOsDig]; bool done[kOsDig]; bool all = false;
#pragma unroll
        for (int q = 0; q < kOsDig; ++q) { at[q] = (long long)tile - 1; done[q] = false; }
        while (!all) {
            uint32_t sv[kOsDig][kLook];
#pragma unroll
            for (int q = 0; q < kOsDig; ++q)
#pragma unroll
                for (int j = 0; j < kLook; ++j) {
                    sv[q][j] = 2u << 30;                             // before tile 0: an empty inclusive prefix
                    if (!done[q] && at[q] - j >= 0) sv[q][j] = status[(size_t)(at[q] - j) * kRadix + dgt0 + q];
                }
            all = true;
#pragma unroll
            for (int q = 0; q < kOsDig; ++q) {
                if (done[q]) continue;
                int used = kLook;
#pragma unroll
                for (int j = 0; j < kLook; ++j) {
                    if (done[q] || used != kLook) continue;
                    if ((sv[q][j] & kFlagMask) == 0) { used = j; continue; }
                    excl[q] += sv[q][j] & ~kFlagMask;
                    if (sv[q][j] & kFlagIncl) done[q] = true;
                }
                at[q] -= used;
                all = all && done[q];
            }
        }
#pragma unroll
        for (int q = 0; q < kOsDig; ++q) status[(size_t)tile * kRadix + dgt0 + q] = (excl[q] + c[q]) | kFlagIncl;
    }
#pragma unroll
    for (int q = 0; q < kOsDig; ++q)                                 // global slot of sorted-tile position j is s_gbase[d] + j
        s_gbase[dgt0 + q] = __ldg(digit_base + dgt0 + q) + excl[q] - loc[q];
    __syncthreads();
    for (uint32_t j = threadIdx.x; j < cnt; j += kOsThreads) {
        const uint32_t key = s_keys[j];
        const uint32_t dst = s_gbase[(key >> shift) & mask] + j;
        out_keys[dst] = key; out_vals[dst] = s_vals[j];
    }
}

int radix_passes(int key_bits) { return std::max(1, (key_bits + kRadixBits - 1) / kRadixBits); }

// sorts (keys, row) by key; returns which of the double buffers holds the result (0 = a, 1 = b).
// d_digit_hist must hold the per-pass digit counts of keys_a (k_keys_pack); d_status (zeroed by this call) has
// passes * sort_tiles(n) * kRadix entries; d_ticket kMaxPasses entries.
int launch_radix_sort(uint32_t* keys_a, uint32_t* keys_b, uint32_t* val_a, uint32_t* val_b, uint32_t n, int key_bits,
                      const uint32_t* d_digit_hist, uint32_t* d_digit_base, uint32_t* d_status, uint32_t* d_ticket,
                      cudaStream_t s) {
    if (n == 0) return 0;
    static bool attr_set[kMaxDevices] = {};          // the opt-in is a per-device function attribute
    const int dev = current_device();
    if (!attr_set[dev]) {
        cudaFuncSetAttribute(k_onesweep<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kOsSmem);
        cudaFuncSetAttribute(k_onesweep<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kOsSmem);
        attr_set[dev] = true;
    }
    const int passes = radix_passes(key_bits);
    const uint32_t n_tiles = (uint32_t)sort_tiles(n);
    cudaMemsetAsync(d_status, 0, (size_t)passes * n_tiles * kRadix * sizeof(uint32_t), s);
    cudaMemsetAsync(d_ticket, 0, kMaxPasses * sizeof(uint32_t), s);
    k_digit_scan<<<1, kRadix, 0, s>>>(d_digit_hist, d_digit_base, passes); count_launch();
    uint32_t *ki = keys_a, *ko = keys_b, *vi = val_a, *vo = val_b;
    for (int p = 0; p < passes; ++p) {
        const int shift = kRadixBits * p;
        const int bits = std::min(kRadixBits, std::max(1, key_bits - shift));
        const uint32_t mask = (1u << bits) - 1u;
        uint32_t* st = d_status + (size_t)p * n_tiles * kRadix;
        if (p == 0) k_onesweep<true><<<n_tiles, kOsThreads, kOsSmem, s>>>(ki, vi, n, shift, mask, d_digit_base + p * kRadix, st, d_ticket + p, ko, vo);
        else        k_onesweep<false><<<n_tiles, kOsThreads, kOsSmem, s>>>(ki, vi, n, shift, mask, d_digit_base + p * kRadix, st, d_ticket + p, ko, vo);
        count_launch();
        std::swap(ki, ko); std::swap(vi, vo);
    }
    return passes & 1;
}

// ------------------------------------------------------------------------------------------
// (a3) gather: sorted row order -> SoA unit vectors + ids.  One 32-byte sector per source.
// ------------------------------------------------------------------------------------------
// A random 32-byte record costs a whole 128-byte line of DRAM traffic on this part whatever its neighbours do
// (profiles/r2_build_experiments.md): the kernel is bound by line fetches in flight.  One row per thread and a grid far
// larger than what is resident measured best (2.9 ms per 1e8 rows; 16 persistent CTAs per SM: 3.5 ms, their last
// wave leaves a third of the SM idle; two or four rows per thread: 3.0-3.8 ms).
__global__ void __launch_bounds__(256)
k_gather(const Rec* __restrict__ rec, const uint32_t* __restrict__ perm, uint32_t n,
         double* __restrict__ x, double* __restrict__ y, double* __restrict__ z, int64_t* __restrict__ out_id,
         float2* __restrict__ pos) {
    for (size_t i = (size_t)blockIdx.x * 256 + threadIdx.x; i < n; i += (size_t)gridDim.x * 256) {
        const double2* q = reinterpret_cast<const double2*>(rec + __ldg(perm + i));
        const double2 a = __ldg(q), b = __ldg(q + 1);          // (ra in [0, 360), dec), (-, id); NaNs mark a bad row
        double ux = a.x, uy = a.x, uz = a.x;
        if (a.x == a.x) unit_vector(a.x, a.y, ux, uy, uz);
        x[i] = ux; y[i] = uy; z[i] = uz; out_id[i] = __double_as_longlong(b.y);
        // fp32 (ra, dec) of the sorted row: the two-grid match locates its search window from it, padded by far more
        // (kEpsRaDeg, kEpsDecDeg) than the rounding to fp32
        pos[i] = make_float2((float)a.x, (float)a.y);
    }
}

void launch_gather(const Rec* rec, const uint32_t* perm, uint32_t n, double* x, double* y, double* z, int64_t* out_id,
                   float2* pos, cudaStream_t s) {
    if (n == 0) return;
    int blocks = (int)std::min<size_t>(((size_t)n + 255) / 256, (size_t)sm_count() * 4096);
    k_gather<<<blocks, 256, 0, s>>>(rec, perm, n, x, y, z, out_id, pos); count_launch();
}

// ------------------------------------------------------------------------------------------
// (a4) cell offset table.  Sorted row i is the first row of every cell in (key[i-1], key[i]]; row n (one past
// the end) closes every cell above key[n-1].  Short runs are written by the owning lane, medium runs by its
// warp, long runs (empty sky) go to a list that k_cell_fill_big spreads over the whole grid.
// ------------------------------------------------------------------------------------------
constexpr uint32_t kFillLane = 4, kFillWarp = 4096, kFillBuf = 1024;

__global__ void __launch_bounds__(256)
k_cell_fill(const uint32_t* __restrict__ keys, uint32_t kmask, uint32_t n, uint32_t n_cells, uint32_t* __restrict__ cell_start,
            uint32_t* __restrict__ big, uint32_t* __restrict__ big_count, uint32_t big_cap) {
    __shared__ uint32_t s_cells[8][kFillBuf];
    const int lane = threadIdx.x & 31;
    uint32_t* sc = s_cells[threadIdx.x >> 5];
    const size_t total = (size_t)n + 1;
    // a warp takes 128 consecutive rows per step, four per lane (one 16-byte load): a pass that moves 4 bytes per
    // row needs that many bytes in flight to cover the DRAM latency
    const size_t stride = (size_t)gridDim.x * 256 * 4;
    for (size_t b = ((size_t)blockIdx.x * 256 + (threadIdx.x & ~31)) * 4; b < total; b += stride) {   // warp-uniform trip count
        const size_t i0 = b + 4 * (size_t)lane;
        uint32_t k[4];
        if (i0 + 3 < n) {
            const uint4 v = __ldg(reinterpret_cast<const uint4*>(keys + i0));
            k[0] = v.x & kmask; k[1] = v.y & kmask; k[2] = v.z & kmask; k[3] = v.w & kmask;
        } else {
#pragma unroll
            for (int j = 0; j < 4; ++j) k[j] = i0 + j < n ? (__ldg(keys + i0 + j) & kmask) : n_cells;
        }
        uint32_t prev = __shfl_up_sync(0xffffffffu, k[3], 1);
        if (lane == 0) prev = b > 0 ? (__ldg(keys + b - 1) & kmask) : 0u;
        // common case, the 128 rows span fewer than kFillBuf cells: every row writes its number under the cells it opens
        // (those above the previous row's key up to its own) into a table of the warp's own in shared memory, then the
        // warp copies the table out -- consecutive words instead of scattered ones, and no chain of dependent look-ups
        {
            const uint32_t lo_cell = b > 0 ? __shfl_sync(0xffffffffu, prev, 0) + 1u : 0u;
            const uint32_t hi_cell = __shfl_sync(0xffffffffu, k[3], 31);
            if (hi_cell - lo_cell < kFillBuf || hi_cell < lo_cell) {     // hi < lo: all 128 rows lie in the previous row's cell
                __syncwarp();
                uint32_t p = prev;
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    const size_t i = i0 + j;
                    if (i < total) {
                        const uint32_t first = i > 0 ? p + 1u : 0u;
                        for (uint32_t c = first; c <= k[j] && c >= first; ++c) sc[c - lo_cell] = (uint32_t)i;
                    }
                    p = k[j];
                }
                __syncwarp();
                if (hi_cell >= lo_cell)
                    for (uint32_t c = lane; c <= hi_cell - lo_cell; c += 32) cell_start[(size_t)lo_cell + c] = sc[c];
                continue;
            }
        }
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const size_t i = i0 + j;
            uint32_t lo = 1, hi = 0;                           // empty
            if (i < total) {
                hi = k[j];                                     // row n (one past the end) closes every cell above key[n-1]
                lo = i > 0 ? prev + 1u : 0u;
                if (i > 0 && i < n && hi + 1u == lo) { lo = 1; hi = 0; }      // same cell as the previous row
            }
            prev = k[j];
            const uint32_t span = hi >= lo ? hi - lo + 1u : 0u;
            if (span && span <= kFillLane) for (uint32_t c = lo; c <= hi; ++c) cell_start[c] = (uint32_t)i;
            unsigned m = __ballot_sync(0xffffffffu, span > kFillLane);
            while (m) {
                const int src = __ffs(m) - 1; m &= m - 1;
                const uint32_t l = __shfl_sync(0xffffffffu, lo, src), h = __shfl_sync(0xffffffffu, hi, src);
                const uint32_t v = (uint32_t)(b + 4 * (size_t)src + j);
                if (h - l + 1u <= kFillWarp) {
                    for (uint64_t cc = (uint64_t)l + lane; cc <= h; cc += 32) cell_start[cc] = v;
                } else if (lane == 0) {
                    uint32_t e = atomicAdd(big_count, 1u);
                    if (e < big_cap) { big[3 * e] = l; big[3 * e + 1] = h; big[3 * e + 2] = v; }
                }
            }
        }
    }
}

__global__ void __launch_bounds__(256)
k_cell_fill_big(const uint32_t* __restrict__ big, const uint32_t* __restrict__ big_count, uint32_t big_cap,
                uint32_t* __restrict__ cell_start) {
    const uint32_t m = min(*big_count, big_cap);
    for (uint32_t e = 0; e < m; ++e) {
        const uint32_t l = big[3 * e], h = big[3 * e + 1], v = big[3 * e + 2];
        for (uint64_t c = (uint64_t)l + (size_t)blockIdx.x * 256 + threadIdx.x; c <= h; c += (uint64_t)gridDim.x * 256) cell_start[c] = v;
    }
}

// per-record error radii (input order, arcsec) -> squares in cell order
__global__ void __launch_bounds__(256)
k_gather_err2(const double* __restrict__ err, const uint32_t* __restrict__ perm, uint32_t n, double* __restrict__ err2) {
    for (size_t i = (size_t)blockIdx.x * 256 + threadIdx.x; i < n; i += (size_t)gridDim.x * 256) {
        const double e = __ldg(err + __ldg(perm + i));
        err2[i] = e >= 0.0 ? e * e : __longlong_as_double(0x7ff8000000000000ll);      // a negative or NaN radius matches nothing
    }
}
void launch_gather_err2(const double* err_arcsec, const uint32_t* perm, uint32_t n, double* err2, cudaStream_t s) {
    if (n == 0) return;
    int blocks = (int)std::min<size_t>(((size_t)n + 255) / 256, (size_t)sm_count() * 16);
    k_gather_err2<<<blocks, 256, 0, s>>>(err_arcsec, perm, n, err2); count_launch();
}

size_t cell_big_cap(size_t n_cells) { return n_cells / kFillWarp + 2; }

void launch_cell_table(const uint32_t* sorted_keys, uint32_t key_mask, uint32_t n, uint32_t n_cells, uint32_t* cell_start,
                       uint32_t* d_big /*[3*cap + 1]*/, cudaStream_t s) {
    const uint32_t cap = (uint32_t)cell_big_cap(n_cells);
    uint32_t* d_count = d_big + 3 * (size_t)cap;
    cudaMemsetAsync(d_count, 0, sizeof(uint32_t), s);
#ifndef HLC2_FILL_CTAS
#define HLC2_FILL_CTAS 64
#endif
    int blocks = (int)std::min<size_t>(((size_t)n + 1 + 1023) / 1024, (size_t)sm_count() * HLC2_FILL_CTAS);
    k_cell_fill<<<blocks, 256, 0, s>>>(sorted_keys, key_mask, n, n_cells, cell_start, d_big, d_count, cap); count_launch();
    k_cell_fill_big<<<sm_count() * 4, 256, 0, s>>>(d_big, d_count, cap, cell_start); count_launch();
}

// ------------------------------------------------------------------------------------------
// (a4) tile descriptors: tile = up to kTile consecutive sorted rows of ONE zone (the role of the paper's
// calculation blocks: there cut to fit the N^2 result matrix, here to fit one CTA).
// ------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(1024)
k_zone_tiles(const uint32_t* __restrict__ cell_start, const uint32_t* __restrict__ cell_base, uint32_t n_zones,
             uint32_t* __restrict__ tile_first /*[n_zones + 1]*/, uint32_t* __restrict__ n_tiles) {
    __shared__ uint32_t sm[33];
    uint32_t carry = 0;
    for (uint32_t b = 0; b < n_zones; b += 1024) {
        const uint32_t z = b + threadIdx.x;
        uint32_t t = 0;
        if (z < n_zones) {
            const uint32_t cnt = __ldg(cell_start + __ldg(cell_base + z + 1)) - __ldg(cell_start + __ldg(cell_base + z));
            t = (cnt + kTile - 1) / kTile;
        }
        uint32_t tot;
        const uint32_t inc = block_scan_incl(t, &tot, sm);
        if (z < n_zones) tile_first[z] = carry + inc - t;
        carry += tot;
    }
    if (threadIdx.x == 0) { tile_first[n_zones] = carry; *n_tiles = carry; }
}

// one warp per tile: descriptor + the OR of the rows' window flags (so the same-grid match knows without looking at
// the rows whether any of them reaches into the zone below / above or needs the general path)
__global__ void __launch_bounds__(256)
k_tile_desc(const uint32_t* __restrict__ tile_first, uint32_t n_zones, const uint32_t* __restrict__ cell_start,
            const uint32_t* __restrict__ cell_base, const uint32_t* __restrict__ n_ra, const uint32_t* __restrict__ keys, uint32_t kmask,
            TileDesc* __restrict__ tiles) {
    const uint32_t nt = __ldg(tile_first + n_zones);
    const int lane = threadIdx.x & 31;
    // kTd tiles per warp and step, their look-up chains (zone search -> cell_base -> cell_start -> keys) side by side:
    // one chain is a dozen dependent memory latencies, and a warp with a single one in flight mostly waits
    constexpr int kTd = 4;
    int iters = 1; while ((1u << iters) < n_zones + 1u) ++iters;
    for (uint32_t t0 = (blockIdx.x * 8 + (threadIdx.x >> 5)) * kTd; t0 < nt; t0 += gridDim.x * 8 * kTd) {
        uint32_t lo[kTd], hi[kTd];
#pragma unroll
        for (int q = 0; q < kTd; ++q) { lo[q] = 0; hi[q] = n_zones; }          // largest z with tile_first[z] <= t
        for (int it = 0; it < iters; ++it) {
#pragma unroll
            for (int q = 0; q < kTd; ++q) {
                if (hi[q] - lo[q] > 1) { const uint32_t mid = (lo[q] + hi[q]) >> 1; if (__ldg(tile_first + mid) <= min(t0 + q, nt - 1)) lo[q] = mid; else hi[q] = mid; }
            }
        }
        uint32_t cb[kTd], cbn[kTd], tf[kTd], zs[kTd], ze[kTd], s0[kTd], m[kTd], fl[kTd];
#pragma unroll
        for (int q = 0; q < kTd; ++q) { cb[q] = __ldg(cell_base + lo[q]); cbn[q] = __ldg(cell_base + lo[q] + 1); tf[q] = __ldg(tile_first + lo[q]); }
#pragma unroll
        for (int q = 0; q < kTd; ++q) { zs[q] = __ldg(cell_start + cb[q]); ze[q] = __ldg(cell_start + cbn[q]); }
        uint32_t kv[kTd][kTile / 32];
#pragma unroll
        for (int q = 0; q < kTd; ++q) {
            const uint32_t t = min(t0 + q, nt - 1);
            s0[q] = zs[q] + (t - tf[q]) * kTile;
            m[q] = min((uint32_t)kTile, ze[q] - s0[q]);
#pragma unroll
            for (int r = 0; r < kTile / 32; ++r) kv[q][r] = lane + 32 * r < m[q] ? __ldg(keys + s0[q] + lane + 32 * r) : 0u;
        }
#pragma unroll
        for (int q = 0; q < kTd; ++q) {
            uint32_t f_or = 0;
#pragma unroll
            for (int r = 0; r < kTile / 32; ++r) {
                const uint32_t f = kv[q][r] & ~kmask;
                f_or |= (f & kKeyGeneral) == kKeyGeneral ? kTileGeneral : ((f & kKeyDecLo ? kTileDecLo : 0u) | (f & kKeyDecHi ? kTileDecHi : 0u));
            }
            fl[q] = __reduce_or_sync(0xffffffffu, f_or);
        }
#pragma unroll
        for (int q = 0; q < kTd; ++q) {
            if (lane == q && t0 + q < nt) {                     // lane q writes tile q's descriptor
                const uint32_t z = lo[q];
                TileDesc d;
                d.first = s0[q]; d.count = m[q]; d.zone = z;
                d.k_first = (__ldg(keys + s0[q]) & kmask) - cb[q]; d.k_last = (__ldg(keys + s0[q] + m[q] - 1) & kmask) - cb[q];
                d.flags = fl[q]; d.cb = cb[q];
                d.n = __ldg(n_ra + z); d.n_lo = z > 0 ? __ldg(n_ra + z - 1) : 0u; d.n_hi = z + 1 < n_zones ? __ldg(n_ra + z + 1) : 0u;
                d.inv_n = 1.0 / (double)d.n;
                tiles[t0 + q] = d;
            }
        }
    }
}

void launch_tiles(const uint32_t* cell_start, const uint32_t* cell_base, const int32_t* n_ra, uint32_t n_zones, const uint32_t* sorted_keys,
                  uint32_t key_mask, uint32_t tile_cap, uint32_t* d_tile_first, TileDesc* tiles, uint32_t* d_n_tiles, cudaStream_t s) {
    k_zone_tiles<<<1, 1024, 0, s>>>(cell_start, cell_base, n_zones, d_tile_first, d_n_tiles); count_launch();
#ifndef HLC2_TILE_CTAS
#define HLC2_TILE_CTAS 64
#endif
    int blocks = (int)std::min<size_t>(((size_t)tile_cap + 31) / 32, (size_t)sm_count() * HLC2_TILE_CTAS);
    k_tile_desc<<<std::max(blocks, 1), 256, 0, s>>>(d_tile_first, n_zones, cell_start, cell_base, reinterpret_cast<const uint32_t*>(n_ra), sorted_keys, key_mask, tiles); count_launch();
}

}  // namespace hlc2
