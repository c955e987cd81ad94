// hlc2_match.cu -- the match kernels (NS (b)).
//
// One lane per A source (the paper's thread-per-A-record hierarchy), but instead of looping
// over a whole calculation block (L271) a lane visits only the B cells its search window can reach:
//   dec window  [dec - r, dec + r]                         -> 1..3 zones of B's grid
//   RA  window  [ra - w, ra + w], w = asin(sin r / cos dec) -> 1..2 contiguous cell ranges per zone
//               (full ring when cos dec <= ~4 sin r, i.e. at the poles; two ranges when the
//               window crosses RA = 0/360).  These are the cells the quad-direction strategy
//               probes (L122-169) plus the diagonal neighbours and the 1/cos(dec) widening it
//               omits, so no pair is lost (the "No Index" result, L344).
// The window is located from the index's fp32 (ra, dec) estimate padded by a rigorous error bound;
// over-inclusion only costs time.  Decisions are fp64: chord^2 <= 4 sin^2(r/2).
//
// Warp = worker.  A persistent grid of 256-thread CTAs; each warp takes chunks of 32 consecutive
// cell-sorted A rows.  The kernel is bound by instruction issue, not by bytes (profiles/), hence:
//   * fast path: a lane whose window lies in one zone and does not wrap scans ONE contiguous row range;
//   * every other lane (zone-spanning, RA wrap, polar ring, outside B's box: a few % of the sky) is
//     deferred to a per-warp list and handled 32 at a time by the general path, so that path runs
//     with full lanes instead of once for every warp that owns one such lane;
//   * hits (the role of d_out_dis, L282): a lane keeps its first hit in registers, the warp appends all
//     first hits to its shared-memory queue by ballot + popcount, further hits of a lane go there by a
//     shared atomic; every 32 queued rows are flushed with ONE global atomic and coalesced stores of
//     (idA, idB, sep) -- the id look-ups, sqrt and asin run on full warps.
// No __syncthreads anywhere: warps never wait on each other.
#include <math.h>

#include "hlc2_grid.cuh"

namespace hlc2 {

constexpr int kMatchThreads = 256;
constexpr int kMatchWarps = kMatchThreads / 32;
constexpr int kQCap = 128;        // rows in a warp's hit queue
constexpr int kQSoft = 96;        // in-scan pushes stop here so that 32 first hits always fit behind them
constexpr int kDeferCap = 64;     // <= 31 pending + 32 new
constexpr double kRad2Arcsec = 206264.80624709636;   // 648000 / pi
constexpr unsigned kFull = 0xffffffffu;

// padding of the fp32 position estimate (degrees); derivation in DESIGN.md section 5 (~3x the worst case)
constexpr double kEpsRaDeg = 2.5e-4;
constexpr double kEpsDecDeg = 1.5e-4;

struct MatchArgs {
    double thr2;          // 4 sin^2(r/2)
    double pad_dec;       // r in degrees + kEpsDecDeg
    float sin_r_up;       // sin(r) * (1 + 1e-5)
    int64_t* out_ida; int64_t* out_idb; double* out_sep;
    unsigned long long capacity;
    unsigned long long* count;
    uint32_t n_chunks;
};

struct WarpShared {
    double q_c2[kQCap];
    uint32_t q_a[kQCap], q_b[kQCap];
    uint32_t defer[kDeferCap];
    unsigned q_n;
    unsigned pad[3];
};

// sep = 2 asin(chord / 2) in arcsec.  Below 2^-10 rad (403 arcsec) the series h + h^3/6 + 3 h^5/40 is exact to
// 4e-20 relative; above it the library asin.
__device__ __forceinline__ double sep_from_chord2(double c2) {
    const double h = 0.5 * sqrt(c2);
    double a;
    if (h < 0.0009765625) { const double t = h * h; a = fma(h * t, fma(t, 0.075, 1.0 / 6.0), h); }
    else a = asin(fmin(1.0, h));
    return a * (2.0 * kRad2Arcsec);
}

struct Hit { double c2; uint32_t j; bool has; };

__device__ __forceinline__ void emit_direct(const IndexView& A, const IndexView& B, const MatchArgs& p,
                                            uint32_t a, uint32_t j, double c2) {
    const unsigned long long o = atomicAdd(p.count, 1ull);
    if (o < p.capacity) { p.out_ida[o] = __ldg(A.id + a); p.out_idb[o] = __ldg(B.id + j); p.out_sep[o] = sep_from_chord2(c2); }
}

// scan B rows [j0, j1) for A row a
template <int MODE>
__device__ __forceinline__ void scan_range(const IndexView& A, const IndexView& B, const MatchArgs& p, WarpShared& ws,
                                           uint32_t a, double ax, double ay, double az, uint32_t j0, uint32_t j1, Hit& h) {
    for (uint32_t j = j0; j < j1; ++j) {
        const double dx = ax - __ldg(B.x + j), dy = ay - __ldg(B.y + j), dz = az - __ldg(B.z + j);
        const double c2 = fma(dx, dx, fma(dy, dy, dz * dz));
        if (c2 <= p.thr2) {
            if (MODE == HLC2_ALL_PAIRS) {
                if (!h.has) { h.has = true; h.j = j; h.c2 = c2; }
                else {
                    const unsigned slot = atomicAdd(&ws.q_n, 1u);
                    if (slot < (unsigned)kQSoft) { ws.q_a[slot] = a; ws.q_b[slot] = j; ws.q_c2[slot] = c2; }
                    else emit_direct(A, B, p, a, j, c2);
                }
            } else {
                if (!h.has || c2 < h.c2 || (c2 == h.c2 && __ldg(B.id + j) < __ldg(B.id + h.j))) { h.has = true; h.j = j; h.c2 = c2; }
            }
        }
    }
}

// everything the fast path does not take: several zones, RA wrap, polar ring, window partly outside B's box
template <int MODE>
__device__ __noinline__ void scan_general(const IndexView& A, const IndexView& B, const MatchArgs& p, WarpShared& ws,
                                          uint32_t a, Hit& h) {
    const GridView& g = B.g;
    const double ax = __ldg(A.x + a), ay = __ldg(A.y + a), az = __ldg(A.z + a);
    const float2 pf = __ldg(A.pos + a);
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
        scan_range<MODE>(A, B, p, ws, a, ax, ay, az, __ldg(B.cell_start + base + k0), __ldg(B.cell_start + base + k1 + 1), h);
        if (k3 >= k2)
            scan_range<MODE>(A, B, p, ws, a, ax, ay, az, __ldg(B.cell_start + base + k2), __ldg(B.cell_start + base + k3 + 1), h);
    }
}

// flush `cnt` (<= 32) queued rows starting at queue slot `first`
__device__ __forceinline__ void flush_rows(const IndexView& A, const IndexView& B, const MatchArgs& p, const WarpShared& ws,
                                           unsigned first, unsigned cnt, int lane) {
    unsigned long long base = 0;
    if (lane == 0) base = atomicAdd(p.count, (unsigned long long)cnt);
    base = __shfl_sync(kFull, base, 0);
    if ((unsigned)lane < cnt) {
        const unsigned k = first + lane;
        const unsigned long long o = base + lane;
        if (o < p.capacity) {
            p.out_ida[o] = __ldg(A.id + ws.q_a[k]); p.out_idb[o] = __ldg(B.id + ws.q_b[k]);
            p.out_sep[o] = sep_from_chord2(ws.q_c2[k]);
        }
    }
}

// after a scan: append the lanes' first hits behind whatever the scan pushed, flush full groups of 32.
// `row` is the A row this lane scanned.  Returns the new queue length (warp-uniform, < 32).
__device__ __forceinline__ unsigned collect(const IndexView& A, const IndexView& B, const MatchArgs& p, WarpShared& ws,
                                            uint32_t row, const Hit& h, int lane) {
    __syncwarp();
    unsigned qn = min(ws.q_n, (unsigned)kQSoft);
    const unsigned m = __ballot_sync(kFull, h.has);
    if (h.has) {
        const unsigned k = qn + __popc(m & ((1u << lane) - 1u));
        ws.q_a[k] = row; ws.q_b[k] = h.j; ws.q_c2[k] = h.c2;
    }
    qn += __popc(m);
    __syncwarp();
    while (qn >= 32) { qn -= 32; flush_rows(A, B, p, ws, qn, 32, lane); }
    __syncwarp();
    if (lane == 0) ws.q_n = qn;
    __syncwarp();
    return qn;
}

template <int MODE>
__global__ void __launch_bounds__(kMatchThreads)
k_match(const __grid_constant__ IndexView A, const __grid_constant__ IndexView B, const __grid_constant__ MatchArgs p) {
    __shared__ WarpShared s_ws[kMatchWarps];
    const int lane = threadIdx.x & 31;
    WarpShared& ws = s_ws[threadIdx.x >> 5];
    const GridView& g = B.g;
    if (lane == 0) ws.q_n = 0;
    __syncwarp();
    unsigned dn = 0;                                   // deferred rows pending (warp-uniform)
    const uint32_t warps = gridDim.x * kMatchWarps;
    const unsigned lt = (1u << lane) - 1u;

    for (uint32_t chunk = blockIdx.x * kMatchWarps + (threadIdx.x >> 5); chunk < p.n_chunks; chunk += warps) {
        const uint32_t i = chunk * 32u + lane;
        Hit h; h.has = false; h.j = 0; h.c2 = 0.0;
        bool defer = false;
        if (i < A.n) {
            const double ax = __ldg(A.x + i), ay = __ldg(A.y + i), az = __ldg(A.z + i);
            const float2 pf = __ldg(A.pos + i);
            const double dlo = (double)pf.y - p.pad_dec, dhi = (double)pf.y + p.pad_dec;
            if (!(dhi < g.dec_min) && !(dlo > g.dec_max)) {
                const float fx = (float)ax, fy = (float)ay;
                const float s = p.sin_r_up * rsqrtf(fx * fx + fy * fy);
                const double w = (double)(s * (1.011f * 57.29577951f)) + kEpsRaDeg;
                const double u = box_u(g, (double)pf.x);
                const double ulo = u - w, uhi = u + w;
                const int z = zone_of(g, dlo);
                if (s < 0.25f && z == zone_of(g, dhi) && ulo >= 0.0 && uhi < 360.0 && ulo <= g.span) {
                    const int n = __ldg(g.n_ra + z);
                    const uint32_t* cs = B.cell_start + __ldg(g.cell_base + z);
                    const uint32_t j0 = __ldg(cs + cell_of_u(g, ulo, n)), j1 = __ldg(cs + cell_of_u(g, uhi, n) + 1);
                    scan_range<MODE>(A, B, p, ws, i, ax, ay, az, j0, j1, h);
                } else defer = true;
            }
        }
        collect(A, B, p, ws, i, h, lane);
        const unsigned md = __ballot_sync(kFull, defer);
        if (md) {
            if (defer) ws.defer[dn + __popc(md & lt)] = i;
            dn += __popc(md);
            __syncwarp();
            if (dn >= 32) {
                dn -= 32;
                const uint32_t a = ws.defer[dn + lane];
                Hit hg; hg.has = false; hg.j = 0; hg.c2 = 0.0;
                scan_general<MODE>(A, B, p, ws, a, hg);
                collect(A, B, p, ws, a, hg, lane);
            }
        }
    }
    // drain: the remaining deferred rows, then the remaining queued rows
    {
        uint32_t a = 0;
        Hit hg; hg.has = false; hg.j = 0; hg.c2 = 0.0;
        if ((unsigned)lane < dn) { a = ws.defer[lane]; scan_general<MODE>(A, B, p, ws, a, hg); }
        const unsigned qn = collect(A, B, p, ws, a, hg, lane);
        if (qn) flush_rows(A, B, p, ws, 0, qn, lane);
    }
}

size_t match_temp_bytes(const IndexView&, const IndexView&) { return 0; }

void launch_match(const IndexView& A, const IndexView& B, double radius_arcsec, int mode,
                  int64_t* out_ida, int64_t* out_idb, double* out_sep, unsigned long long capacity,
                  unsigned long long* d_count, void* d_temp, cudaStream_t s) {
    (void)d_temp;
    if (A.n == 0 || B.n == 0) return;
    MatchArgs p;
    long double r_rad = (long double)radius_arcsec * (3.141592653589793238462643383279502884L / 648000.0L);
    long double hs = sinl(0.5L * r_rad);
    p.thr2 = (double)(4.0L * hs * hs);
    p.pad_dec = radius_arcsec / 3600.0 + kEpsDecDeg;
    p.sin_r_up = (float)((double)sinl(r_rad) * (1.0 + 1e-5));
    p.out_ida = out_ida; p.out_idb = out_idb; p.out_sep = out_sep; p.capacity = capacity; p.count = d_count;
    p.n_chunks = (uint32_t)(((size_t)A.n + 31) / 32);
    static int per_sm[2] = {0, 0};
    const int m = mode == HLC2_NEAREST ? 1 : 0;
    if (!per_sm[m]) {
        int v = 0;
        if (m) cudaOccupancyMaxActiveBlocksPerMultiprocessor(&v, k_match<HLC2_NEAREST>, kMatchThreads, 0);
        else   cudaOccupancyMaxActiveBlocksPerMultiprocessor(&v, k_match<HLC2_ALL_PAIRS>, kMatchThreads, 0);
        per_sm[m] = v > 0 ? v : 4;
    }
    // persistent grid: SM count x resident CTAs, never more warps than chunks
    const size_t want = ((size_t)p.n_chunks + kMatchWarps - 1) / kMatchWarps;
    const unsigned blocks = (unsigned)std::min<size_t>(want, (size_t)sm_count() * per_sm[m]);
    if (m) k_match<HLC2_NEAREST><<<blocks, kMatchThreads, 0, s>>>(A, B, p);
    else   k_match<HLC2_ALL_PAIRS><<<blocks, kMatchThreads, 0, s>>>(A, B, p);
    count_launch();
}

}  // namespace hlc2
