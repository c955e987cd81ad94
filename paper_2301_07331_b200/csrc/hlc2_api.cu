// hlc2_api.cu -- the C ABI of include/hlc2.h: argument checks, buffer layout, the host-side grid
// planner (no per-source CPU work), and the launch sequences of build and crossmatch.
#include <math.h>
#include <stdio.h>
#include <string.h>

#include <algorithm>
#include <atomic>
#include <new>
#include <vector>

#include "hlc2_grid.cuh"

using namespace hlc2;

namespace hlc2 {
static std::atomic<unsigned long long> g_launches{0};
void count_launch(int k) { g_launches.fetch_add((unsigned long long)k, std::memory_order_relaxed); }
static thread_local cudaError_t t_last_cuda = cudaSuccess;
void note_cuda_error(cudaError_t e) { t_last_cuda = e; }      // for the entry points that live in other files
}  // namespace hlc2

#define CU(call)                                                    \
    do {                                                            \
        cudaError_t e__ = (call);                                   \
        if (e__ != cudaSuccess) { hlc2::t_last_cuda = e__; return HLC2_ERR_CUDA; } \
    } while (0)

static inline size_t align_up(size_t v, size_t a = 256) { return (v + a - 1) / a * a; }

// ---- host copy of a grid -------------------------------------------------------------------
struct HostGrid {
    double dec_lo = -90.0, h = 180.0, ra0 = 0.0, span = 360.0, cell_arcsec = 0.0;
    double dec_min = INFINITY, dec_max = -INFINITY;
    int64_t n_zones = 1;
    std::vector<int32_t> n_ra;        // [n_zones]
    std::vector<uint32_t> cell_base;  // [n_zones + 1]
    uint32_t n_cells() const { return cell_base.empty() ? 0u : cell_base.back(); }
};

struct Layout {           // byte offsets inside the index buffer
    size_t x, y, z, id, pos, key, cell_start, n_ra, cell_base, tiles, n_tiles, stats, err2, total;   // err2 = 0: no error radii
    size_t cap_cells, cap_zones, cap_tiles, n_pad;
};
struct TempLayout { size_t key_b, perm_a, perm_b, rec, digit_hist, digit_base, ticket, status, big, tile_first, total; };

struct hlc2_index {
    uint32_t magic;
    int64_t n;
    hlc2_opts opts;
    HostGrid grid;
    Layout lay;
    char* d_buf;
    size_t index_bytes;
    cudaStream_t stream;
    int device;
    Stats h_stats;        // copy of the extent pass
    bool stats_valid;
    Stats* d_stats;       // device copy of the status record (read lazily after an asynchronous build)
    bool outside_box;     // asynchronous build: some source lies outside the grid's RA box
    bool flagged;         // the sorted keys carry window flags in their top bits (grids of <= 2^28 cells)
};
static const uint32_t kMagic = 0x484C4332u;   // "HLC2"

static bool opts_ok(const hlc2_opts* o) {
    if (!o) return true;
    if (!(o->r_max_arcsec > 0.0) || !(o->r_max_arcsec <= 36000.0)) return false;
    if (!(o->target_occupancy >= 0.0) || !std::isfinite(o->target_occupancy)) return false;
    if (!(o->cell_arcsec >= 0.0) || !std::isfinite(o->cell_arcsec)) return false;
    if (o->grid_like && o->grid_like->magic != kMagic) return false;
    if (o->zone_aspect < 0 || o->zone_aspect > 64) return false;
    return true;
}
// target_occupancy 0 = automatic: cells as fine as the radix sort allows for free.  Finer cells of the scanned
// catalogue mean fewer candidates per source in the match (config 3: occupancy 0.5 instead of 1 takes 7 % off the match),
// but a cell count that needs one more key digit costs a whole extra sort pass in the build; so take the finest
// occupancy in [0.4, 1] whose cell count still fits the digits that occupancy 1 needs.
static double auto_occupancy(int64_t n) {
    if (n <= 0) return 1.0;
    int bits = 1; while (bits < 32 && (1ull << bits) < (unsigned long long)n) ++bits;      // key bits at occupancy 1
    const int passes = std::max(1, (bits + kRadixBits - 1) / kRadixBits);
    const double max_cells = std::ldexp(1.0, std::min(32, passes * kRadixBits));
    return std::min(1.0, std::max(0.4, 1.15 * (double)n / max_cells));
}
static hlc2_opts opts_or_default(const hlc2_opts* o, int64_t n) {
    hlc2_opts d; memset(&d, 0, sizeof d); d.r_max_arcsec = 1.0;
    if (o) d = *o;
    if (d.target_occupancy == 0.0) d.target_occupancy = auto_occupancy(n);
    if (d.target_occupancy < 0.05) d.target_occupancy = 0.05;
    return d;
}

static const double kSphereArcsec2 = 4.0 * M_PI * 206264.80624709636 * 206264.80624709636;

static void caps(int64_t n, const hlc2_opts& o, size_t* cap_cells, size_t* cap_zones) {
    if (o.grid_like) { *cap_cells = o.grid_like->grid.n_cells(); *cap_zones = (size_t)o.grid_like->grid.n_zones; return; }
    double cell = std::max(o.cell_arcsec, 0.0);
    if (cell > 0.0) {
        cell = std::max(cell, o.r_max_arcsec);
        size_t zones = (size_t)ceil(648000.0 / cell) + 2;
        *cap_zones = zones;
        // an explicit cell size is honoured up to a table budget of max(16 n, 2^25) cells; beyond that the
        // planner coarsens the cells until the table fits
        double full = kSphereArcsec2 / (cell * cell) * 1.01 + (double)zones + 16.0;
        double budget = std::max(16.0 * (double)n, 33554432.0);
        *cap_cells = (size_t)std::min(full, budget);
    } else {
        *cap_cells = (size_t)ceil((double)n / o.target_occupancy * 1.25) + 4096;
        *cap_zones = std::min<size_t>(*cap_cells, (size_t)1 << 20);
    }
}

static Layout make_layout(int64_t n, const hlc2_opts& o) {
    Layout L; caps(n, o, &L.cap_cells, &L.cap_zones);
    L.n_pad = align_up((size_t)n, 64) + 64;
    size_t off = 0;
    L.x = off; off += align_up(L.n_pad * 8);
    L.y = off; off += align_up(L.n_pad * 8);
    L.z = off; off += align_up(L.n_pad * 8);
    L.id = off; off += align_up(L.n_pad * 8);
    L.pos = off; off += align_up(L.n_pad * 8);
    L.key = off; off += align_up(L.n_pad * 4);
    L.cell_start = off; off += align_up((L.cap_cells + 1) * 4 + 64);   // slack: bulk copies round up to 16 bytes
    L.n_ra = off; off += align_up(L.cap_zones * 4);
    L.cell_base = off; off += align_up((L.cap_zones + 1) * 4);
    L.cap_tiles = (size_t)n / kTile + L.cap_zones + 1;
    L.tiles = off; off += align_up(L.cap_tiles * sizeof(TileDesc));
    L.n_tiles = off; off += 256;
    L.stats = off; off += align_up(sizeof(Stats));
    L.err2 = 0;
    if (o.d_err_arcsec) { L.err2 = off; off += align_up(L.n_pad * 8); }
    L.total = off;
    return L;
}
static TempLayout make_temp(int64_t n, const Layout& L) {
    TempLayout T; size_t off = 0;
    T.key_b = off; off += align_up(L.n_pad * 4);
    T.perm_a = off; off += align_up(L.n_pad * 4);
    T.perm_b = off; off += align_up(L.n_pad * 4);
    T.rec = off; off += align_up(L.n_pad * sizeof(Rec));
    T.digit_hist = off; off += align_up((size_t)kMaxPasses * kRadix * 4);
    T.digit_base = off; off += align_up((size_t)kMaxPasses * kRadix * 4);
    T.ticket = off; off += 256;
    T.status = off; off += align_up((size_t)kMaxPasses * sort_tiles((uint32_t)n) * kRadix * 4 + 256);
    T.big = off; off += align_up((3 * cell_big_cap(L.cap_cells) + 1) * 4);
    T.tile_first = off; off += align_up((L.cap_zones + 2) * 4);
    T.total = off;
    return T;
}

namespace hlc2 {
size_t match_temp_bound(int64_t n_a, const hlc2_opts* opts) {
    hlc2_opts o = opts_or_default(opts, n_a);
    o.grid_like = nullptr;
    Layout L = make_layout(n_a, o);
    return std::max(match_temp_for_tiles(L.cap_tiles), (size_t)256 + (size_t)n_a * sizeof(uint32_t));
}
}  // namespace hlc2

// ---- the planner: grid from the catalogue's extent and density (host, O(n_zones)) ----------
static void fill_zones(HostGrid& g, double c_arcsec) {
    const double c_rad = c_arcsec / 206264.80624709636;
    const double span_rad = g.span * (M_PI / 180.0);
    g.n_ra.resize((size_t)g.n_zones); g.cell_base.resize((size_t)g.n_zones + 1);
    uint64_t acc = 0;
    for (int64_t z = 0; z < g.n_zones; ++z) {
        double lo = g.dec_lo + (double)z * g.h, hi = g.dec_lo + (double)(z + 1) * g.h;
        double worst = std::min(90.0, std::max(fabs(lo), fabs(hi)));       // poleward edge: narrowest arc
        double n = floor(span_rad * cos(worst * (M_PI / 180.0)) / c_rad);
        int32_t k = (int32_t)std::min(std::max(n, 1.0), 1073741824.0);
        g.n_ra[(size_t)z] = k; g.cell_base[(size_t)z] = (uint32_t)std::min<uint64_t>(acc, 0xFFFFFFFFull);
        acc += (uint64_t)k;
    }
    g.cell_base[(size_t)g.n_zones] = (uint32_t)std::min<uint64_t>(acc, 0xFFFFFFFFull);
}

static void plan_grid(const Stats& st, int64_t n_valid, const hlc2_opts& o, size_t cap_cells, size_t cap_zones, HostGrid& g) {
    g = HostGrid();
    if (n_valid > 0) { g.dec_min = f64_from_order_bits(st.dec_min_bits); g.dec_max = f64_from_order_bits(st.dec_max_bits); }
    double dec_lo = -90.0, range = 180.0;
    g.ra0 = 0.0; g.span = 360.0;
    if (!o.full_sky && n_valid > 0) {
        dec_lo = g.dec_min; range = g.dec_max - g.dec_min;
        // largest circular run of empty coarse RA bins
        int best_len = 0, best_start = 0, run = 0;
        for (int i = 0; i < 2 * kRaBins; ++i) {
            if (st.ra_hist[i % kRaBins] == 0) { ++run; if (run > best_len && run <= kRaBins) { best_len = run; best_start = i - run + 1; } }
            else run = 0;
        }
        if (best_len >= 8 && best_len < kRaBins) {
            int first_occ = (best_start + best_len) % kRaBins;          // first occupied bin after the gap
            int occ_bins = kRaBins - best_len;
            g.ra0 = (double)((first_occ - 1 + kRaBins) % kRaBins) * kRaBinDeg;      // one guard bin either side
            g.span = (double)(occ_bins + 2) * kRaBinDeg;
        }
    }
    // fine-cell size: density-derived, never below r_max ("cells sized to r", NS (a))
    double c = o.cell_arcsec;
    if (!(c > 0.0)) {
        double area = kSphereArcsec2;
        if (!o.full_sky && n_valid > 0) {
            double s1 = sin(std::min(90.0, g.dec_max) * (M_PI / 180.0)), s0 = sin(std::max(-90.0, g.dec_min) * (M_PI / 180.0));
            area = std::max(g.span * 3600.0 * (s1 - s0) * 206264.80624709636, 1.0);
        }
        c = sqrt(o.target_occupancy * area / (double)std::max<int64_t>(n_valid, 1));
    }
    c = std::max(c, o.r_max_arcsec);
    c = std::min(c, 648000.0);
    double ra_contrast = 1.0;
    if (n_valid > 0) {
        uint64_t occ = 0, mx = 0;
        for (int i = 0; i < kRaBins; ++i) { if (st.ra_hist[i]) ++occ; mx = std::max<uint64_t>(mx, st.ra_hist[i]); }
        if (occ) ra_contrast = (double)mx * (double)occ / (double)n_valid;
    }
    for (int iter = 0; iter < 2000; ++iter) {
        // zones `aspect` times as high as the cell size, RA cells that much narrower (never below r_max): same cell area,
        // but a search window leaves its zone (the expensive neighbour) aspect times less often
        // automatic: RA cells three r_max wide (measured on config 3: the match time falls until about there) -- unless the
        // catalogue is concentrated in RA (a dense strip along a meridian, config 4's seam): tall cells would then hold
        // the whole strip's height.  The coarse RA histogram of the extent pass tells: contrast = fullest bin / mean
        // occupied bin; beyond 4 the aspect is scaled back in proportion (config 3: 1.3 -> 24; config 4: 200 -> 1).
        double want = (double)o.zone_aspect;
        if (o.zone_aspect <= 0) {
            want = std::min(32.0, floor(c / (3.0 * o.r_max_arcsec)));
            if (ra_contrast > 4.0) want = floor(want * 4.0 / ra_contrast);
        }
        const double aspect = std::max(1.0, std::min(want, c / o.r_max_arcsec));
        double zh_deg = std::min(c * aspect, 648000.0) / 3600.0;
        double rng = std::max(range, zh_deg);
        int64_t nz = std::max<int64_t>(1, (int64_t)floor(rng / zh_deg));
        g.n_zones = nz; g.h = rng / (double)nz; g.dec_lo = dec_lo; g.cell_arcsec = c;
        if ((size_t)nz <= cap_zones) {
            fill_zones(g, c / aspect);
            uint64_t tot = 0; for (int32_t k : g.n_ra) tot += (uint64_t)k;
            if (tot <= cap_cells && tot < 0xFFFFFFF0ull) return;
        }
        c *= 1.05;
    }
}

static GridView grid_view(const hlc2_index* ix) {
    GridView v;
    v.n_ra = (const int32_t*)(ix->d_buf + ix->lay.n_ra);
    v.cell_base = (const uint32_t*)(ix->d_buf + ix->lay.cell_base);
    v.dec_lo = ix->grid.dec_lo; v.h = ix->grid.h; v.inv_h = 1.0 / ix->grid.h; v.ra0 = ix->grid.ra0; v.span = ix->grid.span;
    v.inv_span = 1.0 / ix->grid.span; v.dec_min = ix->grid.dec_min; v.dec_max = ix->grid.dec_max;
    v.n_zones = (int32_t)ix->grid.n_zones; v.n_cells = ix->grid.n_cells();
    return v;
}
static IndexView index_view(const hlc2_index* ix) {
    IndexView v;
    v.x = (const double*)(ix->d_buf + ix->lay.x); v.y = (const double*)(ix->d_buf + ix->lay.y);
    v.z = (const double*)(ix->d_buf + ix->lay.z); v.id = (const int64_t*)(ix->d_buf + ix->lay.id);
    v.pos = (const float2*)(ix->d_buf + ix->lay.pos);
    v.err2 = ix->lay.err2 ? (const double*)(ix->d_buf + ix->lay.err2) : nullptr;
    v.key = (const uint32_t*)(ix->d_buf + ix->lay.key); v.key_mask = ix->flagged ? kKeyMask : 0xFFFFFFFFu;
    v.cell_start = (const uint32_t*)(ix->d_buf + ix->lay.cell_start);
    v.tiles = (const TileDesc*)(ix->d_buf + ix->lay.tiles); v.n_tiles = (const uint32_t*)(ix->d_buf + ix->lay.n_tiles);
    v.g = grid_view(ix); v.n = (uint32_t)ix->n;
    v.tile_cap = (uint32_t)((size_t)ix->n / kTile + (size_t)ix->grid.n_zones + 1);
    return v;
}

// do two indices share one grid (same zones, same cells, same box)?  Then a source's cell key means the same in both and
// A's window flags select its cells (hlc2_match_same.cu).  That path hands every row within r_max of a zone edge to
// its per-lane edge kernel, which pays off while such rows are few: zones at least 4 r_max high (else the general
// path, which stages all three zones, is the better one).
static bool same_grid(const hlc2_index* a, const hlc2_index* b) {
    const HostGrid& x = a->grid; const HostGrid& y = b->grid;
    return a->flagged && b->flagged && x.n_zones == y.n_zones && x.dec_lo == y.dec_lo && x.h == y.h && x.ra0 == y.ra0 &&
           x.span == y.span && x.n_ra == y.n_ra && 4.0 * a->opts.r_max_arcsec / 3600.0 <= x.h;
}

// does every occupied coarse RA bin of `st` lie inside grid g's RA box?
static bool ra_box_covers(const HostGrid& g, const Stats& st) {
    if (g.span >= 360.0) return true;
    for (int b = 0; b < kRaBins; ++b) {
        if (!st.ra_hist[b]) continue;
        double lo = (double)b * kRaBinDeg - g.ra0; if (lo < 0.0) lo += 360.0;
        if (lo + kRaBinDeg > g.span) return false;
    }
    return true;
}

extern "C" {

int hlc2_index_sizes(int64_t n, const hlc2_opts* opts, size_t* index_bytes, size_t* temp_bytes) {
    if (n < 0 || !opts_ok(opts) || (!index_bytes && !temp_bytes)) return HLC2_ERR_INVALID_ARG;
    if ((uint64_t)n > kMaxN) return HLC2_ERR_TOO_MANY;
    hlc2_opts o = opts_or_default(opts, n);
    Layout L = make_layout(n, o);
    TempLayout T = make_temp(n, L);
    if (index_bytes) *index_bytes = L.total;
    if (temp_bytes) *temp_bytes = T.total;
    return HLC2_OK;
}

int hlc2_build_index(const double* d_ra, const double* d_dec, const int64_t* d_id, int64_t n,
                     const hlc2_opts* opts, void* d_index_buf, size_t index_bytes,
                     void* d_temp, size_t temp_bytes, void* cuda_stream, hlc2_index** out) {
    if (!out) return HLC2_ERR_INVALID_ARG;
    *out = nullptr;
    if (n < 0 || !opts_ok(opts) || !d_index_buf || !d_temp || (n > 0 && (!d_ra || !d_dec))) return HLC2_ERR_INVALID_ARG;
    if ((uint64_t)n > kMaxN) return HLC2_ERR_TOO_MANY;
    hlc2_opts o = opts_or_default(opts, n);
    Layout L = make_layout(n, o);
    TempLayout T = make_temp(n, L);
    if (index_bytes < L.total || temp_bytes < T.total) return HLC2_ERR_BUFFER_TOO_SMALL;
    cudaStream_t s = (cudaStream_t)cuda_stream;

    hlc2_index* ix = new (std::nothrow) hlc2_index();
    if (!ix) return HLC2_ERR_INVALID_ARG;
    ix->magic = kMagic; ix->n = n; ix->opts = o; ix->opts.grid_like = nullptr; ix->opts.d_err_arcsec = nullptr; ix->lay = L;
    ix->d_buf = (char*)d_index_buf; ix->index_bytes = index_bytes; ix->stream = s; ix->stats_valid = false;
    ix->d_stats = nullptr; ix->outside_box = false;
    int rc = HLC2_OK;
    auto fail = [&](int code) { delete ix; return code; };
    if (cudaGetDevice(&ix->device) != cudaSuccess) { t_last_cuda = cudaGetLastError(); return fail(HLC2_ERR_CUDA); }

    char* buf = ix->d_buf; char* tmp = (char*)d_temp;
    Stats* d_stats = (Stats*)(buf + L.stats);
    uint32_t nn = (uint32_t)n;

    const bool async_like = o.grid_like && o.async_like;
    Stats* collect = nullptr;
    int64_t n_valid = n;
    if (async_like) {
        // the grid is given: no extent pass, no synchronisation.  k_keys_pack gathers the status record on the way
        // (read by hlc2_index_status).  The declination extent only prunes windows in the two-grid planner, so the
        // whole sphere (a superset) stands in for it; sources beyond the end zones are filed in them, as always.
        launch_stats_init(d_stats, s);
        collect = d_stats;
        ix->d_stats = d_stats;
        ix->grid = o.grid_like->grid;
        ix->grid.dec_min = -90.0; ix->grid.dec_max = 90.0;
    } else {
        // (a1) extent pass, then plan the grid on the host (one small D2H + sync)
        launch_stats(d_ra, d_dec, nn, d_stats, s);
        if (cudaMemcpyAsync(&ix->h_stats, d_stats, sizeof(Stats), cudaMemcpyDeviceToHost, s) != cudaSuccess ||
            cudaStreamSynchronize(s) != cudaSuccess) { t_last_cuda = cudaGetLastError(); return fail(HLC2_ERR_CUDA); }
        ix->stats_valid = true;
        n_valid = n - (int64_t)ix->h_stats.n_bad;
    }
    if (async_like) {
        // nothing to plan
    } else if (o.grid_like) {
        ix->grid = o.grid_like->grid;
        if (n_valid > 0) {
            ix->grid.dec_min = f64_from_order_bits(ix->h_stats.dec_min_bits);
            ix->grid.dec_max = f64_from_order_bits(ix->h_stats.dec_max_bits);
            if (!ra_box_covers(ix->grid, ix->h_stats)) return fail(HLC2_ERR_GRID_MISMATCH);
        } else { ix->grid.dec_min = INFINITY; ix->grid.dec_max = -INFINITY; }
    } else {
        plan_grid(ix->h_stats, n_valid, o, L.cap_cells, L.cap_zones, ix->grid);
    }
    const HostGrid& g = ix->grid;
    if ((size_t)g.n_zones > L.cap_zones || (size_t)g.n_cells() > L.cap_cells) return fail(HLC2_ERR_BUFFER_TOO_SMALL);
    // zone tables: from the host plan, or (asynchronous build) device to device from the index that owns the grid
    const hlc2_index* like = o.grid_like;
    const void* src_n_ra = async_like ? (const void*)(like->d_buf + like->lay.n_ra) : (const void*)g.n_ra.data();
    const void* src_base = async_like ? (const void*)(like->d_buf + like->lay.cell_base) : (const void*)g.cell_base.data();
    const cudaMemcpyKind kind = async_like ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice;
    if (cudaMemcpyAsync(buf + L.n_ra, src_n_ra, (size_t)g.n_zones * 4, kind, s) != cudaSuccess ||
        cudaMemcpyAsync(buf + L.cell_base, src_base, ((size_t)g.n_zones + 1) * 4, kind, s) != cudaSuccess) {
        t_last_cuda = cudaGetLastError(); return fail(HLC2_ERR_CUDA);
    }
    GridView gv = grid_view(ix);

    // (a1) keys + packed records + digit counts -> (a2) radix sort (key, row) -> (a3) gather -> (a4) cell table, tiles
    uint32_t n_cells = g.n_cells();
    ix->flagged = n_cells <= (1u << kKeyFlagShift);
    const uint32_t kmask = ix->flagged ? kKeyMask : 0xFFFFFFFFu;
    int key_bits = 1; while (key_bits < 32 && (1ull << key_bits) < (unsigned long long)n_cells) ++key_bits;
    int passes = radix_passes(key_bits);
    uint32_t* key_idx = (uint32_t*)(buf + L.key);           // the sorted keys must end up here
    uint32_t* key_tmp = (uint32_t*)(tmp + T.key_b);
    uint32_t* ka = (passes & 1) ? key_tmp : key_idx;        // start buffer chosen by pass parity
    uint32_t* kb = (passes & 1) ? key_idx : key_tmp;
    uint32_t* pa = (uint32_t*)(tmp + T.perm_a); uint32_t* pb = (uint32_t*)(tmp + T.perm_b);
    Rec* rec = (Rec*)(tmp + T.rec);
    uint32_t* digit_hist = (uint32_t*)(tmp + T.digit_hist);
    if (cudaMemsetAsync(digit_hist, 0, (size_t)kMaxPasses * kRadix * 4, s) != cudaSuccess) { t_last_cuda = cudaGetLastError(); return fail(HLC2_ERR_CUDA); }
    launch_keys_pack(d_ra, d_dec, d_id, nn, gv, passes, o.r_max_arcsec, ix->flagged, ka, rec, digit_hist, s, collect);
    int where = launch_radix_sort(ka, kb, pa, pb, nn, key_bits, digit_hist, (uint32_t*)(tmp + T.digit_base),
                                  (uint32_t*)(tmp + T.status), (uint32_t*)(tmp + T.ticket), s);
    const uint32_t* perm = where ? pb : pa;
    launch_gather(rec, perm, nn, (double*)(buf + L.x), (double*)(buf + L.y), (double*)(buf + L.z), (int64_t*)(buf + L.id), (float2*)(buf + L.pos), s);
    if (L.err2) launch_gather_err2(o.d_err_arcsec, perm, nn, (double*)(buf + L.err2), s);
    launch_cell_table(key_idx, kmask, nn, n_cells, (uint32_t*)(buf + L.cell_start), (uint32_t*)(tmp + T.big), s);
    launch_tiles((const uint32_t*)(buf + L.cell_start), gv.cell_base, gv.n_ra, (uint32_t)g.n_zones, key_idx, kmask,
                 (uint32_t)((size_t)n / kTile + (size_t)g.n_zones + 1), (uint32_t*)(tmp + T.tile_first),
                 (TileDesc*)(buf + L.tiles), (uint32_t*)(buf + L.n_tiles), s);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) { t_last_cuda = e; return fail(HLC2_ERR_CUDA); }
    // the host grid vectors were copied with cudaMemcpyAsync from pageable memory: that call
    // returns after staging the source, so the vectors may be reused immediately.
    *out = ix;
    return rc;
}

int hlc2_index_status(const hlc2_index* idx, int64_t* first_bad_row) {
    if (!idx || idx->magic != kMagic) return HLC2_ERR_INVALID_ARG;
    CU(cudaStreamSynchronize(idx->stream));
    CU(cudaGetLastError());
    if (first_bad_row) *first_bad_row = -1;
    if (idx->d_stats) {       // asynchronous build: the record lives on the device (re-read: a graph replay rewrites it)
        hlc2_index* ix = const_cast<hlc2_index*>(idx);
        CU(cudaMemcpy(&ix->h_stats, idx->d_stats, sizeof(Stats), cudaMemcpyDeviceToHost));
        ix->stats_valid = true; ix->outside_box = ix->h_stats.ra_hist[0] != 0;
    }
    if (idx->outside_box) return HLC2_ERR_GRID_MISMATCH;
    if (idx->stats_valid && idx->h_stats.n_bad) {
        if (first_bad_row) *first_bad_row = (int64_t)idx->h_stats.first_bad_row;
        return HLC2_ERR_BAD_COORD;
    }
    return HLC2_OK;
}

int hlc2_grid_describe(const hlc2_index* idx, hlc2_grid_info* info, const int32_t** h_n_ra) {
    if (!idx || idx->magic != kMagic || (!info && !h_n_ra)) return HLC2_ERR_INVALID_ARG;
    if (info) {
        info->dec_lo_deg = idx->grid.dec_lo; info->zone_height_deg = idx->grid.h; info->n_zones = idx->grid.n_zones;
        info->ra0_deg = idx->grid.ra0; info->ra_span_deg = idx->grid.span; info->n_cells = idx->grid.n_cells();
        info->cell_arcsec = idx->grid.cell_arcsec; info->n = idx->n;
    }
    if (h_n_ra) *h_n_ra = idx->grid.n_ra.data();
    return HLC2_OK;
}

int hlc2_index_arrays(const hlc2_index* idx, const double** d_x, const double** d_y, const double** d_z,
                      const int64_t** d_id, const uint32_t** d_cell_start, const uint32_t** d_cell_key,
                      int64_t* n, int64_t* n_cells) {
    if (!idx || idx->magic != kMagic) return HLC2_ERR_INVALID_ARG;
    const Layout& L = idx->lay; const char* b = idx->d_buf;
    if (d_x) *d_x = (const double*)(b + L.x);
    if (d_y) *d_y = (const double*)(b + L.y);
    if (d_z) *d_z = (const double*)(b + L.z);
    if (d_id) *d_id = (const int64_t*)(b + L.id);
    if (d_cell_start) *d_cell_start = (const uint32_t*)(b + L.cell_start);
    if (d_cell_key) *d_cell_key = (const uint32_t*)(b + L.key);
    if (n) *n = idx->n;
    if (n_cells) *n_cells = idx->grid.n_cells();
    return HLC2_OK;
}

int hlc2_crossmatch_sizes(const hlc2_index* A, const hlc2_index* B, size_t* temp_bytes) {
    if (!A || !B || A->magic != kMagic || B->magic != kMagic || !temp_bytes) return HLC2_ERR_INVALID_ARG;
    *temp_bytes = match_temp_bytes(index_view(A), index_view(B));
    return HLC2_OK;
}

int hlc2_crossmatch_events(const hlc2_index* A, const hlc2_index* B, double radius_arcsec, int mode,
                           int64_t* d_out_idA, int64_t* d_out_idB, double* d_out_sep, int64_t capacity,
                           unsigned long long* d_count, void* d_temp, size_t temp_bytes, void* cuda_stream,
                           void* ev_kernel_start, void* ev_kernel_stop) {
    if (!A || !B || A->magic != kMagic || B->magic != kMagic || !d_count || capacity < 0 ||
        (capacity > 0 && (!d_out_idA || !d_out_idB || !d_out_sep)) ||
        (mode != HLC2_ALL_PAIRS && mode != HLC2_NEAREST) ||
        !(radius_arcsec > 0.0) || !std::isfinite(radius_arcsec)) return HLC2_ERR_INVALID_ARG;
    if (radius_arcsec > std::min(A->opts.r_max_arcsec, B->opts.r_max_arcsec)) return HLC2_ERR_RADIUS_TOO_LARGE;
    IndexView va = index_view(A), vb = index_view(B);
    size_t need = match_temp_bytes(va, vb);
    if (need > 0 && (!d_temp || temp_bytes < need)) return HLC2_ERR_BUFFER_TOO_SMALL;
    cudaStream_t s = (cudaStream_t)cuda_stream;
    CU(cudaMemsetAsync(d_count, 0, sizeof(unsigned long long), s));
    launch_match(va, vb, radius_arcsec, mode, d_out_idA, d_out_idB, d_out_sep,
                 (unsigned long long)capacity, d_count, d_temp, s, same_grid(A, B) ? kMatchSameGrid : 0u,
                 (cudaEvent_t)ev_kernel_start, (cudaEvent_t)ev_kernel_stop);
    CU(cudaGetLastError());
    return HLC2_OK;
}

static int match_extra(const hlc2_index* A, const hlc2_index* B, double radius_arcsec, int mode, const MatchExtra& ex,
                       int64_t* d_out_idA, int64_t* d_out_idB, double* d_out_sep, int64_t capacity,
                       unsigned long long* d_count, void* d_temp, size_t temp_bytes, void* cuda_stream) {
    if (!A || !B || A->magic != kMagic || B->magic != kMagic || !d_count || capacity < 0 ||
        (capacity > 0 && (!d_out_idA || !d_out_idB || !d_out_sep)) ||
        (mode != HLC2_ALL_PAIRS && mode != HLC2_NEAREST) ||
        !(radius_arcsec > 0.0) || !std::isfinite(radius_arcsec)) return HLC2_ERR_INVALID_ARG;
    if (radius_arcsec > std::min(A->opts.r_max_arcsec, B->opts.r_max_arcsec)) return HLC2_ERR_RADIUS_TOO_LARGE;
    IndexView va = index_view(A), vb = index_view(B);
    if (ex.k_factor > 0.0 && (!va.err2 || !vb.err2)) return HLC2_ERR_INVALID_ARG;
    size_t need = match_temp_bytes(va, vb);
    if (need > 0 && (!d_temp || temp_bytes < need)) return HLC2_ERR_BUFFER_TOO_SMALL;
    cudaStream_t s = (cudaStream_t)cuda_stream;
    CU(cudaMemsetAsync(d_count, 0, sizeof(unsigned long long), s));
    launch_match(va, vb, radius_arcsec, mode, d_out_idA, d_out_idB, d_out_sep, (unsigned long long)capacity, d_count,
                 d_temp, s, same_grid(A, B) ? kMatchSameGrid : 0u, nullptr, nullptr, &ex);
    CU(cudaGetLastError());
    return HLC2_OK;
}

int hlc2_selfmatch(const hlc2_index* idx, double radius_arcsec, int mode, int include_self,
                   int64_t* d_out_idA, int64_t* d_out_idB, double* d_out_sep, int64_t capacity,
                   unsigned long long* d_count, void* d_temp, size_t temp_bytes, void* cuda_stream) {
    MatchExtra ex; ex.k_factor = 0.0;
    ex.self_mode = mode == HLC2_NEAREST ? 3 : (include_self ? 2 : 1);
    return match_extra(idx, idx, radius_arcsec, mode, ex, d_out_idA, d_out_idB, d_out_sep, capacity, d_count, d_temp, temp_bytes, cuda_stream);
}

int hlc2_crossmatch_radii(const hlc2_index* A, const hlc2_index* B, double radius_cap_arcsec, double k_factor, int mode,
                          int64_t* d_out_idA, int64_t* d_out_idB, double* d_out_sep, int64_t capacity,
                          unsigned long long* d_count, void* d_temp, size_t temp_bytes, void* cuda_stream) {
    if (!(k_factor > 0.0) || !std::isfinite(k_factor)) return HLC2_ERR_INVALID_ARG;
    MatchExtra ex; ex.self_mode = 0; ex.k_factor = k_factor;
    return match_extra(A, B, radius_cap_arcsec, mode, ex, d_out_idA, d_out_idB, d_out_sep, capacity, d_count, d_temp, temp_bytes, cuda_stream);
}

int hlc2_crossmatch(const hlc2_index* A, const hlc2_index* B, double radius_arcsec, int mode,
                    int64_t* d_out_idA, int64_t* d_out_idB, double* d_out_sep, int64_t capacity,
                    unsigned long long* d_count, void* d_temp, size_t temp_bytes, void* cuda_stream) {
    return hlc2_crossmatch_events(A, B, radius_arcsec, mode, d_out_idA, d_out_idB, d_out_sep, capacity, d_count,
                                  d_temp, temp_bytes, cuda_stream, nullptr, nullptr);
}

void hlc2_index_destroy(hlc2_index* idx) {
    if (idx && idx->magic == kMagic) { idx->magic = 0; delete idx; }
}

const char* hlc2_strerror(int status) {
    switch (status) {
        case HLC2_OK: return "ok";
        case HLC2_ERR_INVALID_ARG: return "invalid argument";
        case HLC2_ERR_RADIUS_TOO_LARGE: return "radius larger than the r_max the indices were built for";
        case HLC2_ERR_BUFFER_TOO_SMALL: return "buffer smaller than the size query reports";
        case HLC2_ERR_BAD_COORD: return "non-finite coordinate or |dec| > 90 in the catalogue";
        case HLC2_ERR_CUDA: return "CUDA runtime error (see hlc2_last_cuda_error)";
        case HLC2_ERR_GRID_MISMATCH: return "catalogue does not fit inside the grid_like index's RA box";
        case HLC2_ERR_TOO_MANY: return "too many sources for one index (>= 2^30)";
        case HLC2_ERR_STATIC_LIMIT: return "hlc2_crossmatch_static: the match needs more scratch than the static array holds (HLC2_STATIC_SCRATCH_BYTES = 8 MiB, about 2 million A rows); use hlc2_crossmatch with a caller buffer";
        default: return "unknown status";
    }
}

int hlc2_last_cuda_error(const char** message) {
    if (message) *message = cudaGetErrorString(hlc2::t_last_cuda);
    return (int)hlc2::t_last_cuda;
}

unsigned long long hlc2_kernel_launches(void) { return hlc2::g_launches.load(std::memory_order_relaxed); }

const char* hlc2_version(void) { return "hlc2-b200 0.3 (sm_100a)"; }

}  // extern "C"
