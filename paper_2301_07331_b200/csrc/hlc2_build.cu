// hlc2_build.cu -- index-build kernels (NS (a)): extent statistics, cell keys,
// LSD radix sort of (key, row), gather into SoA unit vectors, cell offset table by scan.
// All kernels are HBM-bound streaming passes; grids are sized in multiples of the SM count.
#include <string.h>
#include <algorithm>

#include "hlc2_grid.cuh"

namespace hlc2 {

static int g_sm_count = 0;
static int sm_count() {
    if (!g_sm_count) {
        int dev = 0; cudaGetDevice(&dev);
        cudaDeviceGetAttribute(&g_sm_count, cudaDevAttrMultiProcessorCount, dev);
        if (g_sm_count <= 0) g_sm_count = 148;
    }
    return g_sm_count;
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

void launch_stats(const double* ra, const double* dec, uint32_t n, Stats* d_stats, cudaStream_t s) {
    k_stats_init<<<(kRaBins + 255) / 256, 256, 0, s>>>(d_stats); count_launch();
    if (n == 0) return;
    int blocks = (int)std::min<size_t>(((size_t)n + kStatsThreads - 1) / kStatsThreads, (size_t)sm_count() * 4);
    k_stats<<<blocks, kStatsThreads, 0, s>>>(ra, dec, n, d_stats); count_launch();
}

// ------------------------------------------------------------------------------------------
// (a1) cell keys
// ------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256)
k_keys(const double* __restrict__ ra, const double* __restrict__ dec, uint32_t n, GridView g, uint32_t* __restrict__ keys) {
    for (size_t i = (size_t)blockIdx.x * 256 + threadIdx.x; i < n; i += (size_t)gridDim.x * 256) {
        double a = __ldg(ra + i), d = __ldg(dec + i);
        uint32_t key = 0;
        if (coord_ok(a, d)) {
            int z = zone_of(g, d);
            int nra = __ldg(g.n_ra + z);
            key = __ldg(g.cell_base + z) + (uint32_t)cell_of_u(g, box_u(g, norm_ra(a)), nra);
        }
        keys[i] = key;
    }
}

void launch_keys(const double* ra, const double* dec, uint32_t n, GridView g, uint32_t* keys, cudaStream_t s) {
    if (n == 0) return;
    int blocks = (int)std::min<size_t>(((size_t)n + 255) / 256, (size_t)sm_count() * 16);
    k_keys<<<blocks, 256, 0, s>>>(ra, dec, n, g, keys); count_launch();
}

// ------------------------------------------------------------------------------------------
// device-wide scan (three kernels: block reduce, scan of partials, block scan with carry-in)
//   Sum, forward, exclusive  -> radix-sort digit offsets
//   Min, reverse, inclusive  -> cell table (next occupied cell's first row)
// ------------------------------------------------------------------------------------------
constexpr int kScanThreads = 256;
constexpr int kScanItems = 16;
constexpr int kScanChunk = kScanThreads * kScanItems;

struct OpSum { static __device__ __forceinline__ uint32_t id() { return 0u; }
               static __device__ __forceinline__ uint32_t ap(uint32_t a, uint32_t b) { return a + b; } };
struct OpMin { static __device__ __forceinline__ uint32_t id() { return 0xFFFFFFFFu; }
               static __device__ __forceinline__ uint32_t ap(uint32_t a, uint32_t b) { return min(a, b); } };

size_t scan_partials_entries(size_t m) { return (m + kScanChunk - 1) / kScanChunk + 1; }

// inclusive scan of one value per thread across the block; returns the inclusive prefix, *total = block aggregate
template <class Op>
__device__ __forceinline__ uint32_t block_scan_incl(uint32_t v, uint32_t* total, uint32_t* sm /*[33]*/) {
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    for (int o = 1; o < 32; o <<= 1) { uint32_t t = __shfl_up_sync(0xffffffffu, v, o); if (lane >= o) v = Op::ap(t, v); }
    if (lane == 31) sm[w] = v;
    __syncthreads();
    if (w == 0) {
        uint32_t t = lane < (int)(blockDim.x >> 5) ? sm[lane] : Op::id();
        for (int o = 1; o < 32; o <<= 1) { uint32_t u = __shfl_up_sync(0xffffffffu, t, o); if (lane >= o) t = Op::ap(u, t); }
        sm[lane] = t;
        if (lane == 31) sm[32] = t;
    }
    __syncthreads();
    if (w > 0) v = Op::ap(sm[w - 1], v);
    *total = sm[32];
    __syncthreads();
    return v;
}

template <class Op, bool Rev>
__global__ void __launch_bounds__(kScanThreads)
k_scan_reduce(const uint32_t* __restrict__ a, size_t m, uint32_t* __restrict__ partials) {
    __shared__ uint32_t sm[33];
    size_t base = (size_t)blockIdx.x * kScanChunk;
    uint32_t acc = Op::id();
#pragma unroll
    for (int r = 0; r < kScanItems; ++r) {
        size_t i = base + (size_t)r * kScanThreads + threadIdx.x;
        if (i < m) acc = Op::ap(acc, a[Rev ? m - 1 - i : i]);
    }
    uint32_t tot; block_scan_incl<Op>(acc, &tot, sm);
    if (threadIdx.x == 0) partials[blockIdx.x] = tot;
}

// single block: partials[b] <- exclusive scan over blocks
template <class Op>
__global__ void __launch_bounds__(1024)
k_scan_partials(uint32_t* __restrict__ partials, size_t nb) {
    __shared__ uint32_t sm[33];
    uint32_t carry = Op::id();
    for (size_t base = 0; base < nb; base += 1024) {
        size_t i = base + threadIdx.x;
        uint32_t v = i < nb ? partials[i] : Op::id();
        uint32_t tot; uint32_t inc = block_scan_incl<Op>(v, &tot, sm);
        // exclusive = carry (op) inclusive-of-previous
        uint32_t prev = __shfl_up_sync(0xffffffffu, inc, 1);
        __shared__ uint32_t last[32];
        if ((threadIdx.x & 31) == 31) last[threadIdx.x >> 5] = inc;
        __syncthreads();
        uint32_t ex = (threadIdx.x & 31) ? prev : (threadIdx.x ? last[(threadIdx.x >> 5) - 1] : Op::id());
        if (i < nb) partials[i] = Op::ap(carry, ex);
        carry = Op::ap(carry, tot);
        __syncthreads();
    }
}

template <class Op, bool Rev, bool Incl>
__global__ void __launch_bounds__(kScanThreads)
k_scan_apply(uint32_t* __restrict__ a, size_t m, const uint32_t* __restrict__ partials) {
    __shared__ uint32_t sm[33];
    // thread t owns kScanItems consecutive logical entries
    size_t base = (size_t)blockIdx.x * kScanChunk + (size_t)threadIdx.x * kScanItems;
    uint32_t v[kScanItems];
    uint32_t acc = Op::id();
#pragma unroll
    for (int r = 0; r < kScanItems; ++r) {
        size_t i = base + r;
        v[r] = i < m ? a[Rev ? m - 1 - i : i] : Op::id();
        acc = Op::ap(acc, v[r]);
    }
    uint32_t tot; uint32_t inc = block_scan_incl<Op>(acc, &tot, sm);
    // exclusive prefix of this thread = inclusive prefix of the previous thread
    __shared__ uint32_t s_inc[kScanThreads];
    s_inc[threadIdx.x] = inc;
    __syncthreads();
    uint32_t run = Op::ap(partials[blockIdx.x], threadIdx.x ? s_inc[threadIdx.x - 1] : Op::id());
#pragma unroll
    for (int r = 0; r < kScanItems; ++r) {
        size_t i = base + r;
        uint32_t nxt = Op::ap(run, v[r]);
        if (i < m) a[Rev ? m - 1 - i : i] = Incl ? nxt : run;
        run = nxt;
    }
}

template <class Op, bool Rev, bool Incl>
static void device_scan(uint32_t* a, size_t m, uint32_t* partials, cudaStream_t s) {
    if (m == 0) return;
    size_t nb = (m + kScanChunk - 1) / kScanChunk;
    k_scan_reduce<Op, Rev><<<(unsigned)nb, kScanThreads, 0, s>>>(a, m, partials);
    k_scan_partials<Op><<<1, 1024, 0, s>>>(partials, nb);
    k_scan_apply<Op, Rev, Incl><<<(unsigned)nb, kScanThreads, 0, s>>>(a, m, partials);
    count_launch(3);
}

// ------------------------------------------------------------------------------------------
// (a2) LSD radix sort of (key, row), 8-bit digits: per-tile digit histogram -> device scan ->
// stable scatter.  Tile = 256 threads x 16 keys; warp w of a tile owns 512 consecutive keys.
// ------------------------------------------------------------------------------------------
constexpr int kSortThreads = 256;
constexpr int kSortItems = 16;
constexpr int kSortTile = kSortThreads * kSortItems;   // 4096
constexpr int kSortWarps = kSortThreads / 32;

size_t sort_counts_entries(uint32_t n) { return 256 * (((size_t)n + kSortTile - 1) / kSortTile); }

__global__ void __launch_bounds__(kSortThreads)
k_sort_hist(const uint32_t* __restrict__ keys, uint32_t n, int shift, uint32_t mask,
            uint32_t* __restrict__ counts, uint32_t n_tiles) {
    __shared__ uint32_t hist[256];
    hist[threadIdx.x] = 0;
    __syncthreads();
    size_t base = (size_t)blockIdx.x * kSortTile;
#pragma unroll
    for (int r = 0; r < kSortItems; ++r) {
        size_t i = base + (size_t)r * kSortThreads + threadIdx.x;
        bool ok = i < n;
        uint32_t d = ok ? ((__ldg(keys + i) >> shift) & mask) : 0xFFFFFFFFu;
        unsigned peers = __match_any_sync(0xffffffffu, d);
        if (ok && (peers & ((1u << (threadIdx.x & 31)) - 1)) == 0) atomicAdd(&hist[d], (uint32_t)__popc(peers));
    }
    __syncthreads();
    counts[(size_t)threadIdx.x * n_tiles + blockIdx.x] = hist[threadIdx.x];
}

template <bool FirstPass>
__global__ void __launch_bounds__(kSortThreads)
k_sort_scatter(const uint32_t* __restrict__ keys, const uint32_t* __restrict__ vals, uint32_t n, int shift, uint32_t mask,
               const uint32_t* __restrict__ offs, uint32_t n_tiles,
               uint32_t* __restrict__ out_keys, uint32_t* __restrict__ out_vals) {
    __shared__ uint32_t wh[kSortWarps][256];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    for (int i = threadIdx.x; i < kSortWarps * 256; i += kSortThreads) (&wh[0][0])[i] = 0;
    __syncthreads();
    const size_t base = (size_t)blockIdx.x * kSortTile + (size_t)w * (kSortItems * 32) + lane;
    uint32_t k[kSortItems], v[kSortItems], rk[kSortItems];
#pragma unroll
    for (int r = 0; r < kSortItems; ++r) {
        size_t i = base + (size_t)r * 32;
        k[r] = i < n ? __ldg(keys + i) : 0xFFFFFFFFu;
        v[r] = FirstPass ? (uint32_t)i : (i < n ? __ldg(vals + i) : 0u);
    }
    const unsigned lt = (1u << lane) - 1;
#pragma unroll
    for (int r = 0; r < kSortItems; ++r) {
        bool ok = base + (size_t)r * 32 < n;
        uint32_t d = ok ? ((k[r] >> shift) & mask) : 0xFFFFFFFFu;
        unsigned peers = __match_any_sync(0xffffffffu, d);
        uint32_t old = ok ? wh[w][d] : 0u;
        __syncwarp();
        if (ok && (peers & lt) == 0) wh[w][d] = old + (uint32_t)__popc(peers);
        __syncwarp();
        rk[r] = old + (uint32_t)__popc(peers & lt);
    }
    __syncthreads();
    {   // digit d = threadIdx.x: exclusive scan over the warps of this tile, plus the tile's global offset
        uint32_t run = __ldg(offs + (size_t)threadIdx.x * n_tiles + blockIdx.x);
#pragma unroll
        for (int ww = 0; ww < kSortWarps; ++ww) { uint32_t t = wh[ww][threadIdx.x]; wh[ww][threadIdx.x] = run; run += t; }
    }
    __syncthreads();
#pragma unroll
    for (int r = 0; r < kSortItems; ++r) {
        if (base + (size_t)r * 32 < n) {
            uint32_t d = (k[r] >> shift) & mask;
            uint32_t dst = wh[w][d] + rk[r];
            out_keys[dst] = k[r];
            out_vals[dst] = v[r];
        }
    }
}

int launch_radix_sort(uint32_t* keys_a, uint32_t* keys_b, uint32_t* val_a, uint32_t* val_b, uint32_t n,
                      int key_bits, uint32_t* d_counts, size_t counts_entries, uint32_t* d_partials, cudaStream_t s) {
    if (n == 0) return 0;
    if (key_bits < 1) key_bits = 1;
    int passes = (key_bits + 7) / 8;
    uint32_t n_tiles = (uint32_t)(((size_t)n + kSortTile - 1) / kSortTile);
    (void)counts_entries;
    uint32_t *ki = keys_a, *ko = keys_b, *vi = val_a, *vo = val_b;
    for (int p = 0; p < passes; ++p) {
        int shift = 8 * p;
        int bits = std::min(8, key_bits - shift);
        uint32_t mask = (1u << bits) - 1u;
        k_sort_hist<<<n_tiles, kSortThreads, 0, s>>>(ki, n, shift, mask, d_counts, n_tiles); count_launch();
        device_scan<OpSum, false, false>(d_counts, (size_t)256 * n_tiles, d_partials, s);
        if (p == 0) k_sort_scatter<true><<<n_tiles, kSortThreads, 0, s>>>(ki, vi, n, shift, mask, d_counts, n_tiles, ko, vo);
        else        k_sort_scatter<false><<<n_tiles, kSortThreads, 0, s>>>(ki, vi, n, shift, mask, d_counts, n_tiles, ko, vo);
        count_launch();
        uint32_t* t = ki; ki = ko; ko = t; t = vi; vi = vo; vo = t;
    }
    return passes & 1;
}

// ------------------------------------------------------------------------------------------
// (a3) gather into cell order + fp64 unit vectors.
// Accuracy: RA is reduced to |t| <= 45 deg in the degree domain (t = ra - 90 rint(ra/90) is exact),
// Dec uses the colatitude 90 - |dec| (exact) beyond 45 deg, so the radian conversion never rounds
// an angle larger than pi/4; unit-vector chords are then good to ~5e-11 arcsec.
// ------------------------------------------------------------------------------------------
__device__ __forceinline__ void unit_vector(double ra_norm, double dec, double& x, double& y, double& z) {
    const double D2R = 0.017453292519943295;   // pi / 180
    double q = rint(ra_norm * (1.0 / 90.0));
    double t = fma(-90.0, q, ra_norm);
    double st, ct; sincos(t * D2R, &st, &ct);
    int iq = ((int)q) & 3;
    double ca = (iq == 0) ? ct : (iq == 1) ? -st : (iq == 2) ? -ct : st;
    double sa = (iq == 0) ? st : (iq == 1) ? ct : (iq == 2) ? -st : -ct;
    double ad = fabs(dec), sd, cd;
    if (ad > 45.0) { double s, c; sincos((90.0 - ad) * D2R, &s, &c); sd = c; cd = s; }
    else           { sincos(ad * D2R, &sd, &cd); }
    sd = copysign(sd, dec);
    x = cd * ca; y = cd * sa; z = sd;
}

__global__ void __launch_bounds__(256)
k_gather(const double* __restrict__ ra, const double* __restrict__ dec, const int64_t* __restrict__ id,
         const uint32_t* __restrict__ perm, uint32_t n,
         double* __restrict__ x, double* __restrict__ y, double* __restrict__ z, int64_t* __restrict__ out_id) {
    for (size_t i = (size_t)blockIdx.x * 256 + threadIdx.x; i < n; i += (size_t)gridDim.x * 256) {
        uint32_t p = __ldg(perm + i);
        double a = __ldg(ra + p), d = __ldg(dec + p);
        int64_t v = id ? __ldg(id + p) : (int64_t)p;
        double ux = 0.0, uy = 0.0, uz = 2.0;      // bad coordinate: a point no chord test can reach
        if (coord_ok(a, d)) unit_vector(norm_ra(a), d, ux, uy, uz);
        x[i] = ux; y[i] = uy; z[i] = uz; out_id[i] = v;
    }
}

void launch_gather(const double* ra, const double* dec, const int64_t* id, const uint32_t* perm, uint32_t n,
                   double* x, double* y, double* z, int64_t* out_id, cudaStream_t s) {
    if (n == 0) return;
    int blocks = (int)std::min<size_t>(((size_t)n + 255) / 256, (size_t)sm_count() * 16);
    k_gather<<<blocks, 256, 0, s>>>(ra, dec, id, perm, n, x, y, z, out_id); count_launch();
}

// ------------------------------------------------------------------------------------------
// (a4) cell offset table: mark the first sorted row of every occupied cell, then a reverse
// inclusive min-scan gives every (also empty) cell the first row at or after it.
// ------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256)
k_mark_heads(const uint32_t* __restrict__ keys, uint32_t n, uint32_t n_cells, uint32_t* __restrict__ cell_start) {
    for (size_t i = (size_t)blockIdx.x * 256 + threadIdx.x; i <= n; i += (size_t)gridDim.x * 256) {
        if (i == n) { cell_start[n_cells] = n; break; }
        uint32_t k = __ldg(keys + i);
        if (i == 0 || __ldg(keys + i - 1) != k) cell_start[k] = (uint32_t)i;
    }
}

void launch_cell_table(const uint32_t* sorted_keys, uint32_t n, uint32_t n_cells, uint32_t* cell_start,
                       uint32_t* d_partials, cudaStream_t s) {
    cudaMemsetAsync(cell_start, 0xFF, ((size_t)n_cells + 1) * sizeof(uint32_t), s);
    int blocks = (int)std::min<size_t>(((size_t)n + 1 + 255) / 256, (size_t)sm_count() * 16);
    k_mark_heads<<<blocks, 256, 0, s>>>(sorted_keys, n, n_cells, cell_start); count_launch();
    device_scan<OpMin, true, true>(cell_start, (size_t)n_cells + 1, d_partials, s);
}

}  // namespace hlc2
