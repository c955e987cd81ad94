// hlc2_stream.cu -- partition streaming from pinned host memory (NS (c)).
//
// The paper overlaps transfer and compute with pinned host memory, several CUDA streams and asynchronous
// copies because transfer was ~90 % of its run time (L246), and cuts the catalogues
// into calculation blocks that fit the device (L253-257).  Here the blocks are declination bands:
//
//   copy stream     H2D of the raw columns (ra, dec, id) of A band k+1 and B band k+2 while band k computes
//   compute stream  B window of band k = B band k + the rows of bands k-1 / k+1 within r of band k's edges
//                   (a device filter: no source is replicated on the host, no pair is lost across band edges);
//                   hlc2_build_index of the window and of A band k; hlc2_crossmatch into an output slot
//   out stream      D2H of the finished rows of band k into the pinned outputs while band k+1 computes
//
// Every A source lives in exactly one band and sees one B window, so nearest mode needs no merge step.
// Device memory is the caller's arena (hlc2_stream_sizes): 2 raw A slots, 4 raw B slots, the window's raw
// columns, two index buffers, build / match scratch and 2 output slots.
#include <string.h>

#include <algorithm>

#include "hlc2_internal.cuh"

namespace hlc2 {

// rows of a neighbouring B band whose declination lies in [lo, hi] are appended to the window
__global__ void __launch_bounds__(256)
k_halo_append(const double* __restrict__ ra, const double* __restrict__ dec, const long long* __restrict__ id,
              long long id_base, uint32_t n, double lo, double hi,
              double* __restrict__ o_ra, double* __restrict__ o_dec, long long* __restrict__ o_id,
              uint32_t* __restrict__ counter, uint32_t cap) {
    const unsigned lane = threadIdx.x & 31;
    const size_t stride = (size_t)gridDim.x * 256;
    for (size_t b = (size_t)blockIdx.x * 256 + (threadIdx.x & ~31u); b < n; b += stride) {
        const size_t i = b + lane;
        double d = 0.0;
        bool keep = false;
        if (i < n) { d = __ldg(dec + i); keep = d >= lo && d <= hi; }       // NaN dec: not kept here, reported by its own band
        const unsigned m = __ballot_sync(0xffffffffu, keep);
        if (m == 0) continue;
        uint32_t base = 0;
        if (lane == 0) base = atomicAdd(counter, (uint32_t)__popc(m));
        base = __shfl_sync(0xffffffffu, base, 0);
        if (keep) {
            const uint32_t o = base + __popc(m & ((1u << lane) - 1u));
            if (o < cap) { o_ra[o] = __ldg(ra + i); o_dec[o] = d; o_id[o] = id ? __ldg(id + i) : id_base + (long long)i; }
        }
    }
}

// ids = global row numbers when the caller passes none
__global__ void __launch_bounds__(256)
k_iota_ids(long long* __restrict__ o, long long base, uint32_t n) {
    for (size_t i = (size_t)blockIdx.x * 256 + threadIdx.x; i < n; i += (size_t)gridDim.x * 256) o[i] = base + (long long)i;
}

static inline size_t up256(size_t v) { return (v + 255) / 256 * 256; }

struct StreamArena {
    size_t raw_a[2], raw_b[4], win, idx_a, idx_b, temp, out[2], counters, total;
    size_t ib_a, ib_b, tb;          // index / scratch sizes
    size_t win_cap;                 // rows the B window can hold
};

static int stream_arena(int64_t max_a, int64_t max_b, const hlc2_opts* opts, int64_t max_out, StreamArena* L) {
    if (max_a < 0 || max_b < 0 || max_out < 0) return HLC2_ERR_INVALID_ARG;
    L->win_cap = (size_t)max_b * 3;                                   // band k + at most both whole neighbours
    if (L->win_cap >= ((size_t)1 << 30) || (size_t)max_a >= ((size_t)1 << 30)) return HLC2_ERR_TOO_MANY;
    size_t ia = 0, ta = 0, ib = 0, tb = 0;
    int rc = hlc2_index_sizes(max_a, opts, &ia, &ta); if (rc != HLC2_OK) return rc;
    rc = hlc2_index_sizes((int64_t)L->win_cap, opts, &ib, &tb); if (rc != HLC2_OK) return rc;
    L->ib_a = std::max(ia, ib); L->ib_b = ib;      // A bands are filed on the window's grid: its cell table can be the larger one
    L->tb = std::max(std::max(ta, tb), match_temp_bound(max_a, opts));
    size_t off = 0;
    for (int i = 0; i < 2; ++i) { L->raw_a[i] = off; off += up256((size_t)max_a * 8) * 3; }
    for (int i = 0; i < 4; ++i) { L->raw_b[i] = off; off += up256((size_t)max_b * 8) * 3; }
    L->win = off; off += up256(L->win_cap * 8) * 3;
    L->idx_a = off; off += up256(L->ib_a);
    L->idx_b = off; off += up256(ib);
    L->temp = off; off += up256(L->tb);
    for (int i = 0; i < 2; ++i) { L->out[i] = off; off += up256((size_t)max_out * 8) * 3; }
    L->counters = off; off += 256;
    L->total = off;
    return HLC2_OK;
}

}  // namespace hlc2

using namespace hlc2;

extern "C" {

int hlc2_stream_sizes(int64_t max_band_a, int64_t max_band_b, const hlc2_opts* opts, int64_t max_band_out,
                      size_t* arena_bytes) {
    if (!arena_bytes) return HLC2_ERR_INVALID_ARG;
    StreamArena L;
    int rc = stream_arena(max_band_a, max_band_b, opts, max_band_out, &L);
    if (rc != HLC2_OK) return rc;
    *arena_bytes = L.total;
    return HLC2_OK;
}

namespace {
struct StreamRes {
    cudaStream_t copy = nullptr, comp = nullptr, out = nullptr;
    cudaEvent_t in_a[2] = {}, in_b[4] = {}, free_out[2] = {}, matched[2] = {};
    bool ok = true;
    StreamRes() {
        ok &= cudaStreamCreateWithFlags(&copy, cudaStreamNonBlocking) == cudaSuccess;
        ok &= cudaStreamCreateWithFlags(&comp, cudaStreamNonBlocking) == cudaSuccess;
        ok &= cudaStreamCreateWithFlags(&out, cudaStreamNonBlocking) == cudaSuccess;
        for (auto& e : in_a) ok &= cudaEventCreateWithFlags(&e, cudaEventDisableTiming) == cudaSuccess;
        for (auto& e : in_b) ok &= cudaEventCreateWithFlags(&e, cudaEventDisableTiming) == cudaSuccess;
        for (auto& e : free_out) ok &= cudaEventCreateWithFlags(&e, cudaEventDisableTiming) == cudaSuccess;
        for (auto& e : matched) ok &= cudaEventCreateWithFlags(&e, cudaEventDisableTiming) == cudaSuccess;
    }
    ~StreamRes() {
        if (copy) { cudaStreamSynchronize(copy); cudaStreamDestroy(copy); }
        if (comp) { cudaStreamSynchronize(comp); cudaStreamDestroy(comp); }
        if (out) { cudaStreamSynchronize(out); cudaStreamDestroy(out); }
        for (auto& e : in_a) if (e) cudaEventDestroy(e);
        for (auto& e : in_b) if (e) cudaEventDestroy(e);
        for (auto& e : free_out) if (e) cudaEventDestroy(e);
        for (auto& e : matched) if (e) cudaEventDestroy(e);
    }
};
struct IndexGuard {
    hlc2_index* h = nullptr;
    ~IndexGuard() { if (h) hlc2_index_destroy(h); }
};
}  // namespace

#define CK(call) do { if ((call) != cudaSuccess) return HLC2_ERR_CUDA; } while (0)
#define RC(call) do { int rc__ = (call); if (rc__ != HLC2_OK) return rc__; } while (0)

int hlc2_stream_crossmatch(const double* h_a_ra, const double* h_a_dec, const int64_t* h_a_id, const int64_t* h_a_off,
                           const double* h_b_ra, const double* h_b_dec, const int64_t* h_b_id, const int64_t* h_b_off,
                           const double* band_edges_deg, int64_t n_bands,
                           double radius_arcsec, int mode, const hlc2_opts* opts,
                           int64_t* h_out_idA, int64_t* h_out_idB, double* h_out_sep_arcsec, int64_t capacity,
                           unsigned long long* h_count, void* d_arena, size_t arena_bytes, int64_t max_band_out) {
    if (!h_count || n_bands < 0 || capacity < 0 || max_band_out < 0 || !(radius_arcsec > 0.0) ||
        (mode != HLC2_ALL_PAIRS && mode != HLC2_NEAREST)) return HLC2_ERR_INVALID_ARG;
    *h_count = 0;
    if (n_bands == 0) return HLC2_OK;
    if (!h_a_off || !h_b_off || !band_edges_deg || !d_arena ||
        (capacity > 0 && (!h_out_idA || !h_out_idB || !h_out_sep_arcsec))) return HLC2_ERR_INVALID_ARG;
    const double r_deg = radius_arcsec / 3600.0;
    int64_t max_a = 0, max_b = 0;
    for (int64_t k = 0; k < n_bands; ++k) {
        const int64_t na = h_a_off[k + 1] - h_a_off[k], nb = h_b_off[k + 1] - h_b_off[k];
        if (na < 0 || nb < 0 || !(band_edges_deg[k + 1] > band_edges_deg[k])) return HLC2_ERR_INVALID_ARG;
        // a band lower than r would need more than the two neighbouring bands
        if (n_bands > 1 && band_edges_deg[k + 1] - band_edges_deg[k] < r_deg) return HLC2_ERR_INVALID_ARG;
        max_a = std::max(max_a, na); max_b = std::max(max_b, nb);
    }
    if ((h_a_off[n_bands] > h_a_off[0] && (!h_a_ra || !h_a_dec)) || (h_b_off[n_bands] > h_b_off[0] && (!h_b_ra || !h_b_dec)))
        return HLC2_ERR_INVALID_ARG;
    StreamArena L;
    RC(stream_arena(max_a, max_b, opts, max_band_out, &L));
    if (arena_bytes < L.total) return HLC2_ERR_BUFFER_TOO_SMALL;
    char* base = (char*)d_arena;
    const size_t sa = up256((size_t)max_a * 8), sb = up256((size_t)max_b * 8), sw = up256(L.win_cap * 8), so = up256((size_t)max_band_out * 8);
    uint32_t* d_halo = (uint32_t*)(base + L.counters);
    unsigned long long* d_cnt = (unsigned long long*)(base + L.counters + 64);

    StreamRes R;
    if (!R.ok) return HLC2_ERR_CUDA;

    auto h2d_a = [&](int64_t k) -> cudaError_t {
        const size_t n = (size_t)(h_a_off[k + 1] - h_a_off[k]), o = (size_t)h_a_off[k];
        char* s = base + L.raw_a[k & 1];
        cudaError_t e = cudaSuccess;
        if (n) {
            e = cudaMemcpyAsync(s, h_a_ra + o, n * 8, cudaMemcpyHostToDevice, R.copy);
            if (e == cudaSuccess) e = cudaMemcpyAsync(s + sa, h_a_dec + o, n * 8, cudaMemcpyHostToDevice, R.copy);
            if (e == cudaSuccess && h_a_id) e = cudaMemcpyAsync(s + 2 * sa, h_a_id + o, n * 8, cudaMemcpyHostToDevice, R.copy);
        }
        if (e == cudaSuccess) e = cudaEventRecord(R.in_a[k & 1], R.copy);
        return e;
    };
    auto h2d_b = [&](int64_t k) -> cudaError_t {
        const size_t n = (size_t)(h_b_off[k + 1] - h_b_off[k]), o = (size_t)h_b_off[k];
        char* s = base + L.raw_b[k & 3];
        cudaError_t e = cudaSuccess;
        if (n) {
            e = cudaMemcpyAsync(s, h_b_ra + o, n * 8, cudaMemcpyHostToDevice, R.copy);
            if (e == cudaSuccess) e = cudaMemcpyAsync(s + sb, h_b_dec + o, n * 8, cudaMemcpyHostToDevice, R.copy);
            if (e == cudaSuccess && h_b_id) e = cudaMemcpyAsync(s + 2 * sb, h_b_id + o, n * 8, cudaMemcpyHostToDevice, R.copy);
        }
        if (e == cudaSuccess) e = cudaEventRecord(R.in_b[k & 3], R.copy);
        return e;
    };

    CK(h2d_b(0));
    if (n_bands > 1) CK(h2d_b(1));
    CK(h2d_a(0));
    unsigned long long total = 0, written = 0;
    bool too_small = false, bad = false;
    const int sms = sm_count();

    for (int64_t k = 0; k < n_bands; ++k) {
        // prefetch: the slots these go into were last read by work the host has already waited for
        if (k + 1 < n_bands) CK(h2d_a(k + 1));
        if (k + 2 < n_bands) CK(h2d_b(k + 2));
        const size_t na = (size_t)(h_a_off[k + 1] - h_a_off[k]);
        const size_t nbk = (size_t)(h_b_off[k + 1] - h_b_off[k]);
        if (na == 0) continue;
        CK(cudaStreamWaitEvent(R.comp, R.in_a[k & 1], 0));
        CK(cudaStreamWaitEvent(R.comp, R.in_b[k & 3], 0));
        if (k > 0) CK(cudaStreamWaitEvent(R.comp, R.in_b[(k - 1) & 3], 0));
        if (k + 1 < n_bands) CK(cudaStreamWaitEvent(R.comp, R.in_b[(k + 1) & 3], 0));

        // ---- B window: band k, then the rows of bands k-1 and k+1 within r of this band's edges
        double* w_ra = (double*)(base + L.win); double* w_dec = (double*)(base + L.win + sw);
        long long* w_id = (long long*)(base + L.win + 2 * sw);
        const char* bk = base + L.raw_b[k & 3];
        if (nbk) {
            CK(cudaMemcpyAsync(w_ra, bk, nbk * 8, cudaMemcpyDeviceToDevice, R.comp));
            CK(cudaMemcpyAsync(w_dec, bk + sb, nbk * 8, cudaMemcpyDeviceToDevice, R.comp));
            if (h_b_id) CK(cudaMemcpyAsync(w_id, bk + 2 * sb, nbk * 8, cudaMemcpyDeviceToDevice, R.comp));
            else {
                k_iota_ids<<<(unsigned)std::min<size_t>((nbk + 255) / 256, (size_t)sms * 8), 256, 0, R.comp>>>(w_id, (long long)h_b_off[k], (uint32_t)nbk);
                count_launch();
            }
        }
        CK(cudaMemsetAsync(d_halo, 0, sizeof(uint32_t), R.comp));
        const uint32_t halo_cap = (uint32_t)(L.win_cap - nbk);
        for (int side = -1; side <= 1; side += 2) {
            const int64_t j = k + side;
            if (j < 0 || j >= n_bands) continue;
            const size_t nj = (size_t)(h_b_off[j + 1] - h_b_off[j]);
            if (!nj) continue;
            const char* bj = base + L.raw_b[j & 3];
            const double lo = side < 0 ? band_edges_deg[k] - r_deg - 1e-9 : -1e300;
            const double hi = side < 0 ? 1e300 : band_edges_deg[k + 1] + r_deg + 1e-9;
            k_halo_append<<<(unsigned)std::min<size_t>((nj + 255) / 256, (size_t)sms * 8), 256, 0, R.comp>>>(
                (const double*)bj, (const double*)(bj + sb), h_b_id ? (const long long*)(bj + 2 * sb) : nullptr,
                (long long)h_b_off[j], (uint32_t)nj, lo, hi, w_ra + nbk, w_dec + nbk, w_id + nbk, d_halo, halo_cap);
            count_launch();
        }
        uint32_t n_halo = 0;
        CK(cudaMemcpyAsync(&n_halo, d_halo, sizeof(uint32_t), cudaMemcpyDeviceToHost, R.comp));
        CK(cudaStreamSynchronize(R.comp));
        const size_t nwin = nbk + std::min<size_t>(n_halo, halo_cap);
        if (nwin == 0) continue;

        // ---- index both sides, match, count
        IndexGuard gb, ga;
        RC(hlc2_build_index(w_ra, w_dec, (const int64_t*)w_id, (int64_t)nwin, opts, base + L.idx_b, L.ib_b, base + L.temp, L.tb, R.comp, &gb.h));
        char* ak = base + L.raw_a[k & 1];
        if (!h_a_id) {
            k_iota_ids<<<(unsigned)std::min<size_t>((na + 255) / 256, (size_t)sms * 8), 256, 0, R.comp>>>((long long*)(ak + 2 * sa), (long long)h_a_off[k], (uint32_t)na);
            count_launch();
        }
        // A band k is filed on the window's grid (opts.grid_like), so that the match takes its same-grid path; a band
        // that does not fit inside the window's RA box (a patch of A with no B nearby) gets a grid of its own
        {
            hlc2_opts oa;
            if (opts) oa = *opts; else { memset(&oa, 0, sizeof oa); oa.r_max_arcsec = 1.0; }
            oa.grid_like = gb.h;
            int rc_a = hlc2_build_index((const double*)ak, (const double*)(ak + sa), (const int64_t*)(ak + 2 * sa), (int64_t)na, &oa,
                                        base + L.idx_a, L.ib_a, base + L.temp, L.tb, R.comp, &ga.h);
            if (rc_a == HLC2_ERR_GRID_MISMATCH || rc_a == HLC2_ERR_BUFFER_TOO_SMALL)
                rc_a = hlc2_build_index((const double*)ak, (const double*)(ak + sa), (const int64_t*)(ak + 2 * sa), (int64_t)na, opts,
                                        base + L.idx_a, L.ib_a, base + L.temp, L.tb, R.comp, &ga.h);
            RC(rc_a);
        }
        char* ok_ = base + L.out[k & 1];
        CK(cudaStreamWaitEvent(R.comp, R.free_out[k & 1], 0));      // band k-2's rows have left this slot
        RC(hlc2_crossmatch(ga.h, gb.h, radius_arcsec, mode, (int64_t*)ok_, (int64_t*)(ok_ + so), (double*)(ok_ + 2 * so),
                           max_band_out, d_cnt, base + L.temp, L.tb, R.comp));
        unsigned long long found = 0;
        CK(cudaMemcpyAsync(&found, d_cnt, sizeof found, cudaMemcpyDeviceToHost, R.comp));
        CK(cudaEventRecord(R.matched[k & 1], R.comp));
        CK(cudaStreamSynchronize(R.comp));
        if (hlc2_index_status(ga.h, nullptr) == HLC2_ERR_BAD_COORD || hlc2_index_status(gb.h, nullptr) == HLC2_ERR_BAD_COORD) bad = true;
        total += found;
        unsigned long long rows = std::min<unsigned long long>(found, (unsigned long long)max_band_out);
        if (found > rows) too_small = true;
        const unsigned long long fit = std::min<unsigned long long>(rows, (unsigned long long)capacity - written);
        if (fit < rows) too_small = true;
        // ---- rows of band k go home on the out stream while band k+1 computes
        CK(cudaStreamWaitEvent(R.out, R.matched[k & 1], 0));
        if (fit) {
            CK(cudaMemcpyAsync(h_out_idA + written, ok_, fit * 8, cudaMemcpyDeviceToHost, R.out));
            CK(cudaMemcpyAsync(h_out_idB + written, ok_ + so, fit * 8, cudaMemcpyDeviceToHost, R.out));
            CK(cudaMemcpyAsync(h_out_sep_arcsec + written, ok_ + 2 * so, fit * 8, cudaMemcpyDeviceToHost, R.out));
        }
        CK(cudaEventRecord(R.free_out[k & 1], R.out));
        written += fit;
    }
    CK(cudaStreamSynchronize(R.out));
    CK(cudaStreamSynchronize(R.copy));
    *h_count = total;
    if (too_small) return HLC2_ERR_BUFFER_TOO_SMALL;
    return bad ? HLC2_ERR_BAD_COORD : HLC2_OK;
}

}  // extern "C"
