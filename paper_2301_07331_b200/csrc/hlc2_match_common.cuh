// hlc2_match_common.cuh -- device code shared by the two match paths (hlc2_match.cu: any two grids;
// hlc2_match_same.cu: both indices on one grid): mbarrier / bulk-copy primitives, the separation from a chord,
// the warp hit queue and the general per-lane path from global memory.
#pragma once
#include <math.h>

#include "hlc2_grid.cuh"

namespace hlc2 {

constexpr int kCW = kTile / 32;              // consumer warps (one lane per A row of the tile)
constexpr int kMatchThreads = kTile + 32;    // + the producer warp
constexpr int kQCap = 64;                    // rows in a warp's hit queue
constexpr int kQFlush = kQCap - 32;          // flushed as soon as this many are queued (at most kQFlush - 1 + 32 are ever held)
constexpr double kRad2Arcsec = 206264.80624709636;   // 648000 / pi
constexpr unsigned kFull = 0xffffffffu;

// padding of the fp32 position estimate (degrees); derivation in DESIGN.md section 5 (~3x the worst case)
constexpr double kEpsRaDeg = 2.5e-4;
constexpr double kEpsDecDeg = 1.5e-4;
constexpr double kTinyDeg = 1e-9;            // fp64 slop on cell / zone edges in the planner

struct Job;

struct MatchArgs {
    double thr2;          // 4 sin^2(r/2)
    double pad_dec;       // r in degrees + kEpsDecDeg
    double r_deg;
    float sin_r_up;       // sin(r) * (1 + 1e-5)
    int64_t* out_ida; int64_t* out_idb; double* out_sep;
    unsigned long long capacity;
    unsigned long long* count;
    Job* jobs;            // [tile_cap] first jobs, then [pool_cap] chained jobs
    uint32_t* pool_count;
    uint32_t tile_cap, pool_cap;
    // one catalogue matched with itself (PAPER.md D4, L286, L295): 0 no; 1 every unordered pair once (B row > A row);
    // 2 those and the diagonal (B row >= A row); 3 every B row but the A row itself (nearest: not its own neighbour)
    int self_mode;
    // per-record error radii (Eq. (4)): squares in arcsec^2 in cell order, or null; threshold of a pair =
    // min(radius, k sqrt(e1^2 + e2^2)), k^2 (pi / 648000)^2 folded into kfac2rad
    const double* ea2; const double* eb2; double kfac2rad;
};

// 4 sin^2(t / 2) from t^2 (radians^2): t^2 - t^4/12 + t^6/360 - t^8/20160; the next term is below 1e-14 relative up to
// t = 10 degrees (the largest radius an index accepts)
__device__ __forceinline__ double chord2_of_angle2(double t2) {
    return t2 * fma(t2, fma(t2, fma(t2, -1.0 / 20160.0, 1.0 / 360.0), -1.0 / 12.0), 1.0);
}

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
// try_wait suspends the thread in hardware until the phase completes or the time hint (ns) runs out, so a long
// hint costs no wake-up latency and spares the issue slots a polling loop would burn
__device__ __forceinline__ void mbar_wait(unsigned long long* b, unsigned parity) {
    const uint32_t a = smem_u32(b);
    unsigned done;
    do {
        asm volatile("{\n .reg .pred p;\n mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2, %3;\n selp.u32 %0, 1, 0, p;\n}"
                     : "=r"(done) : "r"(a), "r"(parity), "r"(0x4000u) : "memory");
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
// the general per-lane path: any number of zones, RA wrap, polar ring, window partly outside B's box.  Reads B
// through global memory / L2.
// ------------------------------------------------------------------------------------------------------
struct Best { double c2; uint32_t row; bool has; };      // row: global B row

// one row straight to the output; lanes that arrive together share one global atomic
__device__ __forceinline__ void emit_direct(const IndexView& A, const IndexView& B, const MatchArgs& p, uint32_t a_row, uint32_t b_row, double c2) {
    const unsigned m = __activemask();
    const int lane = threadIdx.x & 31, leader = __ffs(m) - 1;
    unsigned long long base = 0;
    if (lane == leader) base = atomicAdd(p.count, (unsigned long long)__popc(m));
    base = __shfl_sync(m, base, leader);
    const unsigned long long o = base + __popc(m & ((1u << lane) - 1u));
    if (o < p.capacity) { p.out_ida[o] = __ldg(A.id + a_row); p.out_idb[o] = __ldg(B.id + b_row); p.out_sep[o] = sep_from_chord2(c2); }
}

template <int MODE>
__device__ __forceinline__ void scan_global(const IndexView& A, const IndexView& B, const MatchArgs& p, uint32_t a_row,
                                            double ax, double ay, double az, uint32_t j0, uint32_t j1, Best& h,
                                            uint32_t off = 0, uint32_t stride = 1) {
    // (off, stride) = (0, 1): the calling lane walks the whole range; (lane, 32): a warp shares one A row and its lanes
    // take every 32nd candidate (coalesced loads: the way to walk long ranges, e.g. dense cells at the RA seam)
    if (p.self_mode == 1) j0 = max(j0, a_row + 1u); else if (p.self_mode == 2) j0 = max(j0, a_row);
    const double ea2 = p.eb2 ? __ldg(p.ea2 + a_row) : 0.0;
    for (uint32_t j = j0 + off; j < j1; j += stride) {
        if (p.self_mode == 3 && j == a_row) continue;
        const double dx = ax - __ldg(B.x + j), dy = ay - __ldg(B.y + j), dz = az - __ldg(B.z + j);
        const double c2 = fma(dx, dx, fma(dy, dy, dz * dz));
        const double thr2 = p.eb2 ? fmin(p.thr2, chord2_of_angle2((ea2 + __ldg(p.eb2 + j)) * p.kfac2rad)) : p.thr2;
        if (c2 <= thr2) {
            if (MODE == HLC2_ALL_PAIRS) emit_direct(A, B, p, a_row, j, c2);
            else if (!h.has || c2 < h.c2 || (c2 == h.c2 && __ldg(B.id + j) < __ldg(B.id + h.row))) { h.has = true; h.row = j; h.c2 = c2; }
        }
    }
}

template <int MODE>
__device__ __noinline__ void scan_general(const IndexView& A, const IndexView& B, const MatchArgs& p, uint32_t a_row,
                                          double ax, double ay, double az, float2 pf, Best& h,
                                          uint32_t off = 0, uint32_t stride = 1) {
    const GridView& g = B.g;
    const double dlo = (double)pf.y - p.pad_dec, dhi = (double)pf.y + p.pad_dec;
    if (!(dhi >= g.dec_min && dlo <= g.dec_max)) return;          // also rows with a bad coordinate (NaN vector)
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
        scan_global<MODE>(A, B, p, a_row, ax, ay, az, __ldg(B.cell_start + base + k0), __ldg(B.cell_start + base + k1 + 1), h, off, stride);
        if (k3 >= k2)
            scan_global<MODE>(A, B, p, a_row, ax, ay, az, __ldg(B.cell_start + base + k2), __ldg(B.cell_start + base + k3 + 1), h, off, stride);
    }
}

// ------------------------------------------------------------------------------------------------------
// hit queue of one consumer warp: ids are looked up when a queue is flushed (32 rows at a time,
// overlapped with the atomic), so neither catalogue's id column is staged: the queue holds global row numbers
// ------------------------------------------------------------------------------------------------------
struct WarpQueue { uint32_t a[kQCap], b[kQCap]; double c2[kQCap]; };

// write queue rows [first, first + cnt) to the output: one global atomic, coalesced stores
__device__ __forceinline__ void flush_rows(const IndexView& A, const IndexView& B, const MatchArgs& p, const WarpQueue& q,
                                           unsigned first, unsigned cnt, int lane) {
    unsigned long long base = 0;
    if (lane == 0) base = atomicAdd(p.count, (unsigned long long)cnt);
    base = __shfl_sync(kFull, base, 0);
    for (unsigned k = lane; k < cnt; k += 32) {
        const unsigned long long o = base + k;
        if (o < p.capacity) {
            p.out_ida[o] = __ldg(A.id + q.a[first + k]); p.out_idb[o] = __ldg(B.id + q.b[first + k]);
            p.out_sep[o] = sep_from_chord2(q.c2[first + k]);
        }
    }
}

// append the lanes with `hit`; flush the top kQFlush rows once that many are queued.  qn is warp-uniform.
__device__ __forceinline__ void push_hits(const IndexView& A, const IndexView& B, const MatchArgs& p, WarpQueue& q, unsigned& qn,
                                          bool hit, uint32_t a_row, uint32_t b_row, double c2, int lane) {
    const unsigned m = __ballot_sync(kFull, hit);
    if (m == 0) return;
    if (hit) {
        const unsigned k = qn + __popc(m & ((1u << lane) - 1u));
        q.a[k] = a_row; q.b[k] = b_row; q.c2[k] = c2;
    }
    qn += __popc(m);
    if (qn >= (unsigned)kQFlush) {
        __syncwarp();
        qn -= kQFlush;
        flush_rows(A, B, p, q, qn, kQFlush, lane);
        __syncwarp();
    }
}

// launchers of the same-grid path (hlc2_match_same.cu)
size_t match_same_temp_bytes(const IndexView& A);
void launch_match_all_general(const IndexView& A, const IndexView& B, const MatchArgs& p, int mode, cudaStream_t s,
                              cudaEvent_t ev_start, cudaEvent_t ev_stop);
void launch_match_same(const IndexView& A, const IndexView& B, const MatchArgs& p, int mode, void* d_temp, cudaStream_t s,
                       cudaEvent_t ev_start, cudaEvent_t ev_stop);

}  // namespace hlc2
