// hlc2_match_same.cu -- the match when both indices were filed on ONE grid (opts.grid_like): SURVEY rows a5-a7, NS (b).
//
// A source's cell key then means the same in both catalogues, and its window flags (top bits of the key, set by the
// index build from r_max) say which cells around its own cell its search window can reach.  With zones several r_max
// high almost every source needs its own cell only, some one neighbouring RA cell, a few one neighbouring zone (the
// cells the quad-direction strategy probes, taken only by the sources that are actually within r of
// that edge, plus the diagonal it misses).  One kernel, no planner and no job records:
//
//   k_match_same   persistent CTAs of kCW consumer warps + 1 producer warp around a ring of small stages.
//     Producer: keeps the next 32 tiles of its CTA in flight, one per lane (descriptor, then the cell_start entries that
//       bound the tile's windows).  A tile becomes a short run of stages: the B rows (x, y, z) and the cell_start slice of
//       cells k_first-1 .. k_last+1 of the tile's OWN zone, then -- only if the tile descriptor says some row of the tile
//       reaches into the zone below / above -- the same for the matching cells of that zone; a piece larger than a stage
//       is cut into row chunks (the paper's calculation blocks, L253-257).  Everything moves by 1-D bulk copies
//       (cp.async.bulk, the TMA engine).  The A rows of the tile a few stages ahead are prefetched into L2.
//     Consumers: one lane per A row (the paper's thread-per-A-record hierarchy, L271-276); the rows are loaded coalesced
//       straight into registers one tile ahead, so the ring holds B only.  In an own-zone stage a lane reads its row
//       range from the staged slice at [key - ExtLo, key + ExtHi + 1]; in a neighbour stage only the lanes with that Dec
//       flag work, on the cells that can hold an RA between their own cells' outer edges (the edges scale with the two
//       zones' cell counts: a superset).  Test: chord^2 <= 4 sin^2(r/2) in fp64.
//     Output (row a6): hits are compacted by ballot into a per-warp ring of (A row, B row, chord^2).  At the end of a tile
//       the 32 output slots of a full block are reserved (one global atomic) and its ids are requested; they are written
//       at the end of the NEXT tile, so neither latency is waited for.
//     Rows flagged kKeyGeneral (window through RA = 0/360, polar rows) are set aside and take the general per-lane path.
//
// Decisions are fp64; the flags only ever select a superset of cells.
#include <assert.h>

#include <algorithm>

#include "hlc2_match_common.cuh"

// -DHLC2_DEBUG_BOUNDS: device-side checks of every shared-memory index the kernel computes (compute-sanitizer is
// closed on the B200 pool; the GPU tests are run once per round against a library built this way)
#ifdef HLC2_DEBUG_BOUNDS
#define HLC2_CHECK(c) assert(c)
#else
#define HLC2_CHECK(c) ((void)0)
#endif

namespace hlc2 {

#ifndef HLC2_SSTAGES
#define HLC2_SSTAGES 2
#endif
#ifndef HLC2_SBCAP
#define HLC2_SBCAP 96
#endif
#ifndef HLC2_SCSCAP
#define HLC2_SCSCAP 512
#endif
#ifndef HLC2_SCTAS
#define HLC2_SCTAS 7
#endif
constexpr int kSStages = HLC2_SSTAGES;
constexpr int kSBCap = HLC2_SBCAP;           // staged B rows per stage, after 16-byte alignment (even)
constexpr int kSCsCap = HLC2_SCSCAP;         // staged cell_start entries per stage, after alignment (multiple of 4)
constexpr int kRing = 64;                    // entries of a warp's hit ring (power of two)

constexpr uint32_t kSFirst = 1u, kSLast = 2u;    // first / last stage of an A tile
constexpr uint32_t kSEnd = 4u;                    // producer -> consumers: no more work
constexpr uint32_t kSWide = 8u;                   // the piece spans more cells than a stage holds: rows read cell_start and B from global memory
constexpr uint32_t kSLo = 16u, kSHi = 32u;        // the piece lies in the zone below / above the tile's: only rows with that Dec flag work

// stage descriptor: four 16-byte words
struct SDesc {
    uint32_t flags, cs_al, row_al, row_lo;              // cs_al: first staged cell_start entry; row_al: first staged B row; chunk = rows [row_lo, row_hi)
    uint32_t row_hi, nn, a_first, a_count;              // nn: RA cells of the piece's zone; the tile's A rows
    uint32_t a_off, k_off, cb_own, cb_nb;               // first stage: offsets of A row 0 in ax.. / ak; first cell of the tile's zone / of the piece's zone
    double c_lo, c_hi;                                  // neighbour pieces: cell-count ratio of the two zones, rounded down / up
};
static_assert(sizeof(SDesc) == 64, "read as four 16-byte words");
// the first stage of a tile also carries the tile's A rows (x, y, z and the flagged keys), rounded out to 16 bytes
struct __align__(16) SStage {
    double bx[kSBCap], by[kSBCap], bz[kSBCap]; uint32_t cs[kSCsCap];
    double ax[kTile + 2], ay[kTile + 2], az[kTile + 2]; uint32_t ak[kTile + 4];
    SDesc d;
};
// per consumer warp: the hit ring (A row, B row, chord^2), the two blocks whose output slots are reserved (ids arriving
// by cp.async)
struct WarpSm {
    uint32_t qa[kRing], qb[kRing]; double qc2[kRing];
    long long pida[2][32], pidb[2][32]; double pc2[2][32];
};
// what the producer needs to issue one tile, computed 32 tiles at a time (one per lane) and parked here
struct __align__(16) TileRec {
    uint32_t a_first, a_count, cb_own, n_own;      // rows; first cell and RA cells of the tile's zone
    uint32_t o_k0g, o_nk, o_r0, o_r1;              // own piece: first cell (global), cells, B rows [r0, r1)
    uint32_t l_k0g, l_nk, l_r0, l_r1;              // piece in the zone below (l_nn = its RA cells; 0: none)
    uint32_t h_k0g, h_nk, h_r0, h_r1;              // piece in the zone above
    uint32_t l_nn, h_nn; double inv_n;
};
static_assert(sizeof(TileRec) == 80, "read as five 16-byte words");
struct __align__(16) SSmem {
    SStage st[kSStages];
    WarpSm w[kCW];
    TileRec rec[32];
    unsigned long long full[kSStages], empty[kSStages];
};
static_assert(kSBCap % 2 == 0 && kSCsCap % 4 == 0 && sizeof(SStage) % 16 == 0, "bulk copies need 16-byte pieces");
static_assert(kSCsCap * 4 + (kTile + 2) * 24 >= kSBCap * 8, "reading bz up to kSBCap rows past its end stays inside the stage");
static_assert((kRing & (kRing - 1)) == 0 && kRing >= 64, "ring indices wrap by masking; 31 rows left over + 32 of a push must fit");

__device__ __forceinline__ void prefetch_l2(const void* p) { asm volatile("prefetch.global.L2 [%0];" ::"l"(p)); }
// per-thread asynchronous copies global -> shared; cp_async_wait_all waits for the calling thread's own copies
__device__ __forceinline__ void cp_async8(void* smem_dst, const void* gsrc) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(smem_u32(smem_dst)), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async4(void* smem_dst, const void* gsrc) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(smem_u32(smem_dst)), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;" ::: "memory"); }

// Cells of a zone with nn RA cells that can hold an RA lying between the west edge of cell klo and the east edge of
// cell khi of a zone with n cells: the edges scale with nn / n.  c_lo / c_hi are that ratio pushed down / up by 1e-13,
// which covers the rounding of both floor(fl(.)) chains (keys and flags were computed from the same u); producer
// (whole tile) and lanes (own cells) evaluate the same monotone expressions, so a lane's cells lie inside the piece.
__device__ __forceinline__ void nb_consts(double inv_n, int nn, double& c_lo, double& c_hi) {
    const double ratio = (double)nn * inv_n;            // inv_n = fl(1 / n) from the tile descriptor: no division here
    c_lo = ratio * (1.0 - 1e-13); c_hi = ratio * (1.0 + 1e-13);
}
__device__ __forceinline__ int nb_first(int klo, double c_lo) { return max(0, __double2int_rd((double)klo * c_lo)); }
__device__ __forceinline__ int nb_last(int khi, int nn, double c_hi) { return min(nn - 1, __double2int_rd((double)(khi + 1) * c_hi)); }

// ---- a warp's output ring (row a6) ---------------------------------------------------------------------
// head / tail count rows since the kernel began (slot = count & (kRing - 1)).  `pend`: the 32 rows in pida / pidb / pc2
// have their output slots reserved (base, lane 0); lane l's ids arrive by lane l's own cp.async.
struct OutState { unsigned head, tail; unsigned pend; unsigned long long base0, base1; };    // pend: bit b = block b is reserved

__device__ __forceinline__ void pend_write(const MatchArgs& p, const WarpSm& w, int b, unsigned long long base, int lane) {
    const unsigned long long o = base + lane;
    if (o < p.capacity) { p.out_ida[o] = w.pida[b][lane]; p.out_idb[o] = w.pidb[b][lane]; p.out_sep[o] = sep_from_chord2(w.pc2[b][lane]); }
}
// everything out, now (end of the kernel, or a ring about to overflow: a tile with very many pairs).  Inlined: a call
// inside the consumer loop would make the compiler keep loop state in local memory.
__device__ __forceinline__ void ring_drain_rows(const IndexView& A, const IndexView& B, const MatchArgs& p, const WarpSm& w,
                                                unsigned head, unsigned tail, unsigned pend, unsigned long long base0, unsigned long long base1, int lane) {
    cp_async_wait_all();
    __syncwarp();
    if (pend & 1u) pend_write(p, w, 0, __shfl_sync(kFull, base0, 0), lane);
    if (pend & 2u) pend_write(p, w, 1, __shfl_sync(kFull, base1, 0), lane);
    const unsigned n = tail - head;
    if (n) {
        unsigned long long base = 0;
        if (lane == 0) base = atomicAdd(p.count, (unsigned long long)n);
        base = __shfl_sync(kFull, base, 0);
        for (unsigned k = lane; k < n; k += 32) {
            const unsigned e = (head + k) & (kRing - 1);
            const unsigned long long o = base + k;
            if (o < p.capacity) { p.out_ida[o] = __ldg(A.id + w.qa[e]); p.out_idb[o] = __ldg(B.id + w.qb[e]); p.out_sep[o] = sep_from_chord2(w.qc2[e]); }
        }
    }
    __syncwarp();
}
// append the lanes with `hit`
__device__ __forceinline__ void ring_push(const IndexView& A, const IndexView& B, const MatchArgs& p, WarpSm& w, OutState& os,
                                          bool hit, uint32_t a_row, uint32_t b_row, double c2, int lane) {
    const unsigned m = __ballot_sync(kFull, hit);
    if (m == 0) return;
    if (os.tail - os.head > (unsigned)(kRing - 32)) {
        ring_drain_rows(A, B, p, w, os.head, os.tail, os.pend, os.base0, os.base1, lane);
        os.head = os.tail; os.pend = 0;
    }
    HLC2_CHECK(os.tail - os.head + __popc(m) <= (unsigned)kRing);
    if (hit) {
        const unsigned e = (os.tail + __popc(m & ((1u << lane) - 1u))) & (kRing - 1);
        w.qa[e] = a_row; w.qb[e] = b_row; w.qc2[e] = c2;
    }
    os.tail += __popc(m);
}
// end of tile number `tile`: write the block reserved two tiles ago (its ids were requested then: every cp.async group
// but the newest is complete), then move the next full block out of the ring into that buffer, reserve its output slots
// (one global atomic) and request its ids; neither result is looked at before the tile after next
__device__ __forceinline__ void ring_step(const IndexView& A, const IndexView& B, const MatchArgs& p, WarpSm& w, OutState& os, unsigned tile, int lane) {
    const int b = (int)(tile & 1u);
    asm volatile("cp.async.wait_group 1;" ::: "memory");
    if (os.pend & (1u << b)) { pend_write(p, w, b, __shfl_sync(kFull, b ? os.base1 : os.base0, 0), lane); os.pend &= ~(1u << b); }
    if (os.tail - os.head >= 32u) {
        const unsigned e = (os.head + lane) & (kRing - 1);
        cp_async8(&w.pida[b][lane], A.id + w.qa[e]); cp_async8(&w.pidb[b][lane], B.id + w.qb[e]); w.pc2[b][lane] = w.qc2[e];
        if (lane == 0) { const unsigned long long v = atomicAdd(p.count, 32ull); if (b) os.base1 = v; else os.base0 = v; }
        os.head += 32u; os.pend |= 1u << b;
    }
    asm volatile("cp.async.commit_group;" ::: "memory");
}

// Rows flagged kKeyGeneral (window through RA = 0/360, polar rows): k_match_same appends them to a list in the caller's
// scratch (no calls inside its consumer loop), this kernel walks the general path for each of them with a whole warp:
// the lanes share the row's window and take every 32nd candidate, so that the long row ranges such rows tend to have
// (a dense strip along the RA = 0 meridian, a polar cap) are read with coalesced loads instead of lane by lane.
template <int MODE>
__global__ void __launch_bounds__(256)
k_match_general_rows(const __grid_constant__ IndexView A, const __grid_constant__ IndexView B, const __grid_constant__ MatchArgs p,
                     const uint32_t* __restrict__ list, const uint32_t* __restrict__ list_count) {
    const uint32_t n = __ldg(list_count);
    const uint32_t lane = threadIdx.x & 31u;
    for (uint32_t i = blockIdx.x * 8 + (threadIdx.x >> 5); i < n; i += gridDim.x * 8) {
        const uint32_t row = __ldg(list + i);
        Best h; h.has = false; h.c2 = 0.0; h.row = 0;
        scan_general<MODE>(A, B, p, row, __ldg(A.x + row), __ldg(A.y + row), __ldg(A.z + row), __ldg(A.pos + row), h, lane, 32u);
        __syncwarp();
        if (MODE == HLC2_NEAREST) {          // the nearest of the lanes' nearest; ties -> smaller idB
            double c = h.has ? h.c2 : 1e300;
            for (int o = 16; o; o >>= 1) c = fmin(c, __shfl_xor_sync(kFull, c, o));
            const bool cand = h.has && h.c2 == c;
            long long v = cand ? (long long)__ldg(B.id + h.row) : 0x7fffffffffffffffll;
            for (int o = 16; o; o >>= 1) v = min(v, __shfl_xor_sync(kFull, v, o));
            const unsigned m = __ballot_sync(kFull, cand && (long long)__ldg(B.id + h.row) == v);
            if (m && (int)lane == __ffs(m) - 1) emit_direct(A, B, p, row, h.row, h.c2);
        }
    }
}

// SELF: the catalogue is matched with itself (p.self_mode != 0); a template switch so that the ordinary match does not
// pay for the filters in its candidate loop
template <int MODE, bool SELF>
__global__ void __launch_bounds__(kMatchThreads, HLC2_SCTAS)
k_match_same(const __grid_constant__ IndexView A, const __grid_constant__ IndexView B, const __grid_constant__ MatchArgs p,
             uint32_t* __restrict__ glist, uint32_t* __restrict__ glist_count) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    SSmem& sm = *reinterpret_cast<SSmem*>(smem_raw);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    if (threadIdx.x == 0) {
        for (int s = 0; s < kSStages; ++s) { mbar_init(&sm.full[s], 1); mbar_init(&sm.empty[s], kCW); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    const uint32_t nt = __ldg(A.n_tiles), G = gridDim.x;

    if (warp == kCW) {
        // ---------------- producer warp ----------------
        // 32 tiles of this CTA at a time, one per lane (SIMD across tiles), in two phases whose inputs arrived long
        // before: phase 1 requests the tile descriptors of the NEXT batch, phase 2 (a dozen tiles later) turns them into
        // the tiles' windows (own zone, and the zone below / above if the descriptor's flags ask for them) and requests
        // the cell_start entries that bound them.  When a batch begins, the lanes park their results in shared memory;
        // the serial part -- one tile after the other into the stage ring -- then reads warp-uniform values.
        const uint32_t* __restrict__ cs = B.cell_start;
        uint4 q0 = make_uint4(0, 0, 0, 0), q1 = q0; uint2 q2 = make_uint2(0, 0); double q_inv = 1.0;     // the descriptor
        uint32_t o_k0g = 0, o_nk = 0, o_r0 = 0, o_r1 = 0, l_k0g = 0, l_nk = 0, l_r0 = 0, l_r1 = 0, h_k0g = 0, h_nk = 0, h_r0 = 0, h_r1 = 0;
        uint32_t l_nn = 0, h_nn = 0;
        auto phase1 = [&](uint32_t t) {
            q0 = make_uint4(0, 0, 0, 0); q1 = make_uint4(0, 0, 1, 0); q2 = make_uint2(0, 0); q_inv = 1.0;
            if (t < nt) {
                const uint4* d = reinterpret_cast<const uint4*>(A.tiles + t);
                q0 = __ldg(d); q1 = __ldg(d + 1);
                const uint4 v = __ldg(d + 2); q2 = make_uint2(v.x, v.y); q_inv = __hiloint2double((int)v.w, (int)v.z);
            }
        };
        auto phase2 = [&]() {
            o_k0g = 0; o_nk = 0; o_r0 = 0; o_r1 = 0; l_nn = 0; h_nn = 0;
            if (q0.y) {
                const int n = (int)q1.z;
                const uint32_t cb = q1.w;
                const int ka = max((int)q0.w - 1, 0), kb = min((int)q1.x + 1, n - 1);
                o_k0g = cb + (uint32_t)ka; o_nk = (uint32_t)(kb - ka + 1);
                o_r0 = __ldg(cs + o_k0g); o_r1 = __ldg(cs + o_k0g + o_nk);
                if ((q1.y & kTileDecLo) && q2.x) {
                    l_nn = q2.x;
                    double c_lo, c_hi; nb_consts(q_inv, (int)l_nn, c_lo, c_hi);
                    const int k0 = nb_first(ka, c_lo), k1 = nb_last(kb, (int)l_nn, c_hi);
                    l_k0g = cb - l_nn + (uint32_t)k0; l_nk = (uint32_t)(k1 - k0 + 1);
                    l_r0 = __ldg(cs + l_k0g); l_r1 = __ldg(cs + l_k0g + l_nk);
                }
                if ((q1.y & kTileDecHi) && q2.y) {
                    h_nn = q2.y;
                    double c_lo, c_hi; nb_consts(q_inv, (int)h_nn, c_lo, c_hi);
                    const int k0 = nb_first(ka, c_lo), k1 = nb_last(kb, (int)h_nn, c_hi);
                    h_k0g = cb + (uint32_t)n + (uint32_t)k0; h_nk = (uint32_t)(k1 - k0 + 1);
                    h_r0 = __ldg(cs + h_k0g); h_r1 = __ldg(cs + h_k0g + h_nk);
                }
            }
        };
        auto park = [&]() {             // this lane's tile -> shared memory (waits for phase 2's loads: requested long ago)
            uint4* r = reinterpret_cast<uint4*>(&sm.rec[lane]);
            r[0] = make_uint4(q0.x, q0.y, q1.w, q1.z); r[1] = make_uint4(o_k0g, o_nk, o_r0, o_r1);
            r[2] = make_uint4(l_k0g, l_nk, l_r0, l_r1); r[3] = make_uint4(h_k0g, h_nk, h_r0, h_r1);
            r[4] = make_uint4(l_nn, h_nn, (uint32_t)__double2loint(q_inv), (uint32_t)__double2hiint(q_inv));
        };
        uint32_t it = 0;
        uint32_t a_first = 0, a_count = 0, cb_own = 0; double inv_own = 1.0;
        // one piece -> stages (row chunks of <= kSBCap).  fl_first / fl_last: the tile's first / last piece
        auto piece = [&](uint32_t kind, bool fl_first, bool fl_last, uint32_t k0g, uint32_t nk, uint32_t r0, uint32_t r1, uint32_t cb_nb, int nn) {
            const uint32_t cs_al = k0g & ~3u;
            uint32_t c_ld = ((k0g + nk + 1u + 3u) & ~3u) - cs_al;
            const bool wide = c_ld > (uint32_t)kSCsCap;
            if (wide) { c_ld = 0; r1 = r0; }
            double c_lo = 0.0, c_hi = 0.0;
            if (kind) nb_consts(inv_own, nn, c_lo, c_hi);
            uint32_t r = r0;
            bool first = fl_first;
            for (;;) {
                const uint32_t row_al = r & ~1u;
                const uint32_t re = min(r1, row_al + (uint32_t)kSBCap - 1u);
                const bool last = re >= r1;
                const uint32_t n_ld = wide ? 0u : ((re + 1u) & ~1u) - row_al;
                const uint32_t flags = kind | (wide ? kSWide : 0u) | (first ? kSFirst : 0u) | (last && fl_last ? kSLast : 0u);
                const int s = (int)(it % kSStages);
                mbar_wait(&sm.empty[s], ((it / kSStages) & 1u) ^ 1u);
                SStage& st = sm.st[s];
                // the tile's first stage takes its A rows along
                const uint32_t a_al = a_first & ~1u, k_al = a_first & ~3u;
                const uint32_t a_ld = first ? ((a_first + a_count + 1u) & ~1u) - a_al : 0u, k_ld = first ? ((a_first + a_count + 3u) & ~3u) - k_al : 0u;
                const uint32_t bytes = n_ld * 24u + c_ld * 4u + a_ld * 24u + k_ld * 4u;
                HLC2_CHECK(n_ld <= (uint32_t)kSBCap && c_ld <= (uint32_t)kSCsCap && a_ld <= (uint32_t)kTile + 2u && k_ld <= (uint32_t)kTile + 4u);
                if (lane == 0) {
                    uint4* d = reinterpret_cast<uint4*>(&st.d);
                    d[0] = make_uint4(flags, cs_al, row_al, r); d[1] = make_uint4(re, (uint32_t)nn, a_first, a_count);
                    d[2] = make_uint4(a_first - a_al, a_first - k_al, cb_own, cb_nb);
                    st.d.c_lo = c_lo; st.d.c_hi = c_hi;
                    if (bytes) mbar_arrive_expect_tx(&sm.full[s], bytes); else mbar_arrive(&sm.full[s]);
                }
                __syncwarp();
                if (n_ld && lane < 3) {
                    const double* src = lane == 0 ? B.x : lane == 1 ? B.y : B.z;
                    double* dst = lane == 0 ? st.bx : lane == 1 ? st.by : st.bz;
                    bulk_g2s(dst, src + row_al, n_ld * 8u, &sm.full[s]);
                }
                if (c_ld && lane == 3) bulk_g2s(st.cs, cs + cs_al, c_ld * 4u, &sm.full[s]);
                if (a_ld && lane >= 4 && lane < 7) {
                    const double* src = lane == 4 ? A.x : lane == 5 ? A.y : A.z;
                    double* dst = lane == 4 ? st.ax : lane == 5 ? st.ay : st.az;
                    bulk_g2s(dst, src + a_al, a_ld * 8u, &sm.full[s]);
                }
                if (k_ld && lane == 7) bulk_g2s(st.ak, A.key + k_al, k_ld * 4u, &sm.full[s]);
                ++it;
                if (last) break;
                r = re; first = false;
            }
        };
        phase1(blockIdx.x + (uint32_t)lane * G);
        phase2();
        for (uint32_t base = blockIdx.x; base < nt; base += 32u * G) {
            park();
            __syncwarp();
            phase1(base + (32u + (uint32_t)lane) * G);                  // the next batch's descriptors
            for (uint32_t i = 0; i < 32u && base + i * G < nt; ++i) {
                if (i == 12u) phase2();                                  // ... have long arrived: its windows
                const uint4* r = reinterpret_cast<const uint4*>(&sm.rec[i]);
                const uint4 r0 = r[0], r1 = r[1], r4 = r[4];
                a_first = r0.x; a_count = r0.y; cb_own = r0.z;
                inv_own = __hiloint2double((int)r4.w, (int)r4.z);
                piece(0u, true, r4.x == 0u && r4.y == 0u, r1.x, r1.y, r1.z, r1.w, cb_own, (int)r0.w);
                if (r4.x) { const uint4 r2 = r[2]; piece(kSLo, false, r4.y == 0u, r2.x, r2.y, r2.z, r2.w, cb_own - r4.x, (int)r4.x); }
                if (r4.y) { const uint4 r3 = r[3]; piece(kSHi, false, true, r3.x, r3.y, r3.z, r3.w, cb_own + r0.w, (int)r4.y); }
            }
            if (nt - base <= 12u * G) phase2();                         // a short last batch never reached tile 12 (nothing follows: harmless)
            __syncwarp();
        }
        {   // tell the consumers that nothing follows
            const int s = (int)(it % kSStages);
            mbar_wait(&sm.empty[s], ((it / kSStages) & 1u) ^ 1u);
            if (lane == 0) { sm.st[s].d.flags = kSEnd; mbar_arrive(&sm.full[s]); }
        }
        return;
    }

    // ---------------- consumer warps: one lane per A row ----------------
    WarpSm& w = sm.w[warp];
    OutState os; os.head = 0; os.tail = 0; os.pend = 0; os.base0 = 0; os.base1 = 0;
    unsigned tile = 0;
    Best best; best.has = false; best.c2 = 0.0; best.row = 0;
    double ax = 0.0, ay = 0.0, az = 0.0; uint32_t kf = 0;
    for (uint32_t it = 0;; ++it) {
        const int s = (int)(it % kSStages);
        mbar_wait(&sm.full[s], (it / kSStages) & 1u);
        const SStage& st = sm.st[s];
        const uint4 dv = reinterpret_cast<const uint4*>(&st.d)[0];          // flags, cs_al, row_al, row_lo
        const uint4 dw = reinterpret_cast<const uint4*>(&st.d)[1];          // row_hi, nn, a_first, a_count
        const uint32_t flags = dv.x;
        if (flags & kSEnd) break;
        const bool mine = threadIdx.x < dw.w;
        const uint32_t a_row = dw.z + threadIdx.x;
        if (flags & kSFirst) {            // a new tile: its rows came with this stage
            const unsigned ra = (mine ? threadIdx.x : 0u) + st.d.a_off;
            HLC2_CHECK(ra < (unsigned)kTile + 2u && (mine ? threadIdx.x : 0u) + st.d.k_off < (unsigned)kTile + 4u);
            ax = st.ax[ra]; ay = st.ay[ra]; az = st.az[ra]; kf = st.ak[(mine ? threadIdx.x : 0u) + st.d.k_off];
            best.has = false;
            const bool gen = mine && (kf >> 30) == 3u;
            const unsigned m = __ballot_sync(kFull, gen);                 // rare: window through RA = 0/360, polar rows
            if (m) {
                uint32_t slot = 0;
                if (lane == 0) slot = atomicAdd(glist_count, (uint32_t)__popc(m));
                slot = __shfl_sync(kFull, slot, 0);
                if (gen) glist[slot + __popc(m & ((1u << lane) - 1u))] = a_row;
            }
        }
        const bool general = (kf >> 30) == 3u;
        const uint32_t key = kf & kKeyMask;
        const int elo = (int)((kf >> 28) & 1u), ehi = (int)((kf >> 29) & 1u);
        bool act = mine && !general;
        uint32_t c0, c1;                   // the lane's cells as global cell numbers [c0, c1]
        uint32_t self_lo = 0;              // self-match, every unordered pair once: only B rows behind the A row count
        if ((flags & (kSLo | kSHi)) == 0u) {
            c0 = key - (uint32_t)elo; c1 = key + (uint32_t)ehi;
            if (SELF) { if (p.self_mode == 1) self_lo = a_row + 1u; else if (p.self_mode == 2) self_lo = a_row; }
        } else {
            act = act && (kf & ((flags & kSLo) ? kKeyDecLo : kKeyDecHi)) != 0u;
            if (SELF && (flags & kSLo) && (p.self_mode == 1 || p.self_mode == 2)) act = false;      // the zone below holds earlier rows only
            const int k = (int)(key - st.d.cb_own);
            c0 = st.d.cb_nb + (uint32_t)nb_first(k - elo, st.d.c_lo); c1 = st.d.cb_nb + (uint32_t)nb_last(k + ehi, (int)dw.y, st.d.c_hi);
        }
        if (flags & kSWide) {
            if (act) scan_global<MODE>(A, B, p, a_row, ax, ay, az, __ldg(B.cell_start + c0), __ldg(B.cell_start + c1 + 1u), best);
            __syncwarp();
        } else {
            unsigned p0 = 0, len = 0;
            if (act) {
                HLC2_CHECK(c0 >= dv.y && c0 <= c1 && c1 + 1u - dv.y < (uint32_t)kSCsCap);
                const uint32_t q1 = min(max(st.cs[c1 + 1u - dv.y], dv.w), dw.x);
                const uint32_t q0 = SELF ? min(max(max(st.cs[c0 - dv.y], dv.w), self_lo), q1) : min(max(st.cs[c0 - dv.y], dv.w), dw.x);
                p0 = q0 - dv.z; len = q1 - q0;
                HLC2_CHECK(q0 >= dv.z && q1 - dv.z <= (uint32_t)kSBCap);
            }
            const unsigned mx = __reduce_max_sync(kFull, len);
            // a lane past its own range keeps reading on (rows of other lanes, at worst the arrays behind bx: all inside
            // the stage) and ignores what it sees: no index clamp in the loop
            for (unsigned i = 0; i < mx; ++i) {
                const bool in = i < len;
                const unsigned j = p0 + i;
                const double dx = ax - st.bx[j], dy = ay - st.by[j], dz = az - st.bz[j];
                const double c2v = fma(dx, dx, fma(dy, dy, dz * dz));
                const uint32_t r = j + dv.z;
                const bool hit = in && c2v <= p.thr2 && (!SELF || p.self_mode != 3 || r != a_row);
                if (hit) {
                    if (MODE == HLC2_ALL_PAIRS) {
                        // a lane holds its first pair of the tile (queued with everybody's at the tile's end: one ballot per
                        // tile instead of one per step); a second pair for the same A row is rare and goes straight out
                        if (best.has) emit_direct(A, B, p, a_row, r, c2v);
                        else { best.has = true; best.row = r; best.c2 = c2v; }
                    } else if (!best.has || c2v < best.c2 || (c2v == best.c2 && __ldg(B.id + r) < __ldg(B.id + best.row))) {
                        best.has = true; best.row = r; best.c2 = c2v;      // ties -> smaller idB: ids are only fetched on an exact tie
                    }
                }
            }
        }
        const bool last = (flags & kSLast) != 0u;
        if (last) ring_push(A, B, p, w, os, mine && !general && best.has, a_row, best.row, best.c2, lane);
        __syncwarp();
        if (lane == 0) mbar_arrive(&sm.empty[s]);
        if (last) { ring_step(A, B, p, w, os, tile, lane); ++tile; }
    }
    __syncwarp();
    ring_drain_rows(A, B, p, w, os.head, os.tail, os.pend, os.base0, os.base1, lane);
}

// every A row through the general per-lane path (per-record radii; a self-match whose grid does not qualify for the
// same-grid kernel): one lane per row, windows from the fp32 estimate, B through L2
template <int MODE>
__global__ void __launch_bounds__(256)
k_match_all_general(const __grid_constant__ IndexView A, const __grid_constant__ IndexView B, const __grid_constant__ MatchArgs p) {
    for (uint32_t row = blockIdx.x * 256 + threadIdx.x; row < A.n; row += gridDim.x * 256) {
        Best h; h.has = false; h.c2 = 0.0; h.row = 0;
        scan_general<MODE>(A, B, p, row, __ldg(A.x + row), __ldg(A.y + row), __ldg(A.z + row), __ldg(A.pos + row), h);
        if (MODE == HLC2_NEAREST && h.has) emit_direct(A, B, p, row, h.row, h.c2);
    }
}

void launch_match_all_general(const IndexView& A, const IndexView& B, const MatchArgs& p, int mode, cudaStream_t s,
                              cudaEvent_t ev_start, cudaEvent_t ev_stop) {
    const unsigned blocks = (unsigned)std::max<size_t>(1, std::min<size_t>(((size_t)A.n + 255) / 256, (size_t)sm_count() * 8));
    if (ev_start) cudaEventRecord(ev_start, s);
    if (mode == HLC2_NEAREST) k_match_all_general<HLC2_NEAREST><<<blocks, 256, 0, s>>>(A, B, p);
    else                      k_match_all_general<HLC2_ALL_PAIRS><<<blocks, 256, 0, s>>>(A, B, p);
    count_launch();
    if (ev_stop) cudaEventRecord(ev_stop, s);
}

size_t match_same_temp_bytes(const IndexView& A) { return 256 + (size_t)A.n * sizeof(uint32_t); }

void launch_match_same(const IndexView& A, const IndexView& B, const MatchArgs& p, int mode, void* d_temp, cudaStream_t s,
                       cudaEvent_t ev_start, cudaEvent_t ev_stop) {
    const int m = mode == HLC2_NEAREST ? 1 : 0;
    const bool self = p.self_mode != 0;
    const void* kern = self ? (m == 0 ? (const void*)k_match_same<HLC2_ALL_PAIRS, true> : (const void*)k_match_same<HLC2_NEAREST, true>)
                            : (m == 0 ? (const void*)k_match_same<HLC2_ALL_PAIRS, false> : (const void*)k_match_same<HLC2_NEAREST, false>);
    static int per_sm_dev[kMaxDevices][4] = {};        // resident CTAs per SM; the smem opt-in is per device
    int* per_sm = per_sm_dev[current_device()];
    const size_t smem = sizeof(SSmem);
    const int mi = m + (self ? 2 : 0);
    if (!per_sm[mi]) {
        int v = 0;
        cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        cudaOccupancyMaxActiveBlocksPerMultiprocessor(&v, kern, kMatchThreads, smem);
        per_sm[mi] = v > 0 ? v : 1;
    }
    // scratch: 256-byte header (count of general rows), then their row numbers
    uint32_t* glist_count = reinterpret_cast<uint32_t*>(d_temp);
    uint32_t* glist = reinterpret_cast<uint32_t*>(reinterpret_cast<char*>(d_temp) + 256);
    cudaMemsetAsync(glist_count, 0, sizeof(uint32_t), s);
    // persistent grid: SM count x resident CTAs, never more CTAs than tiles
    const unsigned blocks = (unsigned)std::max<size_t>(1, std::min<size_t>(A.tile_cap, (size_t)sm_count() * per_sm[mi]));
    if (ev_start) cudaEventRecord(ev_start, s);          // the caller's events bracket the match kernels (hlc2_crossmatch_events)
    void* kargs[5] = {(void*)&A, (void*)&B, (void*)&p, (void*)&glist, (void*)&glist_count};
    cudaLaunchKernel(kern, dim3(blocks), dim3(kMatchThreads), kargs, smem, s);
    count_launch();
    const unsigned gblocks = (unsigned)sm_count() * 4;
    if (m == 0) k_match_general_rows<HLC2_ALL_PAIRS><<<gblocks, 256, 0, s>>>(A, B, p, glist, glist_count);
    else        k_match_general_rows<HLC2_NEAREST><<<gblocks, 256, 0, s>>>(A, B, p, glist, glist_count);
    count_launch();
    if (ev_stop) cudaEventRecord(ev_stop, s);
}

}  // namespace hlc2
