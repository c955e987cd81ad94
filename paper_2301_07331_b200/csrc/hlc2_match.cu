// hlc2_match.cu -- the match kernels (NS (b)).
//
// One thread per A source (the paper's thread-per-A-record hierarchy), but
// instead of looping over a whole calculation block (L271) each thread visits only the B
// cells its search window can reach:
//   dec window  [dec - r, dec + r]                         -> 1..3 zones of B's grid
//   RA  window  [ra - w, ra + w], w = asin(sin r / cos dec) -> 1..2 contiguous cell ranges per zone
//               (full ring when cos dec <= ~4 sin r, i.e. at the poles; two ranges when the
//               window crosses RA = 0/360).  These are the cells the quad-direction strategy
//               probes (L122-169) plus the diagonal neighbours and the 1/cos(dec) widening it
//               omits, so no pair is lost (the "No Index" result, L344).
// The window is located from an fp32 estimate of the source's (ra, dec) padded by a rigorous
// error bound; over-inclusion only costs time.  Decisions are fp64: chord^2 <= 4 sin^2(r/2).
// Hits are queued per CTA in shared memory and flushed with ONE global atomic per CTA into
// the compacted (idA, idB, sep) output (the role of d_out_dis, L282).
#include <math.h>

#include "hlc2_grid.cuh"

namespace hlc2 {

constexpr int kMatchThreads = 256;
constexpr int kQueueCap = 1024;
constexpr double kRad2Arcsec = 206264.80624709636;   // 648000 / pi

// padding of the fp32 position estimate (degrees): atan2f (<= 2 ulp) on fp32-rounded unit-vector
// components, then the degree conversion.  Derived in DESIGN.md; ~3x the worst-case bound.
constexpr double kEpsRaDeg = 2.5e-4;
constexpr double kEpsDecDeg = 1.5e-4;

struct MatchArgs {
    double thr2;          // 4 sin^2(r/2)
    double r_deg;         // radius in degrees
    float sin_r_up;       // sin(r) * (1 + 1e-5)
    int64_t* out_ida; int64_t* out_idb; double* out_sep;
    unsigned long long capacity;
    unsigned long long* count;
};

__device__ __forceinline__ double sep_from_chord2(double c2) {
    return 2.0 * asin(fmin(1.0, 0.5 * sqrt(c2))) * kRad2Arcsec;
}

template <int MODE>
__global__ void __launch_bounds__(kMatchThreads)
k_match(IndexView A, IndexView B, MatchArgs p) {
    __shared__ uint32_t q_a[kQueueCap], q_b[kQueueCap];
    __shared__ double q_c2[kQueueCap];
    __shared__ unsigned q_n;
    __shared__ unsigned long long q_base;
    if (threadIdx.x == 0) q_n = 0;
    __syncthreads();

    const uint32_t i = blockIdx.x * kMatchThreads + threadIdx.x;
    const GridView& g = B.g;
    if (i < A.n && B.n > 0) {
        const double ax = __ldg(A.x + i), ay = __ldg(A.y + i), az = __ldg(A.z + i);
        const float fx = (float)ax, fy = (float)ay, fz = (float)az;
        const float rxy = sqrtf(fx * fx + fy * fy);
        float ra_f = atan2f(fy, fx) * 57.29577951f;
        if (ra_f < 0.0f) ra_f += 360.0f;
        const float dec_f = atan2f(fz, rxy) * 57.29577951f;
        const double dlo = (double)dec_f - (p.r_deg + kEpsDecDeg), dhi = (double)dec_f + (p.r_deg + kEpsDecDeg);

        double best_c2 = INFINITY; uint32_t best_j = 0;

        if (!(dhi < g.dec_min) && !(dlo > g.dec_max)) {
            const float s = p.sin_r_up / rxy;                        // sin(dRA_max) = sin r / cos dec
            const bool ring = !(s < 0.25f);
            const double w = ring ? 360.0 : (double)(s * (1.011f * 57.29577951f)) + kEpsRaDeg;   // asin(s) <= 1.011 s
            const double u = box_u(g, (double)ra_f);
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
#pragma unroll 1
                for (int seg = 0; seg < 2; ++seg) {
                    const int ka = seg ? k2 : k0, kb = seg ? k3 : k1;
                    if (kb < ka) continue;
                    const uint32_t j0 = __ldg(B.cell_start + base + ka), j1 = __ldg(B.cell_start + base + kb + 1);
                    for (uint32_t j = j0; j < j1; ++j) {
                        const double dx = ax - __ldg(B.x + j), dy = ay - __ldg(B.y + j), dz = az - __ldg(B.z + j);
                        const double c2 = dx * dx + dy * dy + dz * dz;
                        if (c2 <= p.thr2) {
                            if (MODE == HLC2_ALL_PAIRS) {
                                unsigned slot = atomicAdd(&q_n, 1u);
                                if (slot < kQueueCap) { q_a[slot] = i; q_b[slot] = j; q_c2[slot] = c2; }
                                else {      // queue full (very dense sky): emit directly
                                    unsigned long long o = atomicAdd(p.count, 1ull);
                                    if (o < p.capacity) {
                                        p.out_ida[o] = __ldg(A.id + i); p.out_idb[o] = __ldg(B.id + j);
                                        p.out_sep[o] = sep_from_chord2(c2);
                                    }
                                }
                            } else {
                                if (c2 < best_c2 || (c2 == best_c2 && __ldg(B.id + j) < __ldg(B.id + best_j))) { best_c2 = c2; best_j = j; }
                            }
                        }
                    }
                }
            }
        }
        if (MODE == HLC2_NEAREST && best_c2 <= p.thr2) {
            unsigned slot = atomicAdd(&q_n, 1u);       // <= one per thread: never overflows
            q_a[slot] = i; q_b[slot] = best_j; q_c2[slot] = best_c2;
        }
    }
    __syncthreads();
    const unsigned nq = min(q_n, (unsigned)kQueueCap);
    if (threadIdx.x == 0 && nq) q_base = atomicAdd(p.count, (unsigned long long)nq);
    __syncthreads();
    for (unsigned k = threadIdx.x; k < nq; k += kMatchThreads) {
        unsigned long long o = q_base + k;
        if (o < p.capacity) {
            p.out_ida[o] = __ldg(A.id + q_a[k]); p.out_idb[o] = __ldg(B.id + q_b[k]);
            p.out_sep[o] = sep_from_chord2(q_c2[k]);
        }
    }
}

size_t match_temp_bytes(const IndexView&, const IndexView&) { return 0; }

void launch_match(const IndexView& A, const IndexView& B, double radius_arcsec, int mode,
                  int64_t* out_ida, int64_t* out_idb, double* out_sep, unsigned long long capacity,
                  unsigned long long* d_count, void* d_temp, cudaStream_t s) {
    (void)d_temp;
    if (A.n == 0) return;
    MatchArgs p;
    long double r_rad = (long double)radius_arcsec * (3.141592653589793238462643383279502884L / 648000.0L);
    long double h = sinl(0.5L * r_rad);
    p.thr2 = (double)(4.0L * h * h);
    p.r_deg = radius_arcsec / 3600.0;
    p.sin_r_up = (float)((double)sinl(r_rad) * (1.0 + 1e-5));
    p.out_ida = out_ida; p.out_idb = out_idb; p.out_sep = out_sep; p.capacity = capacity; p.count = d_count;
    unsigned blocks = (unsigned)(((size_t)A.n + kMatchThreads - 1) / kMatchThreads);
    if (mode == HLC2_NEAREST) k_match<HLC2_NEAREST><<<blocks, kMatchThreads, 0, s>>>(A, B, p);
    else                      k_match<HLC2_ALL_PAIRS><<<blocks, kMatchThreads, 0, s>>>(A, B, p);
    count_launch();
}

}  // namespace hlc2
