// hlc2_grid.cuh -- the zone/cell grid arithmetic shared by the index build (which files every
// source under one cell key) and the match kernel (which maps a search window onto cell
// ranges).  Both sides MUST evaluate the same monotone floor(fl(.)) expressions so that a
// conservatively padded real interval always maps onto a superset of the cells its sources
// were filed under (the role of hp_nestid in PAPER.md Alg. 1).
#pragma once
#include "hlc2_internal.cuh"

namespace hlc2 {

// RA reduced into [0, 360).  360.0 == 0.0 (Table 2 prints 360.0000, L292); -0.0 acts as 0.
__device__ __forceinline__ double norm_ra(double ra) {
    if (!(ra >= 0.0 && ra < 360.0)) {
        ra = fmod(ra, 360.0);
        if (ra < 0.0) ra += 360.0;
        if (!(ra < 360.0)) ra = 0.0;        // -tiny + 360 rounds to 360; NaN lands here too
    }
    return ra;
}

__device__ __forceinline__ bool coord_ok(double ra, double dec) {
    return isfinite(ra) && dec >= -90.0 && dec <= 90.0;
}

// zone of a declination (deg); monotone non-decreasing in dec
__device__ __forceinline__ int zone_of(const GridView& g, double dec) {
    const int z = __double2int_rd((dec - g.dec_lo) * g.inv_h);      // floor, saturating; clamps are integer ops
    return min(max(z, 0), g.n_zones - 1);
}

// box-relative RA coordinate of a normalised RA: u in [0, 360]
__device__ __forceinline__ double box_u(const GridView& g, double ra_norm) {
    double u = ra_norm - g.ra0;
    if (u < 0.0) u += 360.0;
    return u;
}

// RA cell of box coordinate u (u >= 0) in a zone with n cells; monotone non-decreasing in u
__device__ __forceinline__ int cell_of_u(const GridView& g, double u, int n) {
    const int k = __double2int_rd((u * g.inv_span) * (double)n);
    return min(max(k, 0), n - 1);
}

// order-preserving map fp64 -> uint64 (for atomicMin / atomicMax on doubles)
__host__ __device__ __forceinline__ unsigned long long f64_order_bits(double v) {
#ifdef __CUDA_ARCH__
    long long b = __double_as_longlong(v);
#else
    long long b; memcpy(&b, &v, 8);
#endif
    return b < 0 ? ~(unsigned long long)b : ((unsigned long long)b | 0x8000000000000000ull);
}
__host__ __device__ __forceinline__ double f64_from_order_bits(unsigned long long u) {
    long long b = (u & 0x8000000000000000ull) ? (long long)(u & 0x7FFFFFFFFFFFFFFFull) : (long long)~u;
#ifdef __CUDA_ARCH__
    return __longlong_as_double(b);
#else
    double v; memcpy(&v, &b, 8); return v;
#endif
}

}  // namespace hlc2
