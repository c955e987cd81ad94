// hlc2_internal.cuh -- shared declarations of the CUDA path (sm_100a).  Not part of the ABI.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <vector>

#include "../../include/hlc2.h"

namespace hlc2 {

constexpr int kRaBins = 4096;                 // coarse RA histogram of the extent pass
constexpr double kRaBinDeg = 360.0 / kRaBins; // 0.087890625, exact
constexpr uint32_t kMaxN = 0xFFFFFFFEu;

// ---- grid as the kernels see it (passed by value) ----------------------------------------
struct GridView {
    const int32_t* n_ra;        // [n_zones] RA cells per zone
    const uint32_t* cell_base;  // [n_zones + 1] first cell key of each zone
    double dec_lo;              // south edge of zone 0 (deg)
    double inv_h;               // 1 / zone height (1/deg)
    double ra0;                 // west edge of the RA box (deg)
    double span;                // RA extent of the box (deg), 360 = full ring
    double inv_span;
    double dec_min, dec_max;    // exact data extent (deg)
    int32_t n_zones;
    uint32_t n_cells;
};

struct IndexView {
    const double* x; const double* y; const double* z;   // [n] unit vectors, cell order
    const int64_t* id;                                    // [n]
    const uint32_t* cell_start;                           // [n_cells + 1]
    GridView g;
    uint32_t n;
};

// extent statistics written by the stats pass
struct Stats {
    unsigned long long dec_min_bits;   // order-preserving encoding of the fp64 value
    unsigned long long dec_max_bits;
    unsigned long long first_bad_row;  // ~0 = none
    unsigned long long n_bad;
    uint32_t ra_hist[kRaBins];
};

// ---- launchers (hlc2_build.cu, hlc2_match.cu) --------------------------------------------
void launch_stats(const double* ra, const double* dec, uint32_t n, Stats* d_stats, cudaStream_t s);
void launch_keys(const double* ra, const double* dec, uint32_t n, GridView g, uint32_t* keys, cudaStream_t s);
// sorts (keys, row) by key; returns which of the double buffers holds the result (0 = a, 1 = b)
int  launch_radix_sort(uint32_t* keys_a, uint32_t* keys_b, uint32_t* val_a, uint32_t* val_b, uint32_t n,
                       int key_bits, uint32_t* d_counts, size_t counts_entries, uint32_t* d_partials, cudaStream_t s);
void launch_gather(const double* ra, const double* dec, const int64_t* id, const uint32_t* perm, uint32_t n,
                   double* x, double* y, double* z, int64_t* out_id, cudaStream_t s);
void launch_cell_table(const uint32_t* sorted_keys, uint32_t n, uint32_t n_cells, uint32_t* cell_start,
                       uint32_t* d_partials, cudaStream_t s);
size_t sort_counts_entries(uint32_t n);      // entries of the digit-count array for n keys
size_t scan_partials_entries(size_t m);      // entries of the partial-sum array for a scan over m entries

void launch_match(const IndexView& A, const IndexView& B, double radius_arcsec, int mode,
                  int64_t* out_ida, int64_t* out_idb, double* out_sep, unsigned long long capacity,
                  unsigned long long* d_count, cudaStream_t s);

void count_launch(int k = 1);

}  // namespace hlc2
