// hlc2_internal.cuh -- shared declarations of the CUDA path (sm_100a).  Not part of the ABI.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <vector>

#include "../../include/hlc2.h"

namespace hlc2 {

constexpr int kRaBins = 4096;                 // coarse RA histogram of the extent pass
constexpr double kRaBinDeg = 360.0 / kRaBins; // 0.087890625, exact
constexpr uint32_t kMaxN = (1u << 30) - 1;    // the radix sort's chained scan keeps 2 flag bits beside a 30-bit count

constexpr int kRadixBits = 9;                 // LSD radix sort digit
constexpr int kRadix = 1 << kRadixBits;
constexpr int kMaxPasses = 4;                 // 32-bit keys
#ifndef HLC2_TILE
#define HLC2_TILE 128
#endif
constexpr int kTile = HLC2_TILE;                    // sources per match tile (= threads of the match CTA)

// Window flags of a source on its own grid, kept in the top bits of its 32-bit cell key (grids of <= 2^28 cells).  They
// say which cells around the source's own cell a search window of radius <= r_max can reach, so a match between two
// indices that share one grid (opts.grid_like) needs no per-row window arithmetic:
//   kKeyExtLo / kKeyExtHi  the window reaches into the previous / next RA cell of the source's zone
//   kKeyDecLo / kKeyDecHi  it reaches into the zone below / above (never further: zones are at least r_max high)
//   kKeyGeneral (both Dec bits)  anything else -- the window passes RA = 0/360, is wider than one cell (polar rows),
//                          or touches both neighbouring zones: such rows take the general per-lane path
constexpr int kKeyFlagShift = 28;
constexpr uint32_t kKeyMask = (1u << kKeyFlagShift) - 1u;
constexpr uint32_t kKeyExtLo = 1u << 28, kKeyExtHi = 1u << 29, kKeyDecLo = 1u << 30, kKeyDecHi = 1u << 31;
constexpr uint32_t kKeyGeneral = kKeyDecLo | kKeyDecHi;

// ---- grid as the kernels see it (passed by value) ----------------------------------------
struct GridView {
    const int32_t* n_ra;        // [n_zones] RA cells per zone
    const uint32_t* cell_base;  // [n_zones + 1] first cell key of each zone
    double dec_lo;              // south edge of zone 0 (deg)
    double h;                   // zone height (deg)
    double inv_h;               // 1 / zone height (1/deg)
    double ra0;                 // west edge of the RA box (deg)
    double span;                // RA extent of the box (deg), 360 = full ring
    double inv_span;
    double dec_min, dec_max;    // exact data extent (deg)
    int32_t n_zones;
    uint32_t n_cells;
};

// tile of the cell-sorted catalogue: rows [first, first + count) all lie in `zone`, in its cells k_first..k_last
// flags: which neighbours some row of the tile reaches (OR of the rows' window flags)
constexpr uint32_t kTileDecLo = 1u, kTileDecHi = 2u, kTileGeneral = 4u;
// besides its rows the descriptor carries what a match needs to know about the tile's zone and its neighbours, so that
// no look-up depends on another one: RA cells n of the zone (and 1 / n), first cell key cb, cells of the zones below / above
struct TileDesc {
    uint32_t first, count, zone, k_first;
    uint32_t k_last, flags, n, cb;
    uint32_t n_lo, n_hi; double inv_n;          // n_lo / n_hi = 0: no such zone
};
static_assert(sizeof(TileDesc) == 48, "TileDesc is read as three 16-byte words");

struct IndexView {
    const double* x; const double* y; const double* z;   // [n] unit vectors, cell order
    const int64_t* id;                                    // [n]
    const float2* pos;                                    // [n] fp32 (ra, dec) estimate in degrees: locates windows, never decides
    const double* err2;                                   // [n] squared error radius (arcsec^2) of each sorted row, or null
    const uint32_t* key;                                  // [n] sorted cell keys (& key_mask), window flags in the top bits
    uint32_t key_mask;                                    // kKeyMask when the keys carry flags, else 0xFFFFFFFF
    const uint32_t* cell_start;                           // [n_cells + 1]
    const TileDesc* tiles;                                // [*n_tiles]
    const uint32_t* n_tiles;                              // device scalar
    GridView g;
    uint32_t n;
    uint32_t tile_cap;                                    // host-side upper bound of *n_tiles
};

// packed per-source record in INPUT order, written by the key pass and read (one sector) by the gather
struct __align__(32) Rec { double ra, dec, spare; long long id; };     // ra normalised to [0, 360); NaNs: bad row

// extent statistics written by the stats pass
struct Stats {
    unsigned long long dec_min_bits;   // order-preserving encoding of the fp64 value
    unsigned long long dec_max_bits;
    unsigned long long first_bad_row;  // ~0 = none
    unsigned long long n_bad;
    uint32_t ra_hist[kRaBins];
};

// ---- launchers (hlc2_build.cu, hlc2_match.cu) --------------------------------------------
constexpr int kMaxDevices = 64;               // per-device caches of function attributes and device properties
int current_device();
int sm_count();
void launch_stats(const double* ra, const double* dec, uint32_t n, Stats* d_stats, cudaStream_t s);
void launch_keys_pack(const double* ra, const double* dec, const int64_t* id, uint32_t n, GridView g, int passes,
                      double r_max_arcsec, bool flagged, uint32_t* keys, Rec* rec, uint32_t* digit_hist, cudaStream_t s,
                      Stats* collect = nullptr);
void launch_stats_init(Stats* d_stats, cudaStream_t s);
void note_cuda_error(cudaError_t e);          // what hlc2_last_cuda_error reports (thread-local, hlc2_api.cu)
int  radix_passes(int key_bits);
size_t sort_tiles(uint32_t n);
// sorts (keys, row) by key; returns which of the double buffers holds the result (0 = a, 1 = b)
int  launch_radix_sort(uint32_t* keys_a, uint32_t* keys_b, uint32_t* val_a, uint32_t* val_b, uint32_t n, int key_bits,
                       const uint32_t* d_digit_hist, uint32_t* d_digit_base, uint32_t* d_status, uint32_t* d_ticket,
                       cudaStream_t s);
void launch_gather(const Rec* rec, const uint32_t* perm, uint32_t n, double* x, double* y, double* z, int64_t* out_id,
                   float2* pos, cudaStream_t s);
void launch_gather_err2(const double* err_arcsec, const uint32_t* perm, uint32_t n, double* err2, cudaStream_t s);
size_t cell_big_cap(size_t n_cells);
void launch_cell_table(const uint32_t* sorted_keys, uint32_t key_mask, uint32_t n, uint32_t n_cells, uint32_t* cell_start,
                       uint32_t* d_big, cudaStream_t s);
void launch_tiles(const uint32_t* cell_start, const uint32_t* cell_base, const int32_t* n_ra, uint32_t n_zones, const uint32_t* sorted_keys,
                  uint32_t key_mask, uint32_t tile_cap, uint32_t* d_tile_first, TileDesc* tiles, uint32_t* d_n_tiles, cudaStream_t s);

// self-match / per-record radii: self_mode as in MatchArgs; k_factor > 0 switches Eq. (4) per pair on
struct MatchExtra { int self_mode; double k_factor; };
size_t match_temp_bytes(const IndexView& A, const IndexView& B);
constexpr uint32_t kMatchSameGrid = 1u;       // launch_match flag: A and B share one grid and both carry window flags
size_t match_temp_for_tiles(size_t tile_cap);
// upper bound of hlc2_crossmatch_sizes for any A index of <= n sources built with these options (hlc2_api.cu)
size_t match_temp_bound(int64_t n_a, const hlc2_opts* opts);
void launch_match(const IndexView& A, const IndexView& B, double radius_arcsec, int mode,
                  int64_t* out_ida, int64_t* out_idb, double* out_sep, unsigned long long capacity,
                  unsigned long long* d_count, void* d_temp, cudaStream_t s, uint32_t match_flags = 0,
                  cudaEvent_t ev_start = nullptr, cudaEvent_t ev_stop = nullptr, const MatchExtra* ex = nullptr);

void count_launch(int k = 1);

}  // namespace hlc2
