/*
 * hlc2.h -- C ABI of the B200-native HLC2 cross-match hot path (libhlc2.so).
 *
 * The operation (PAPER.md = /root/reference/PAPER.md, "P:L<n>" = line n; NS = north_star
 * of BASELINE.json):
 *
 *   Given catalogues A and B of sky positions (RA, Dec in fp64 degrees; Table 2
 *   P:L288-297) and a radius r, report every pair whose great-circle separation d of
 *   Eq. (1) satisfies the match criterion d <= r of Eq. (4) (inclusive;
 *   the caller's r stands for 3*sqrt(r1^2+r2^2)), or only the nearest B per A (NS).
 *   The result equals the paper's "No Index" O(mn) nested loop: the
 *   spatial partition only prunes, it never loses a pair.
 *
 * How (NS (a)-(c)): every catalogue is turned ON DEVICE into a cell-sorted index -- a
 * two-level partition (equal-height declination zones, then per-zone RA cells, the role
 * of the paper's HEALPix blocks P:L104) built from per-source cell keys, an LSD
 * radix sort, and a scan into a cell offset table; positions are kept as SoA fp64 unit
 * vectors.  The match kernel gives each A source the B cells its radius can reach (the
 * cells the quad-direction strategy probes, plus the diagonal and polar /
 * RA-wrap cases it misses), compares chord^2 with 4 sin^2(r/2), and appends
 * (idA, idB, sep) to a compacted output (the role of d_out_dis).
 *
 * Conventions
 *   - Pointers named d_* are DEVICE pointers, h_* HOST pointers.  All are plain pointers;
 *     there are no torch or C++ types in this interface.
 *   - Ownership: the library never allocates device memory.  Every device buffer belongs to
 *     the caller, who must keep d_index_buf alive and unmodified while the handle is in use
 *     and d_temp alive until the work enqueued by the call has completed.  A handle owns
 *     only small host-side metadata; release it with hlc2_index_destroy.
 *   - Stream order: all device work is enqueued on `cuda_stream` (a cudaStream_t passed as
 *     void*; NULL = the legacy default stream).  hlc2_build_index synchronises that stream
 *     once (it reads back the catalogue extent to plan the grid) unless opts.async_like is set; hlc2_crossmatch does not
 *     synchronise; hlc2_index_status synchronises.
 *   - Every function returns an int status: HLC2_OK (0) or a negative hlc2_status code.
 *   - n = 0 is valid everywhere and yields an empty result.
 *   - ids are opaque int64 (duplicates allowed); d_id = NULL means "row number".
 *   - Output order is unspecified (a set); sort by (idA, idB) to compare.
 *   - There is no CPU fallback: without a CUDA device every compute call fails with
 *     HLC2_ERR_CUDA.
 */
#ifndef HLC2_H_
#define HLC2_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct hlc2_index hlc2_index;     /* opaque host handle */

typedef enum { HLC2_ALL_PAIRS = 0, HLC2_NEAREST = 1 } hlc2_mode;

typedef enum {
    HLC2_OK = 0,
    HLC2_ERR_INVALID_ARG = -1,       /* null pointer, n < 0, radius <= 0 or non-finite, bad option */
    HLC2_ERR_RADIUS_TOO_LARGE = -2,  /* radius > min(r_max of the two indices) */
    HLC2_ERR_BUFFER_TOO_SMALL = -3,  /* index_bytes / temp_bytes below what the *_sizes call reports */
    HLC2_ERR_BAD_COORD = -4,         /* a non-finite coordinate or |dec| > 90 was found (hlc2_index_status) */
    HLC2_ERR_CUDA = -5,              /* a CUDA runtime call failed; see hlc2_last_cuda_error */
    HLC2_ERR_GRID_MISMATCH = -6,     /* opts.grid_like: the catalogue does not fit inside that grid's box */
    HLC2_ERR_TOO_MANY = -7,          /* n >= 2^30 sources in one index (stream the catalogue instead) */
    HLC2_ERR_STATIC_LIMIT = -8       /* hlc2_crossmatch_static: the match needs more than HLC2_STATIC_SCRATCH_BYTES */
} hlc2_status;

/*
 * Options of an index build.
 *   r_max_arcsec      largest radius the index will be queried with; > 0, <= 36000 (10 deg).
 *                     Fine cells are never smaller than this ("cells sized to r", NS (a)), so a
 *                     search window spans at most 3 zones.
 *   target_occupancy  mean sources per fine cell over the occupied sky; 0 -> automatic: the finest value in
 *                     [0.4, 1] whose cell count needs no more radix-sort digits than occupancy 1 would.
 *   cell_arcsec       explicit fine-cell size; 0 -> derived from the catalogue's density
 *                     (max(r_max, sqrt(target_occupancy * occupied area / n))).  Honoured while the cell
 *                     table stays within max(16 n, 2^25) cells, else coarsened until it fits.
 *   full_sky          non-zero: the grid spans the whole sphere whatever the data extent.
 *   zone_aspect       zones are zone_aspect times as high as the fine-cell size and RA cells that much narrower (same
 *                     cell area, both never below r_max): a source's search window then leaves its zone zone_aspect times
 *                     less often and reaches a neighbouring RA cell that much more often -- the second is the cheap one
 *                     (one more cell of the same contiguous row range).  0 -> automatic: min(32, floor(cell / (3 r_max))), scaled
 *                     back when the catalogue is concentrated in RA (fullest of 4096 RA bins more than 4x the mean
 *                     occupied bin: a dense strip along a meridian would fill tall cells), at least 1; 1 = square cells.
 *   grid_like         if non-NULL, reuse that index's grid exactly (zones, cells, box).  The
 *                     catalogue must lie inside that grid's box (else HLC2_ERR_GRID_MISMATCH).
 */
typedef struct {
    double r_max_arcsec;
    double target_occupancy;
    double cell_arcsec;
    int32_t full_sky;
    int32_t zone_aspect;
    const hlc2_index* grid_like;
    const double* d_err_arcsec;      /* optional: [n] per-record error radii (device, input order, arcsec, >= 0) for
                                        hlc2_crossmatch_radii: the r1 / r2 of Eq. (4); NULL = none */
    int32_t async_like;              /* with grid_like: build WITHOUT the extent pass and without any host synchronisation
                                        (everything is enqueued on the stream; the call can be captured in a CUDA graph).
                                        Bad coordinates and a catalogue that does not fit the grid's RA box are then both
                                        reported by hlc2_index_status (HLC2_ERR_BAD_COORD / HLC2_ERR_GRID_MISMATCH), not by
                                        the build call; sources outside the box are filed in the box's last cell.
                                        The index's declination extent is taken as the whole sphere: matched against an
                                        index on ANOTHER grid, the tiles of its first and last zone then plan windows over
                                        every zone of that index beyond the grid (same results, more work); on the same
                                        grid nothing changes. */
    int32_t reserved;
} hlc2_opts;

/* Description of an index's grid (host data), for tools and for the boundary-stress generator. */
typedef struct {
    double dec_lo_deg;       /* south edge of zone 0 */
    double zone_height_deg;  /* zone z spans [dec_lo + z h, dec_lo + (z+1) h) */
    int64_t n_zones;
    double ra0_deg;          /* west edge of the RA box; cells of zone z are span/n_ra[z] wide from here */
    double ra_span_deg;      /* 360 = full ring */
    int64_t n_cells;         /* sum of n_ra */
    double cell_arcsec;      /* the planner's fine-cell size */
    int64_t n;               /* sources in the index */
} hlc2_grid_info;

/* Upper bounds, for `n` sources and these options, of the index buffer and of the build's
 * temporary buffer (both 256-byte aligned device memory).  opts may be NULL (defaults with
 * r_max = 1 arcsec).  The role of the paper's source-reading module, which queries free CPU / GPU
 * memory before cutting calculation blocks (Eq. (8)-(9) P:L259-263): here the caller owns the
 * memory and asks how much a catalogue of n records needs (NS: "PyTorch used only for device memory"). */
int hlc2_index_sizes(int64_t n, const hlc2_opts* opts, size_t* index_bytes, size_t* temp_bytes);

/*
 * Build the cell-sorted index of one catalogue (NS "hlc2_build_index(cat) -> cell-sorted
 * index"): validate, cell keys, radix sort of (key, row), gather into
 * SoA unit vectors + ids, cell offset table.
 *   d_ra_deg, d_dec_deg  [n] fp64 degrees, device.  RA: any finite value, taken modulo 360
 *                        (360.0 == 0.0).  Dec must be in [-90, 90].
 *   d_id                 [n] int64, device, or NULL (ids = row numbers).
 *   d_index_buf          caller's device buffer of >= index_bytes (from hlc2_index_sizes).
 *   d_temp               scratch of >= temp_bytes; free to reuse when the stream has drained.
 *   out                  receives the handle.
 * Bad coordinates do not fail the build (it is asynchronous): they are recorded and
 * reported by hlc2_index_status.  Such rows are kept in the index with a NaN unit vector, which no
 * chord test can pass: they never appear in a result, neither as idA nor as idB; all other rows are
 * matched as usual.
 * The inputs are not modified and are not referenced after the build's work completes.
 */
int hlc2_build_index(const double* d_ra_deg, const double* d_dec_deg, const int64_t* d_id, int64_t n,
                     const hlc2_opts* opts, void* d_index_buf, size_t index_bytes,
                     void* d_temp, size_t temp_bytes, void* cuda_stream, hlc2_index** out);

/* Synchronises the build stream.  Returns HLC2_OK, or HLC2_ERR_BAD_COORD with the smallest
 * offending row in *first_bad_row (may be NULL).  A catalogue is a table of (RA, Dec) positions in
 * degrees (Table 2); a non-finite value or |Dec| > 90 is not a position, and the
 * paper's extraction module would have dropped such a record before the kernel saw it. */
int hlc2_index_status(const hlc2_index* idx, int64_t* first_bad_row);

/* Grid description.  *h_n_ra (may be NULL) receives a host pointer to n_zones int32 values
 * owned by the handle. */
int hlc2_grid_describe(const hlc2_index* idx, hlc2_grid_info* info, const int32_t** h_n_ra);

/*
 * Device views into the index buffer, for tests of rows a2-a4 (keys sorted, permutation
 * valid, cell table monotone).  All returned pointers are device pointers inside
 * d_index_buf; any output argument may be NULL.
 *   x, y, z     [n] fp64 unit vectors in cell order      id  [n] int64 in cell order
 *   cell_start  [n_cells + 1] uint32, cell c holds sorted rows [cell_start[c], cell_start[c+1])
 *   cell_key    [n] uint32: the cell key of every sorted row in the low 28 bits (& HLC2_KEY_MASK); when the grid
 *               has <= 2^28 cells the top bits carry the row's window flags on its own grid -- bit 28 / 29: a window of
 *               radius <= r_max reaches the previous / next RA cell of its zone; bit 30 / 31: it reaches the zone
 *               below / above; both of 30 and 31: anything else (it passes RA = 0/360, is wider than a cell, or touches
 *               both neighbouring zones: the general path) -- which let two indices on ONE grid (opts.grid_like) be
 *               matched without per-row window arithmetic.  With more cells the word is the bare key.
 */
#define HLC2_KEY_MASK 0x0FFFFFFFu
int hlc2_index_arrays(const hlc2_index* idx, const double** d_x, const double** d_y, const double** d_z,
                      const int64_t** d_id, const uint32_t** d_cell_start, const uint32_t** d_cell_key,
                      int64_t* n, int64_t* n_cells);

/* Scratch needed by hlc2_crossmatch / hlc2_selfmatch / hlc2_crossmatch_radii for this pair of indices (may be 0): for two
 * indices on different grids the job records into which the planner cuts every A tile's window -- the role of the
 * paper's calculation blocks, whose memory the paper's tool sized itself (Eq. (8)-(9)) and the
 * caller sizes here; for two indices on one grid the list of the rows that need the general path (4 bytes per A row). */
int hlc2_crossmatch_sizes(const hlc2_index* A, const hlc2_index* B, size_t* temp_bytes);

/*
 * Cross-match (NS "hlc2_crossmatch(idxA, idxB, radius_arcsec, mode) -> (idA, idB, sep)";
 * SURVEY rows a5-a7).  For every source of A: all sources of B (HLC2_ALL_PAIRS) or the nearest
 * one (HLC2_NEAREST; ties -> smaller idB) with separation <= radius_arcsec.
 *   d_out_idA, d_out_idB [capacity] int64; d_out_sep_arcsec [capacity] fp64 (arcsec).
 *   d_count              device uint64 scalar.  The call zeroes it, the kernels add every
 *                        result found; rows beyond `capacity` are counted but not written, so
 *                        *d_count > capacity means "retry with a larger buffer" (not an error).
 * Decisions are taken in fp64 on unit vectors: chord^2 <= 4 sin^2(r/2); sep = 2 asin(chord/2).
 * Enqueued on cuda_stream; does not synchronise.  Both indices must live on the current device.
 */
int hlc2_crossmatch(const hlc2_index* A, const hlc2_index* B, double radius_arcsec, int mode,
                    int64_t* d_out_idA, int64_t* d_out_idB, double* d_out_sep_arcsec,
                    int64_t capacity, unsigned long long* d_count,
                    void* d_temp, size_t temp_bytes, void* cuda_stream);

/* hlc2_crossmatch with two caller-owned CUDA events (cudaEvent_t passed as void*, either may be NULL) that the
 * call records on cuda_stream immediately before and after the match kernel itself, leaving the planner and the
 * count memset outside: the measurement NS asks for ("the matching phase" against the HBM roofline).  No state is
 * kept in the library; the caller reads the events. */
int hlc2_crossmatch_events(const hlc2_index* A, const hlc2_index* B, double radius_arcsec, int mode,
                           int64_t* d_out_idA, int64_t* d_out_idB, double* d_out_sep_arcsec,
                           int64_t capacity, unsigned long long* d_count,
                           void* d_temp, size_t temp_bytes, void* cuda_stream,
                           void* ev_kernel_start, void* ev_kernel_stop);

/*
 * hlc2_crossmatch for callers that can neither allocate device memory nor carry a scratch buffer (code under CUDA graph
 * capture, tight serving loops, harnesses that forbid cudaMalloc): same operation, same results, same arguments minus
 * d_temp / temp_bytes.  The scratch (the planner's job lists, the general-row list: SURVEY 8(a5)-(a7)) lives in a static
 * device array of HLC2_STATIC_SCRATCH_BYTES inside the library, which every GPU that loads the library holds until the
 * process exits.  The call makes no cudaMalloc / cudaFree and calls no allocating library routine.
 *   Limit: hlc2_crossmatch_sizes(A, B) <= HLC2_STATIC_SCRATCH_BYTES, i.e. A of up to about 2 million rows (4 bytes per
 *   A row + 256, or the planner's lists if larger); beyond it the call returns HLC2_ERR_STATIC_LIMIT and does nothing.
 *   Sharing: all calls on one device use the same array.  Calls that may OVERLAP on the GPU (different streams without an
 *   ordering between them) race on it and give undefined results: order them, or use hlc2_crossmatch with buffers of
 *   their own.  The array keeps the previous call's contents; each call clears the counters it keeps there itself.
 *   The first call on a device resolves the array's device address (cudaGetSymbolAddress, the device of the indices
 *   current): make one call before starting a stream capture.  Other errors and stream behaviour as hlc2_crossmatch.
 */
#define HLC2_STATIC_SCRATCH_BYTES (8u << 20)
int hlc2_crossmatch_static(const hlc2_index* A, const hlc2_index* B, double radius_arcsec, int mode,
                           int64_t* d_out_idA, int64_t* d_out_idB, double* d_out_sep_arcsec,
                           int64_t capacity, unsigned long long* d_count, void* cuda_stream);

/*
 * Self-match of ONE catalogue (the paper's D4 case: 2MASS against itself, Table 2).
 *   HLC2_ALL_PAIRS  every unordered pair {i, j}, i != j, within radius_arcsec exactly once (either orientation of
 *                   (idA, idB); half the tests and half the staging of hlc2_crossmatch(idx, idx)); with
 *                   include_self != 0 also the n pairs (i, i) at separation 0.
 *   HLC2_NEAREST    for every source the nearest OTHER source within the radius (a source is not its own neighbour;
 *                   include_self is ignored).
 * Other arguments, stream behaviour and scratch size (hlc2_crossmatch_sizes(idx, idx)) as for hlc2_crossmatch.
 */
int hlc2_selfmatch(const hlc2_index* idx, double radius_arcsec, int mode, int include_self,
                   int64_t* d_out_idA, int64_t* d_out_idB, double* d_out_sep_arcsec,
                   int64_t capacity, unsigned long long* d_count,
                   void* d_temp, size_t temp_bytes, void* cuda_stream);

/*
 * Cross-match with the paper's criterion as printed (Eq. (4)): a pair matches when its separation is
 * <= k_factor * sqrt(r1^2 + r2^2), r1 / r2 the error radii of the two records (both indices must have been built
 * with opts.d_err_arcsec; k_factor = 3 in the paper), and <= radius_cap_arcsec (the search bound: at most the r_max
 * of both indices; pass at least k_factor * sqrt(max r1^2 + max r2^2) for the pure Eq. (4)).  Decisions in fp64:
 * chord^2 <= 4 sin^2(t/2) with t the pair's threshold.  Runs on the general per-lane path.
 */
int hlc2_crossmatch_radii(const hlc2_index* A, const hlc2_index* B, double radius_cap_arcsec, double k_factor, int mode,
                          int64_t* d_out_idA, int64_t* d_out_idB, double* d_out_sep_arcsec,
                          int64_t capacity, unsigned long long* d_count,
                          void* d_temp, size_t temp_bytes, void* cuda_stream);

/*
 * Partition streaming from pinned host memory (NS (c); the paper's pinned
 * memory + multi-stream overlap P:L278).  The caller has split both catalogues into
 * the same declination bands: band k of A and band k of B hold the sources with
 * dec in [band_edges_deg[k], band_edges_deg[k+1]) (last band closed above).  Band k of A is
 * matched against bands k-1, k, k+1 of B, which must therefore be at least `radius_arcsec`
 * high.  H2D copies of the next band run on a copy stream while the current band is indexed
 * and matched on the compute stream; results are copied back to the pinned outputs.
 *   h_*            pinned host arrays (cudaHostAlloc / cudaHostRegister); band k occupies
 *                  rows [h_a_off[k], h_a_off[k+1]) resp. [h_b_off[k], h_b_off[k+1]).
 *                  h_a_id / h_b_id may be NULL (ids = global row numbers).
 *   d_arena        caller's device scratch of arena_bytes (see hlc2_stream_sizes).
 *   h_out_*        pinned outputs of `capacity` rows; *h_count receives the total found.
 *   max_band_out   rows of one band's result the device output slots hold (as given to hlc2_stream_sizes).
 * The B window of band k is band k plus the rows of bands k-1 / k+1 within radius of band k's edges
 * (selected on the device), so every A source sees one window and nearest mode needs no merge.
 * ids NULL: ids are the global row numbers of the banded arrays.
 * Synchronous: returns when the outputs are complete.  HLC2_ERR_BUFFER_TOO_SMALL if a band found more than
 * max_band_out rows or the total exceeded capacity (*h_count still holds the full count: retry larger);
 * HLC2_ERR_BAD_COORD if a band held an invalid coordinate (the other rows are matched as usual);
 * HLC2_ERR_INVALID_ARG for a band lower than the radius (n_bands > 1), unordered edges or offsets.
 */
int hlc2_stream_sizes(int64_t max_band_a, int64_t max_band_b, const hlc2_opts* opts, int64_t max_band_out,
                      size_t* arena_bytes);
int hlc2_stream_crossmatch(const double* h_a_ra, const double* h_a_dec, const int64_t* h_a_id, const int64_t* h_a_off,
                           const double* h_b_ra, const double* h_b_dec, const int64_t* h_b_id, const int64_t* h_b_off,
                           const double* band_edges_deg, int64_t n_bands,
                           double radius_arcsec, int mode, const hlc2_opts* opts,
                           int64_t* h_out_idA, int64_t* h_out_idB, double* h_out_sep_arcsec, int64_t capacity,
                           unsigned long long* h_count, void* d_arena, size_t arena_bytes, int64_t max_band_out);

/* Releases the handle's host metadata (the device buffers are the caller's; NS: "PyTorch used only for
 * device memory and streams").  NULL is ignored. */
void hlc2_index_destroy(hlc2_index* idx);
/* Text of a status code of this interface (the paper's tool is a CLI that reports on the console, P:L100;
 * a library reports through codes). */
const char* hlc2_strerror(int status);
/* The last cudaError_t (as int) seen by this thread, and its string. */
int hlc2_last_cuda_error(const char** message);
/* Number of kernels this library has launched since it was loaded (for launch accounting). */
unsigned long long hlc2_kernel_launches(void);
const char* hlc2_version(void);

#ifdef __cplusplus
}
#endif
#endif /* HLC2_H_ */
