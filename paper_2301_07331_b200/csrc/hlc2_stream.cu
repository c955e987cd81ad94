// hlc2_stream.cu -- partition streaming from pinned host memory (NS (c)).
#include "hlc2_internal.cuh"

extern "C" {

int hlc2_stream_sizes(int64_t max_band_a, int64_t max_band_b, const hlc2_opts* opts, int64_t max_band_out,
                      size_t* arena_bytes) {
    (void)max_band_a; (void)max_band_b; (void)opts; (void)max_band_out; (void)arena_bytes;
    return HLC2_ERR_INVALID_ARG;
}

int hlc2_stream_crossmatch(const double* h_a_ra, const double* h_a_dec, const int64_t* h_a_id, const int64_t* h_a_off,
                           const double* h_b_ra, const double* h_b_dec, const int64_t* h_b_id, const int64_t* h_b_off,
                           const double* band_edges_deg, int64_t n_bands,
                           double radius_arcsec, int mode, const hlc2_opts* opts,
                           int64_t* h_out_idA, int64_t* h_out_idB, double* h_out_sep_arcsec, int64_t capacity,
                           unsigned long long* h_count, void* d_arena, size_t arena_bytes, int64_t max_band_out) {
    (void)h_a_ra; (void)h_a_dec; (void)h_a_id; (void)h_a_off; (void)h_b_ra; (void)h_b_dec; (void)h_b_id; (void)h_b_off;
    (void)band_edges_deg; (void)n_bands; (void)radius_arcsec; (void)mode; (void)opts; (void)h_out_idA; (void)h_out_idB;
    (void)h_out_sep_arcsec; (void)capacity; (void)h_count; (void)d_arena; (void)arena_bytes; (void)max_band_out;
    return HLC2_ERR_INVALID_ARG;
}

}  // extern "C"
