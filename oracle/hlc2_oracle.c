/*
 * hlc2_oracle.c -- CPU ORACLE for the HLC2 cross-match hot path.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference leg may build, load or call it.  It
 * shares no code, header, table or helper with the CUDA path under
 * paper_2301_07331_b200/ and neither side includes or imports the other.
 *
 * What it computes (the plain definition the method reaches, faster):
 *   all_pairs(A, B, r) = { (idA_i, idB_j, theta_ij) : theta_ij <= r }
 *   nearest(A, B, r)   = for every i with a non-empty row, the j minimising theta_ij
 *                        (ties: smaller idB)
 * where theta is the great-circle separation of PAPER.md Eq. (1) (L55) and the match
 * criterion is the inclusive "<=" of Eq. (4) (L68), the user's radius standing for the
 * right-hand side 3*sqrt(r1^2+r2^2).  This is the paper's own accuracy reference, the
 * "No Index" O(mn) nested loop (L70, L344).
 *
 * Readings (DESIGN.md section "Readings of the paper"):
 *   - Eq. (1), not the small-angle Eq. (3): Eq. (3) departs from Eq. (1) by > 1e-9 arcsec
 *     beyond |dec| ~ 80 deg and cannot arbitrate at the 1e-9 arcsec bar of north_star.
 *   - theta is evaluated by the haversine form of Eq. (1) (north_star names it; it is
 *     algebraically the same quantity and is well conditioned at small separations,
 *     which arccos is not), in `long double`, from the fp64 *degree* inputs taken as
 *     exact reals: the coordinate differences are formed in degrees after promotion
 *     (exact), then scaled by pi/180.
 *   - RA is any finite value, reduced modulo 360; |dec| <= 90 required.
 *   - (i,i) pairs are ordinary pairs; ids are opaque int64; output sorted by (idA,idB).
 *
 * Extensions (hlc2_oracle_match_ext):
 *   - per-record error radii: Eq. (4) (L68) as printed, theta <= k * sqrt(e1_i^2 + e2_j^2) with the paper's k = 3 a
 *     parameter, evaluated in long double per pair; radius_arcsec is then a cap on the threshold (the search bound).
 *   - self-match of one catalogue (the paper's D4 case, L286, L295): every unordered pair {i, j}, i < j by row, once;
 *     optionally the n pairs (i, i) as well; nearest mode excludes a source from its own neighbours.
 *
 * Engines:
 *   0  brute force, every (i,j) evaluated in long double          (tiny inputs)
 *   1  brute force with an fp64 chord pre-filter of generous margin, long-double confirm
 *   2  3-D voxel hash on the unit vector (27-neighbourhood), same pre-filter + confirm.
 *      A voxel grid has no pole and no RA seam, unlike the zone/cell grid of the GPU
 *      path, so the two cannot share a boundary failure mode.
 *
 * Pins: tests/test_oracle_pins.py (closed forms, 50-digit Eq. (1), engine agreement,
 * symmetry, self-match, planted truth, rotation invariance, threshold +-2e-9 arcsec).
 * Parity-unpinned: the "<=" vs "<" choice at *exactly* theta == r (north_star exempts
 * |theta - r| < 1e-9 arcsec, so no test can distinguish them).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define PI_L 3.141592653589793238462643383279502884L
#define ORACLE_OK 0
#define ORACLE_BAD_COORD -1
#define ORACLE_BAD_ARG -2
#define ORACLE_NOMEM -3

typedef struct { int64_t ida, idb; double sep; long double sep_l; } pair_t;
typedef struct { pair_t* v; size_t n, cap; } vec_t;

static int vec_push(vec_t* a, pair_t p) {
    if (a->n == a->cap) {
        size_t nc = a->cap ? a->cap * 2 : 1024;
        pair_t* nv = (pair_t*)realloc(a->v, nc * sizeof(pair_t));
        if (!nv) return -1;
        a->v = nv; a->cap = nc;
    }
    a->v[a->n++] = p;
    return 0;
}

/* Great-circle separation in arcsec, Eq. (1) in haversine form, long double. */
static long double sep_arcsec_l(double ra1, double dec1, double ra2, double dec2) {
    long double dra = (long double)ra1 - (long double)ra2;      /* exact */
    dra -= 360.0L * rintl(dra / 360.0L);                        /* into [-180,180], exact */
    long double ddec = (long double)dec1 - (long double)dec2;   /* exact */
    const long double d2r = PI_L / 180.0L;
    long double s1 = sinl(0.5L * ddec * d2r);
    long double s2 = sinl(0.5L * dra * d2r);
    long double hav = s1 * s1 + cosl((long double)dec1 * d2r) * cosl((long double)dec2 * d2r) * s2 * s2;
    if (hav > 1.0L) hav = 1.0L;
    if (hav < 0.0L) hav = 0.0L;
    long double theta = 2.0L * asinl(sqrtl(hav));
    return theta * (648000.0L / PI_L);
}

/* exported: separation rounded to double, and as an unevaluated hi+lo sum */
double hlc2_oracle_sep_arcsec(double ra1, double dec1, double ra2, double dec2) {
    return (double)sep_arcsec_l(ra1, dec1, ra2, dec2);
}
void hlc2_oracle_sep_arcsec_hilo(double ra1, double dec1, double ra2, double dec2, double* hi, double* lo) {
    long double s = sep_arcsec_l(ra1, dec1, ra2, dec2);
    *hi = (double)s;
    *lo = (double)(s - (long double)*hi);
}

static int check_coords(const double* ra, const double* dec, int64_t n) {
    for (int64_t i = 0; i < n; ++i) {
        if (!isfinite(ra[i]) || !isfinite(dec[i]) || dec[i] < -90.0 || dec[i] > 90.0) return ORACLE_BAD_COORD;
    }
    return ORACLE_OK;
}

/* fp64 unit vector, used for pre-filtering and voxel binning only (never for a decision) */
static void unit_vec(double ra, double dec, double* v) {
    double a = ra * (M_PI / 180.0), d = dec * (M_PI / 180.0);
    v[0] = cos(d) * cos(a); v[1] = cos(d) * sin(a); v[2] = sin(d);
}

static int cmp_pair(const void* x, const void* y) {
    const pair_t* a = (const pair_t*)x; const pair_t* b = (const pair_t*)y;
    if (a->ida != b->ida) return a->ida < b->ida ? -1 : 1;
    if (a->idb != b->idb) return a->idb < b->idb ? -1 : 1;
    if (a->sep_l != b->sep_l) return a->sep_l < b->sep_l ? -1 : 1;
    return 0;
}

typedef struct { uint64_t key; int64_t row; } vox_t;
static int cmp_vox(const void* x, const void* y) {
    const vox_t* a = (const vox_t*)x; const vox_t* b = (const vox_t*)y;
    if (a->key != b->key) return a->key < b->key ? -1 : 1;
    if (a->row != b->row) return a->row < b->row ? -1 : 1;
    return 0;
}
static int64_t lower_bound(const vox_t* v, int64_t n, uint64_t key) {
    int64_t lo = 0, hi = n;
    while (lo < hi) { int64_t m = lo + ((hi - lo) >> 1); if (v[m].key < key) lo = m + 1; else hi = m; }
    return lo;
}

typedef struct {
    int mode;                 /* 0 all_pairs, 1 nearest */
    long double r_l;          /* radius, arcsec, promoted exactly */
    double pre2;              /* pre-filter threshold on chord^2 (generous) */
    int use_pre;
    const double* errA;       /* per-record error radii in arcsec (both or neither), Eq. (4) */
    const double* errB;
    long double k_l;          /* the factor of Eq. (4): 3 in the paper */
    int self_mode;            /* 0: two catalogues; 1: one catalogue, pairs i < j; 2: pairs i <= j; 3: j != i (nearest) */
} ctx_t;

/* consider candidate (i, j): confirm in long double; append or update the running best */
static inline int consider(const ctx_t* c, const double* raA, const double* decA, const int64_t* idA, int64_t i,
                           const double* raB, const double* decB, const int64_t* idB, int64_t j,
                           vec_t* out, pair_t* best, int* have_best) {
    if (c->self_mode == 1 && !(i < j)) return 0;            /* an unordered pair is reported once, (i, i) never */
    if (c->self_mode == 2 && !(i <= j)) return 0;
    if (c->self_mode == 3 && i == j) return 0;
    long double s = sep_arcsec_l(raA[i], decA[i], raB[j], decB[j]);
    long double thr = c->r_l;
    if (c->errA) {                                          /* Eq. (4) per pair: k sqrt(e1^2 + e2^2), capped by the radius */
        long double e1 = (long double)c->errA[i], e2 = (long double)c->errB[j];
        long double t = c->k_l * sqrtl(e1 * e1 + e2 * e2);
        if (t < thr) thr = t;
    }
    if (!(s <= thr)) return 0;                              /* Eq. (4): inclusive */
    pair_t p; p.ida = idA ? idA[i] : i; p.idb = idB ? idB[j] : j; p.sep_l = s; p.sep = (double)s;
    if (c->mode == 0) return vec_push(out, p);
    if (!*have_best || s < best->sep_l || (s == best->sep_l && p.idb < best->idb)) { *best = p; *have_best = 1; }
    return 0;
}

/*
 * hlc2_oracle_match: engine 0/1/2 as described in the header.
 * Inputs are host arrays; idA/idB may be NULL (row number).  On success *out_n rows are
 * returned in malloc'ed arrays (*out_ida, *out_idb, *out_sep) sorted by (idA, idB); free
 * them with hlc2_oracle_free.  threads <= 0 means "all OpenMP threads"; *threads_used
 * reports what ran.
 */
int hlc2_oracle_match_ext(const double* raA, const double* decA, const int64_t* idA, int64_t nA,
                          const double* raB, const double* decB, const int64_t* idB, int64_t nB,
                          double radius_arcsec, int mode, int engine, int threads,
                          const double* errA, const double* errB, double k_factor, int self_mode,
                          int64_t* out_n, int64_t** out_ida, int64_t** out_idb, double** out_sep,
                          int* threads_used);

int hlc2_oracle_match(const double* raA, const double* decA, const int64_t* idA, int64_t nA,
                      const double* raB, const double* decB, const int64_t* idB, int64_t nB,
                      double radius_arcsec, int mode, int engine, int threads,
                      int64_t* out_n, int64_t** out_ida, int64_t** out_idb, double** out_sep,
                      int* threads_used) {
    return hlc2_oracle_match_ext(raA, decA, idA, nA, raB, decB, idB, nB, radius_arcsec, mode, engine, threads,
                                 NULL, NULL, 3.0, 0, out_n, out_ida, out_idb, out_sep, threads_used);
}

/* The same with per-record error radii (errA, errB: both or neither; arcsec; >= 0) and / or self-match of one catalogue
 * (self_mode != 0: the caller passes the same arrays as A and B). */
int hlc2_oracle_match_ext(const double* raA, const double* decA, const int64_t* idA, int64_t nA,
                          const double* raB, const double* decB, const int64_t* idB, int64_t nB,
                          double radius_arcsec, int mode, int engine, int threads,
                          const double* errA, const double* errB, double k_factor, int self_mode,
                          int64_t* out_n, int64_t** out_ida, int64_t** out_idb, double** out_sep,
                          int* threads_used) {
    if ((errA == NULL) != (errB == NULL) || !(k_factor > 0.0) || self_mode < 0 || self_mode > 3 ||
        (self_mode != 0 && nA != nB)) return ORACLE_BAD_ARG;
    if (errA) {
        for (int64_t i = 0; i < nA; ++i) if (!(errA[i] >= 0.0) || !isfinite(errA[i])) return ORACLE_BAD_ARG;
        for (int64_t j = 0; j < nB; ++j) if (!(errB[j] >= 0.0) || !isfinite(errB[j])) return ORACLE_BAD_ARG;
    }
    if (nA < 0 || nB < 0 || !(radius_arcsec > 0.0) || !isfinite(radius_arcsec) || radius_arcsec >= 324000.0 ||
        (mode != 0 && mode != 1) || engine < 0 || engine > 2 || !out_n || !out_ida || !out_idb || !out_sep)
        return ORACLE_BAD_ARG;
    int rc = check_coords(raA, decA, nA); if (rc) return rc;
    rc = check_coords(raB, decB, nB); if (rc) return rc;

    ctx_t c; c.mode = mode; c.r_l = (long double)radius_arcsec; c.use_pre = engine != 0;
    c.errA = errA; c.errB = errB; c.k_l = (long double)k_factor; c.self_mode = self_mode;
    {   /* chord of (r + margin): margin = 0.1% of r + 1e-3 arcsec, far above fp64 chord error (~2e-10 arcsec) */
        double r_rad = (radius_arcsec * 1.001 + 1e-3) * (M_PI / 648000.0);
        double ch = 2.0 * sin(0.5 * r_rad);
        c.pre2 = ch * ch;
    }
    int nthr = 1;
#ifdef _OPENMP
    nthr = threads > 0 ? threads : omp_get_max_threads();
#endif
    if (threads_used) *threads_used = nthr;

    double* vB = NULL; vox_t* vox = NULL; double L = 0.0; int64_t ncell = 0;
    if (engine >= 1) {
        vB = (double*)malloc(sizeof(double) * 3 * (size_t)(nB > 0 ? nB : 1));
        if (!vB) return ORACLE_NOMEM;
        for (int64_t j = 0; j < nB; ++j) unit_vec(raB[j], decB[j], vB + 3 * j);
    }
    if (engine == 2) {
        /* voxel edge: > chord of the pre-filter radius, and about one B source per occupied voxel */
        double Lmin = 1.001 * sqrt(c.pre2);
        double Lden = sqrt(4.0 * M_PI / (double)(nB > 0 ? nB : 1));
        L = Lmin > Lden ? Lmin : Lden;
        if (L < 2.0 / 2000000.0) L = 2.0 / 2000000.0;           /* keep 3 x 21 bits */
        vox = (vox_t*)malloc(sizeof(vox_t) * (size_t)(nB > 0 ? nB : 1));
        if (!vox) { free(vB); return ORACLE_NOMEM; }
        for (;;) {
            ncell = (int64_t)floor(2.0 / L) + 2;
            for (int64_t j = 0; j < nB; ++j) {
                uint64_t ix = (uint64_t)floor((vB[3 * j] + 1.0) / L), iy = (uint64_t)floor((vB[3 * j + 1] + 1.0) / L),
                         iz = (uint64_t)floor((vB[3 * j + 2] + 1.0) / L);
                vox[j].key = (ix << 42) | (iy << 21) | iz; vox[j].row = j;
            }
            qsort(vox, (size_t)nB, sizeof(vox_t), cmp_vox);
            /* a catalogue covering only a patch of sky is denser than 4 pi / nB: halve the voxel edge
               until occupied voxels hold ~<= 3 sources on average (never below Lmin) */
            int64_t occupied = 0;
            for (int64_t j = 0; j < nB; ++j) if (j == 0 || vox[j].key != vox[j - 1].key) ++occupied;
            if (occupied == 0 || nB <= 3 * occupied || 0.5 * L < Lmin || 0.5 * L < 2.0 / 2000000.0) break;
            L *= 0.5;
        }
    }

    vec_t* outs = (vec_t*)calloc((size_t)nthr, sizeof(vec_t));
    int fail = 0;
#ifdef _OPENMP
#pragma omp parallel for schedule(dynamic, 256) num_threads(nthr)
#endif
    for (int64_t i = 0; i < nA; ++i) {
        int t = 0;
#ifdef _OPENMP
        t = omp_get_thread_num();
#endif
        vec_t* out = &outs[t];
        pair_t best; int have = 0; memset(&best, 0, sizeof best);
        double va[3]; unit_vec(raA[i], decA[i], va);
        if (engine <= 1) {
            for (int64_t j = 0; j < nB; ++j) {
                if (c.use_pre) {
                    double dx = va[0] - vB[3 * j], dy = va[1] - vB[3 * j + 1], dz = va[2] - vB[3 * j + 2];
                    if (dx * dx + dy * dy + dz * dz > c.pre2) continue;
                }
                if (consider(&c, raA, decA, idA, i, raB, decB, idB, j, out, &best, &have)) fail = 1;
            }
        } else {
            int64_t ix = (int64_t)floor((va[0] + 1.0) / L), iy = (int64_t)floor((va[1] + 1.0) / L),
                    iz = (int64_t)floor((va[2] + 1.0) / L);
            /* the 27 neighbouring voxels, visited as 9 (dx,dy) columns: with iz in the low key bits the
               three dz = -1,0,+1 voxels of a column are one contiguous key range of the sorted array */
            for (int64_t dx = -1; dx <= 1; ++dx) for (int64_t dy = -1; dy <= 1; ++dy) {
                int64_t jx = ix + dx, jy = iy + dy;
                if (jx < 0 || jy < 0 || jx >= ncell || jy >= ncell) continue;
                int64_t z0 = iz - 1 < 0 ? 0 : iz - 1, z1 = iz + 1 >= ncell ? ncell - 1 : iz + 1;
                uint64_t k0 = ((uint64_t)jx << 42) | ((uint64_t)jy << 21) | (uint64_t)z0;
                uint64_t k1 = ((uint64_t)jx << 42) | ((uint64_t)jy << 21) | (uint64_t)z1;
                for (int64_t p = lower_bound(vox, nB, k0); p < nB && vox[p].key <= k1; ++p) {
                    int64_t j = vox[p].row;
                    double ex = va[0] - vB[3 * j], ey = va[1] - vB[3 * j + 1], ez = va[2] - vB[3 * j + 2];
                    if (ex * ex + ey * ey + ez * ez > c.pre2) continue;
                    if (consider(&c, raA, decA, idA, i, raB, decB, idB, j, out, &best, &have)) fail = 1;
                }
            }
        }
        if (mode == 1 && have) if (vec_push(out, best)) fail = 1;
    }
    free(vB); free(vox);

    size_t total = 0;
    for (int t = 0; t < nthr; ++t) total += outs[t].n;
    pair_t* all = (pair_t*)malloc(sizeof(pair_t) * (total ? total : 1));
    if (!all) fail = 1;
    if (!fail) {
        size_t o = 0;
        for (int t = 0; t < nthr; ++t) { if (outs[t].n) memcpy(all + o, outs[t].v, outs[t].n * sizeof(pair_t)); o += outs[t].n; }
        qsort(all, total, sizeof(pair_t), cmp_pair);
    }
    for (int t = 0; t < nthr; ++t) free(outs[t].v);
    free(outs);
    if (fail) { free(all); return ORACLE_NOMEM; }

    *out_ida = (int64_t*)malloc(sizeof(int64_t) * (total ? total : 1));
    *out_idb = (int64_t*)malloc(sizeof(int64_t) * (total ? total : 1));
    *out_sep = (double*)malloc(sizeof(double) * (total ? total : 1));
    if (!*out_ida || !*out_idb || !*out_sep) { free(all); return ORACLE_NOMEM; }
    for (size_t k = 0; k < total; ++k) { (*out_ida)[k] = all[k].ida; (*out_idb)[k] = all[k].idb; (*out_sep)[k] = all[k].sep; }
    free(all);
    *out_n = (int64_t)total;
    return ORACLE_OK;
}

void hlc2_oracle_free(void* p) { free(p); }

int hlc2_oracle_max_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
