/*
 * Seeded synthetic workload generator (input recipe of DESIGN.md §4).
 *
 * This module serves BOTH the CPU oracle and the CUDA path with the same
 * arrays and holds NONE of the method's arithmetic: it only draws sparse rows
 * (term ids + weights) that stand in for SPLADE-encoded MS MARCO vectors
 * (§6.1: V=30522, ~127 nnz/doc, ~50 nnz/query, weights in
 * [0,3.5]).  The distributions are the ones BASELINE.json's `configs` fix:
 *
 *   nnz(row)  = clip(rint(mu + sigma*z), lo, hi), z ~ N(0,1)      (law 0)
 *             = lo + floor(u*(hi-lo+1)),           u ~ U[0,1)      (law 1)
 *   term ids  = ranks drawn from Zipf(s) over V by inverse CDF, repeats
 *               discarded, until nnz distinct; term id = rank-1
 *   weight    = (float) exp(0.5*z'),               z' ~ N(0,1)     LogNormal(0,0.5)
 *   u8 impact = clamp(nearbyint(100*w), 1, 255)    (round-half-even)
 *
 * Randomness is counter based: every draw is a pure function of
 * (seed, stream, row, substream, draw#), so a row can be generated on its own
 * and the first n rows of a larger collection equal the smaller collection.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef struct {
    uint64_t seed;
    uint64_t stream;     /* 0 = documents, 1 = queries */
    int32_t  vocab;      /* V */
    double   zipf_s;     /* Zipf exponent */
    int32_t  nnz_law;    /* 0 = clipped normal, 1 = uniform integer */
    double   nnz_mu, nnz_sigma;
    int32_t  nnz_lo, nnz_hi;
} wl_params_t;

static inline uint64_t sm64(uint64_t x) {
    x += 0x9E3779B97F4A7C15ULL;
    x = (x ^ (x >> 30)) * 0xBF58476D1CE4E5B9ULL;
    x = (x ^ (x >> 27)) * 0x94D049BB133111EBULL;
    return x ^ (x >> 31);
}
static inline uint64_t row_key(const wl_params_t* p, int64_t row) {
    return sm64(sm64(sm64(p->seed) ^ p->stream) ^ (uint64_t)row);
}
static inline uint64_t draw(uint64_t key, uint64_t sub, uint64_t i) {
    return sm64(key + sub * 0xD1B54A32D192ED03ULL + i * 0x9E3779B97F4A7C15ULL);
}
static inline double u01(uint64_t r)      { return (double)(r >> 11) * 0x1.0p-53; }            /* [0,1) */
static inline double u01_open(uint64_t r) { return ((double)(r >> 11) + 1.0) * 0x1.0p-53; }    /* (0,1] */
static inline double std_normal(uint64_t key, uint64_t sub, uint64_t i) {
    double u1 = u01_open(draw(key, sub, 2 * i));
    double u2 = u01(draw(key, sub, 2 * i + 1));
    return sqrt(-2.0 * log(u1)) * cos(6.283185307179586476925286766559 * u2);
}

static int32_t row_nnz(const wl_params_t* p, uint64_t key) {
    long n;
    if (p->nnz_law == 0) {
        double z = std_normal(key, 0, 0);
        n = (long)nearbyint(p->nnz_mu + p->nnz_sigma * z);
    } else {
        double u = u01(draw(key, 0, 0));
        n = p->nnz_lo + (long)floor(u * (double)(p->nnz_hi - p->nnz_lo + 1));
    }
    if (n < p->nnz_lo) n = p->nnz_lo;
    if (n > p->nnz_hi) n = p->nnz_hi;
    if (n > p->vocab) n = p->vocab;
    return (int32_t)n;
}

/* Zipf CDF over ranks 1..V in double, plus a guide table that only speeds up
 * the upper_bound search (the result is identical to a plain binary search). */
#define GUIDE_BITS 16
typedef struct { double* cdf; int32_t* guide; int32_t V; } zipf_t;

static int zipf_init(zipf_t* z, int32_t V, double s) {
    z->V = V;
    z->cdf = (double*)malloc(sizeof(double) * (size_t)V);
    z->guide = (int32_t*)malloc(sizeof(int32_t) * ((1u << GUIDE_BITS) + 1));
    if (!z->cdf || !z->guide) return -1;
    double tot = 0.0;
    for (int32_t r = 1; r <= V; ++r) { tot += pow((double)r, -s); z->cdf[r - 1] = tot; }
    for (int32_t r = 0; r < V; ++r) z->cdf[r] /= tot;
    z->cdf[V - 1] = 1.0;
    int32_t i = 0;
    for (uint32_t j = 0; j <= (1u << GUIDE_BITS); ++j) {
        double x = (double)j / (double)(1u << GUIDE_BITS);
        while (i < V - 1 && z->cdf[i] <= x) ++i;   /* smallest i with cdf[i] > x */
        z->guide[j] = i;
    }
    return 0;
}
static void zipf_free(zipf_t* z) { free(z->cdf); free(z->guide); }
static inline int32_t zipf_rank0(const zipf_t* z, double u) {   /* smallest i with cdf[i] > u */
    int32_t i = z->guide[(uint32_t)(u * (double)(1u << GUIDE_BITS))];
    while (i < z->V - 1 && z->cdf[i] <= u) ++i;
    return i;
}

int wl_max_threads(void);

/* indptr[rows+1]: prefix sums of the per-row nnz of rows [row0, row0+rows). */
int wl_indptr(const wl_params_t* p, int64_t row0, int64_t rows, int64_t* indptr, int nthreads) {
    if (!p || rows < 0 || !indptr) return -1;
#ifdef _OPENMP
    if (nthreads > 0) omp_set_num_threads(nthreads);
#endif
    indptr[0] = 0;
#pragma omp parallel for schedule(static)
    for (int64_t r = 0; r < rows; ++r) indptr[r + 1] = row_nnz(p, row_key(p, row0 + r));
    for (int64_t r = 0; r < rows; ++r) indptr[r + 1] += indptr[r];
    return 0;
}

/* Fill term ids (draw order, NOT sorted) and fp32 weights for the same rows. */
int wl_fill(const wl_params_t* p, int64_t row0, int64_t rows, const int64_t* indptr,
            int32_t* terms, float* weights, int nthreads) {
    if (!p || rows < 0 || !indptr || !terms || !weights) return -1;
    zipf_t z;
    if (zipf_init(&z, p->vocab, p->zipf_s)) return -2;
#ifdef _OPENMP
    if (nthreads > 0) omp_set_num_threads(nthreads);
#endif
    int nthr = wl_max_threads();
    size_t words = ((size_t)p->vocab + 63) / 64;
    uint64_t* seen_all = (uint64_t*)calloc(words * (size_t)nthr, sizeof(uint64_t));
    if (!seen_all) { zipf_free(&z); return -2; }
#pragma omp parallel
    {
#ifdef _OPENMP
        uint64_t* seen = seen_all + words * (size_t)omp_get_thread_num();
#else
        uint64_t* seen = seen_all;
#endif
#pragma omp for schedule(dynamic, 1024)
        for (int64_t r = 0; r < rows; ++r) {
            uint64_t key = row_key(p, row0 + r);
            int64_t o = indptr[r];
            int32_t n = (int32_t)(indptr[r + 1] - o);
            int32_t got = 0;
            for (uint64_t i = 0; got < n; ++i) {
                int32_t t = zipf_rank0(&z, u01(draw(key, 1, i)));
                uint64_t bit = 1ULL << (t & 63);
                if (seen[t >> 6] & bit) continue;
                seen[t >> 6] |= bit;
                terms[o + got++] = t;
            }
            for (int32_t j = 0; j < n; ++j) seen[terms[o + j] >> 6] = 0;
            /* one Box-Muller pair (cos, sin branch) feeds weights 2i and 2i+1 */
            for (int32_t j = 0; j < n; j += 2) {
                double u1 = u01_open(draw(key, 2, (uint64_t)j));
                double u2 = u01(draw(key, 2, (uint64_t)j + 1));
                double rad = sqrt(-2.0 * log(u1)), ang = 6.283185307179586476925286766559 * u2;
                weights[o + j] = (float)exp(0.5 * rad * cos(ang));
                if (j + 1 < n) weights[o + j + 1] = (float)exp(0.5 * rad * sin(ang));
            }
        }
    }
    free(seen_all);
    zipf_free(&z);
    return 0;
}

/* BASELINE.json config 4: uint8 impact = clamp(round(100*w), 1, 255), round-half-even. */
void wl_quantize_u8(const float* w, int64_t n, uint8_t* out, int nthreads) {
#ifdef _OPENMP
    if (nthreads > 0) omp_set_num_threads(nthreads);
#endif
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < n; ++i) {
        double q = nearbyint(100.0 * (double)w[i]);
        if (q < 1.0) q = 1.0;
        if (q > 255.0) q = 255.0;
        out[i] = (uint8_t)q;
    }
}

/* FNV-1a style 64-bit checksum over 8-byte words (tail bytes folded), recorded in reports. */
uint64_t wl_checksum(const void* data, int64_t bytes) {
    const uint8_t* b = (const uint8_t*)data;
    uint64_t h = 0xCBF29CE484222325ULL;
    int64_t i = 0;
    for (; i + 8 <= bytes; i += 8) {
        uint64_t w;
        memcpy(&w, b + i, 8);
        h = (h ^ w) * 0x100000001B3ULL;
        h ^= h >> 29;
    }
    for (; i < bytes; ++i) h = (h ^ b[i]) * 0x100000001B3ULL;
    return h;
}

int wl_max_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
