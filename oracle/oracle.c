/*
 * oracle.c — TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, obviously-correct CPU definition of what the GPUSparse hot path
 * computes.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may build, load or call this file.  It shares no code
 * with the CUDA path (paper_2606_26441_b200/csrc) and includes none of its headers.
 *
 * What it computes (the paper's method is EXACT, §4.3, so the
 * oracle is the plain definition, not the scatter-add algorithm):
 *
 *   score(q,d) = sum_i w_i * s_d(t_i)          PAPER.md L106-111 §4.1 Eq. (4)
 *              = s(q)^T s(d)                   PAPER.md L43 §2.1
 *   with s_d(t) = 0 when d is not in the posting list of t (L111),
 *   followed by top-k over ALL N documents     PAPER.md L61, L125 (the paper runs
 *   torch.topk over the whole zero-initialised [B,N] buffer: zero-score docs compete).
 *   Result order: score descending, ties by lower doc id (BASELINE.json north_star;
 *   the paper leaves tie order open, L129/L396 — DESIGN.md reading R1).
 *
 * How: every (query, document) pair is scored by a two-pointer merge of the two
 * term-sorted sparse rows; then all N (score, id) pairs of a query are fully sorted.
 *   fp32 mode (wtype 0): each product is formed in double (fp32*fp32 is exact in
 *     fp64) and summed in double in ascending term order.
 *   integer-impact mode (wtype 1): uint8*uint8 products summed in int64, checked
 *     to fit int32 (BASELINE.json config 4: int32 accumulation).
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): dense brute force on tiny inputs,
 * scipy.sparse Q @ D.T, the hand-worked 3-document example in
 * tests/golden/handworked_3doc.json, one-hot queries, closed-form tie rankings,
 * and invariants (term-order symmetry, batch independence, prefix property,
 * power-of-two scaling, zero for disjoint rows, query/doc role swap).
 */
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

enum { OR_OK = 0, OR_ERR_ARG = 1, OR_ERR_RANGE = 2, OR_ERR_DUPLICATE = 3, OR_ERR_OOM = 5, OR_ERR_OVERFLOW = 8 };
enum { OR_W_F32 = 0, OR_W_U8 = 1 };

typedef struct { int32_t term; float wf; uint8_t wu; } or_entry_t;

/* Canonical (term-sorted) copy of a CSR batch — step 1 of the definition. */
typedef struct {
    int64_t rows, nnz;
    int32_t vocab, wtype;
    int64_t* indptr;
    or_entry_t* ent;
} or_rows_t;

static int cmp_entry(const void* a, const void* b) {
    int32_t x = ((const or_entry_t*)a)->term, y = ((const or_entry_t*)b)->term;
    return (x > y) - (x < y);
}

void or_rows_free(or_rows_t* r) {
    if (!r) return;
    free(r->indptr);
    free(r->ent);
    free(r);
}

/* Copy + sort each row by term id; reject out-of-range ids and duplicate terms within a row. */
int or_rows_create(int64_t rows, const int64_t* indptr, const int32_t* terms, const void* weights,
                   int32_t wtype, int32_t vocab, int nthreads, or_rows_t** out) {
    if (rows < 0 || !indptr || !out || vocab <= 0 || (wtype != OR_W_F32 && wtype != OR_W_U8)) return OR_ERR_ARG;
    if (indptr[0] != 0) return OR_ERR_ARG;
    for (int64_t r = 0; r < rows; ++r) if (indptr[r + 1] < indptr[r]) return OR_ERR_ARG;
    int64_t nnz = indptr[rows];
    if (nnz > 0 && (!terms || !weights)) return OR_ERR_ARG;
    or_rows_t* R = (or_rows_t*)calloc(1, sizeof(or_rows_t));
    if (!R) return OR_ERR_OOM;
    R->rows = rows; R->nnz = nnz; R->vocab = vocab; R->wtype = wtype;
    R->indptr = (int64_t*)malloc(sizeof(int64_t) * (size_t)(rows + 1));
    R->ent = (or_entry_t*)malloc(sizeof(or_entry_t) * (size_t)(nnz > 0 ? nnz : 1));
    if (!R->indptr || !R->ent) { or_rows_free(R); return OR_ERR_OOM; }
    memcpy(R->indptr, indptr, sizeof(int64_t) * (size_t)(rows + 1));
    int err = OR_OK;
#ifdef _OPENMP
    if (nthreads > 0) omp_set_num_threads(nthreads);
#endif
#pragma omp parallel for schedule(dynamic, 256)
    for (int64_t r = 0; r < rows; ++r) {
        int64_t a = indptr[r], b = indptr[r + 1];
        int bad = OR_OK;
        for (int64_t i = a; i < b; ++i) {
            R->ent[i].term = terms[i];
            R->ent[i].wf = wtype == OR_W_F32 ? ((const float*)weights)[i] : 0.0f;
            R->ent[i].wu = wtype == OR_W_U8 ? ((const uint8_t*)weights)[i] : 0;
            if (terms[i] < 0 || terms[i] >= vocab) bad = OR_ERR_RANGE;
        }
        qsort(R->ent + a, (size_t)(b - a), sizeof(or_entry_t), cmp_entry);
        for (int64_t i = a + 1; i < b; ++i)
            if (R->ent[i].term == R->ent[i - 1].term && bad == OR_OK) bad = OR_ERR_DUPLICATE;
        if (bad != OR_OK) {
#pragma omp atomic write
            err = bad;
        }
    }
    if (err != OR_OK) { or_rows_free(R); return err; }
    *out = R;
    return OR_OK;
}

/* Eq. (4) for one pair, fp32 mode: sorted two-pointer merge, products and sum in double. */
static double merge_f32(const or_entry_t* q, int64_t nq, const or_entry_t* d, int64_t nd) {
    double s = 0.0;
    int64_t i = 0, j = 0;
    while (i < nq && j < nd) {
        if (q[i].term < d[j].term) ++i;
        else if (q[i].term > d[j].term) ++j;
        else { s += (double)q[i].wf * (double)d[j].wf; ++i; ++j; }
    }
    return s;   /* no shared term -> exactly 0 */
}
/* Eq. (4) for one pair, integer-impact mode: u8*u8 products summed in int64. */
static int64_t merge_u8(const or_entry_t* q, int64_t nq, const or_entry_t* d, int64_t nd) {
    int64_t s = 0;
    int64_t i = 0, j = 0;
    while (i < nq && j < nd) {
        if (q[i].term < d[j].term) ++i;
        else if (q[i].term > d[j].term) ++j;
        else { s += (int64_t)q[i].wu * (int64_t)d[j].wu; ++i; ++j; }
    }
    return s;
}

double or_score_f32(const or_rows_t* Q, int64_t b, const or_rows_t* D, int64_t d) {
    return merge_f32(Q->ent + Q->indptr[b], Q->indptr[b + 1] - Q->indptr[b],
                     D->ent + D->indptr[d], D->indptr[d + 1] - D->indptr[d]);
}
int64_t or_score_u8(const or_rows_t* Q, int64_t b, const or_rows_t* D, int64_t d) {
    return merge_u8(Q->ent + Q->indptr[b], Q->indptr[b + 1] - Q->indptr[b],
                    D->ent + D->indptr[d], D->indptr[d + 1] - D->indptr[d]);
}

/* Scores of sampled (query, doc) pairs: out_f64[n] (fp32 mode) or out_i64[n] (integer mode). */
int or_score_pairs(const or_rows_t* Q, const or_rows_t* D, int64_t n, const int64_t* qb, const int64_t* dd,
                   double* out_f64, int64_t* out_i64) {
    if (!Q || !D || Q->wtype != D->wtype || n < 0) return OR_ERR_ARG;
    for (int64_t i = 0; i < n; ++i) {
        if (qb[i] < 0 || qb[i] >= Q->rows || dd[i] < 0 || dd[i] >= D->rows) return OR_ERR_RANGE;
        if (Q->wtype == OR_W_F32) out_f64[i] = or_score_f32(Q, qb[i], D, dd[i]);
        else out_i64[i] = or_score_u8(Q, qb[i], D, dd[i]);
    }
    return OR_OK;
}

typedef struct { double s; int32_t id; } pair_f_t;
typedef struct { int64_t s; int32_t id; } pair_i_t;
/* score descending, then doc id ascending: a strict total order */
static int cmp_pair_f(const void* a, const void* b) {
    const pair_f_t *x = (const pair_f_t*)a, *y = (const pair_f_t*)b;
    if (x->s > y->s) return -1;
    if (x->s < y->s) return 1;
    return (x->id > y->id) - (x->id < y->id);
}
static int cmp_pair_i(const void* a, const void* b) {
    const pair_i_t *x = (const pair_i_t*)a, *y = (const pair_i_t*)b;
    if (x->s > y->s) return -1;
    if (x->s < y->s) return 1;
    return (x->id > y->id) - (x->id < y->id);
}

/*
 * Full search for queries [b0, b1): score every document, full sort, keep the first k.
 *   out_ids    int32 [(b1-b0)*k]
 *   out_f64    double[(b1-b0)*k]   (fp32 mode)   | out_i32 int32[(b1-b0)*k] (integer mode)
 *   all_f64    optional double[(b1-b0)*N] / all_i32 optional int32[(b1-b0)*N]: every score
 * Slots beyond N (k > N) hold id -1 and score -inf / INT32_MIN (reading R4).
 */
int or_search(const or_rows_t* Q, const or_rows_t* D, int64_t b0, int64_t b1, int32_t k,
              int32_t* out_ids, double* out_f64, int32_t* out_i32, double* all_f64, int32_t* all_i32,
              int nthreads) {
    if (!Q || !D || Q->wtype != D->wtype || Q->vocab != D->vocab) return OR_ERR_ARG;
    if (k < 1) return OR_ERR_RANGE;
    if (b0 < 0 || b1 > Q->rows || b0 > b1 || !out_ids) return OR_ERR_ARG;
    const int64_t N = D->rows;
    if (N >= 2147483647LL) return OR_ERR_RANGE;
    const int f32 = Q->wtype == OR_W_F32;
    if ((f32 && !out_f64) || (!f32 && !out_i32)) return OR_ERR_ARG;
    int err = OR_OK;
#ifdef _OPENMP
    if (nthreads > 0) omp_set_num_threads(nthreads);
#endif
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t b = b0; b < b1; ++b) {
        const or_entry_t* q = Q->ent + Q->indptr[b];
        const int64_t nq = Q->indptr[b + 1] - Q->indptr[b];
        const int64_t o = (b - b0) * (int64_t)k, oa = (b - b0) * N;
        void* buf = malloc((f32 ? sizeof(pair_f_t) : sizeof(pair_i_t)) * (size_t)(N > 0 ? N : 1));
        if (!buf) {
#pragma omp atomic write
            err = OR_ERR_OOM;
            continue;
        }
        if (f32) {
            pair_f_t* p = (pair_f_t*)buf;
            for (int64_t d = 0; d < N; ++d) {
                p[d].s = merge_f32(q, nq, D->ent + D->indptr[d], D->indptr[d + 1] - D->indptr[d]);
                p[d].id = (int32_t)d;
                if (all_f64) all_f64[oa + d] = p[d].s;
            }
            qsort(p, (size_t)N, sizeof(pair_f_t), cmp_pair_f);
            for (int64_t i = 0; i < k; ++i) {
                out_ids[o + i] = i < N ? p[i].id : -1;
                out_f64[o + i] = i < N ? p[i].s : -__builtin_inf();
            }
        } else {
            pair_i_t* p = (pair_i_t*)buf;
            for (int64_t d = 0; d < N; ++d) {
                p[d].s = merge_u8(q, nq, D->ent + D->indptr[d], D->indptr[d + 1] - D->indptr[d]);
                p[d].id = (int32_t)d;
                if (p[d].s > 2147483647LL) {
#pragma omp atomic write
                    err = OR_ERR_OVERFLOW;
                }
                if (all_i32) all_i32[oa + d] = (int32_t)p[d].s;
            }
            qsort(p, (size_t)N, sizeof(pair_i_t), cmp_pair_i);
            for (int64_t i = 0; i < k; ++i) {
                out_ids[o + i] = i < N ? p[i].id : -1;
                out_i32[o + i] = i < N ? (int32_t)p[i].s : (-2147483647 - 1);
            }
        }
        free(buf);
    }
    return err;
}

int or_max_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
