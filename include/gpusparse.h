/*
 * gpusparse.h — C ABI of the B200-native GPUSparse hot path (arxiv/paper_2606_26441).
 *
 * What the library computes (citations are PAPER.md line numbers):
 *   exact batched top-k scoring of sparse query vectors against a sparse document collection,
 *       score(q,d) = sum_i w_i * s_d(t_i)                            L106-111 §4.1 Eq. (4)
 *   over a GPU-resident inverted index whose posting lists are doc-id sorted and padded to
 *   32-entry warp blocks with (doc_id=-1, score=0) sentinels         L79-90  §3.2 Eq. (2)
 *   and over a CSR forward index used by the document-parallel kernel L174    §5.3,
 *   followed by top-k over ALL N documents                           L61, L125.
 *   Result rows are sorted by score descending, ties broken by LOWER doc id
 *   (BASELINE.json north_star; the paper leaves tie order open, L129/L396).
 *
 * Conventions
 *   - Plain C: opaque handle, plain pointers and sizes, no C++/torch types.
 *   - Every array pointer is a DEVICE pointer unless the name or comment says HOST.
 *   - The caller owns inputs, outputs and workspaces; the library owns only what hangs off a
 *     gs_index_t handle (allocated through the optional gs_alloc_t callbacks, default cudaMalloc).
 *   - Document id = CSR row number (0-based int32, N < 2^31).  Term ids are int32 in [0, V).
 *   - `gs_stream_t` is a cudaStream_t passed as void* (0 = default stream).
 *   - Errors are return codes, never exceptions or aborts.  Host-checkable arguments are checked
 *     before any launch.  There is NO CPU fallback: a device that is not sm_100 yields
 *     GS_ERR_UNSUPPORTED_DEVICE.
 *   - Two numeric modes: GS_W_F32 (fp32 weights, fp32 accumulate, fp32 scores) and GS_W_U8
 *     (uint8 impacts, int32 accumulate, int32 scores; bit-exact by construction).
 */
#ifndef GPUSPARSE_H
#define GPUSPARSE_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define GS_ABI_VERSION 5
#if defined(__GNUC__)
#define GS_API __attribute__((visibility("default")))
#else
#define GS_API
#endif
#define GS_MAX_K 4096          /* largest supported k (bitonic finish runs in shared memory)   */
#define GS_WARP_BLOCK 32       /* posting-list padding granularity W of Eq. (2)        */

typedef struct gs_index gs_index_t;   /* opaque, immutable after build (paper: no dynamic updates, L412) */
typedef void* gs_stream_t;

typedef enum gs_status {
    GS_OK = 0,
    GS_ERR_INVALID_ARG = 1,        /* null pointer, bad enum, indptr[0] != 0, host pointer where device expected */
    GS_ERR_OUT_OF_RANGE = 2,       /* term id outside [0,V), k < 1 or k > GS_MAX_K, non-monotone indptr          */
    GS_ERR_DUPLICATE_TERM = 3,     /* a term id occurs twice in one row                                          */
    GS_ERR_NONFINITE = 4,          /* NaN/Inf weight (fp32 mode)                                                 */
    GS_ERR_OOM = 5,                /* allocation failed / workspace too small                                     */
    GS_ERR_CUDA = 6,               /* a CUDA runtime call failed (see gs_last_cuda_error)                        */
    GS_ERR_UNSUPPORTED_DEVICE = 7, /* not an sm_100 device                                                       */
    GS_ERR_TYPE_MISMATCH = 8       /* query weight type differs from the index weight type                       */
} gs_status_t;

typedef enum gs_weight { GS_W_F32 = 0, GS_W_U8 = 1 } gs_weight_t;

typedef enum gs_algo {
    GS_ALGO_AUTO = 0,           /* the cheaper path under the cost model of gs_dispatch_model (L176-181 crossover)        */
    GS_ALGO_TERM_PARALLEL = 1,  /* tiled scatter-add over the inverted index   (Eq. 5, §5.2)   */
    GS_ALGO_DOC_PARALLEL = 2    /* CSR forward-index streaming, zero atomics   (L174)                    */
} gs_algo_t;

/* A batch of sparse rows in CSR form (documents for the build, queries for the search). */
typedef struct gs_csr {
    int64_t rows;             /* N (documents) or B (queries)                                          */
    int64_t nnz;              /* total number of entries == indptr[rows] (the caller knows it)         */
    const int64_t* indptr;    /* [rows+1], indptr[0] == 0, non-decreasing                              */
    const int32_t* term_ids;  /* [nnz] in [0,V), unique within a row, any order within a row           */
    const void* weights;      /* [nnz] float (GS_W_F32) or uint8_t (GS_W_U8); any finite value is legal */
    int32_t wtype;            /* gs_weight_t                                                           */
} gs_csr_t;

/* Optional allocator for everything a handle owns (e.g. torch's caching allocator). */
typedef struct gs_alloc {
    void* (*alloc)(size_t bytes, gs_stream_t stream, void* user);   /* returns NULL on failure */
    void (*free)(void* ptr, gs_stream_t stream, void* user);
    void* user;
} gs_alloc_t;

/* Build options; pass NULL for defaults (fields set to 0 also mean "default"). */
typedef struct gs_build_opts {
    int32_t tile_docs;        /* doc-id range covered by one accumulator tile (multiple of 32; default 512)   */
    int32_t head_max;         /* max number of posting lists additionally stored as dense strips (0..64;       */
                              /* default 64; -1 disables).  A list qualifies when |PL(t)| >= head_density * N  */
    float head_density;       /* default 0.25.  4 B/doc beats 8 B/posting from density 0.5 on; below that a    */
                              /* strip costs bytes but saves the per-posting lookup of the doc-parallel kernel */
    int32_t validate;         /* default 1: reject out-of-range ids, duplicates, non-finite weights            */
    int32_t pack_postings;    /* integer-impact mode (GS_W_U8), compressed postings (future work 2;  */
                              /* L75 is the "raw int32 + fp32" layout it replaces): 0 = default: ONE 32-bit word per */
                              /* posting — inverted lists (doc id : 24 | impact : 8) when N < 2^24, forward index    */
                              /* (term : 19 | impact : 8 | doc-in-block : 5) when V < 2^19 — 4 instead of 5 bytes    */
                              /* per posting and one load instead of two; -1 = keep the two-array layout.  fp32      */
                              /* postings stay (int32, fp32): the weights must keep full precision (exactness).     */
} gs_build_opts_t;

typedef struct gs_info {
    int64_t num_docs;          /* N                                                                   */
    int32_t vocab_size;        /* V                                                                   */
    int32_t wtype;
    int64_t nnz;               /* P = number of postings                                              */
    int64_t padded_nnz;        /* sum_t ceil(|PL(t)|/32)*32                        Eq. (2)            */
    int64_t nonempty_terms;
    int32_t tile_docs, num_tiles;
    int32_t head_terms;        /* number of dense-strip posting lists                                 */
    int64_t bytes_inverted;    /* doc_ids + weights of the padded lists            Eq. (3)            */
    int64_t bytes_inverted_meta; /* offsets + lengths + tile-segment table                            */
    int64_t bytes_forward;     /* forward index, CSR part: one row pointer per block of 32 documents + term
                                  words + weights of the postings whose term has no strip, each block padded
                                  to 128 postings (the strips are the dense part of the forward index)  */
    int64_t bytes_head;        /* dense strips                                                        */
    int64_t bytes_total;
    int64_t forward_tail_nnz;  /* postings held by the CSR part of the forward index                  */
    int32_t head_terms_term_parallel; /* strips the term-parallel kernels can read: head_terms + the second tier (up to
                                       * 128 more lists of density >= 0.05, 512-doc tiles only; bytes in bytes_head) */
    int32_t packed_layout;     /* bit 0: inverted lists are packed words, bit 1: forward index is (gs_build_opts_t.pack_postings) */
    int64_t forward_padded_nnz; /* slots of the CSR part: forward_tail_nnz + block padding             */
} gs_info_t;

/* Search options; pass NULL for defaults. */
#define GS_FLAG_VALIDATE_QUERIES 1u   /* check query ids/dups/finite on device, synchronise, return the error   */
#define GS_FLAG_FORCE_DENSE_TOPK 2u   /* materialise every score tile and select from it (no threshold filter) */
#define GS_FLAG_NO_HEAD_STRIPS 4u     /* term-parallel: send every list through the scatter path               */
#define GS_FLAG_TENSOR_CORE_HEAD 8u   /* integer-impact mode, batches of >= 32 queries, 512-doc tiles: contract the dense strips  */
                                      /* with tcgen05.mma kind::i8 (uint8 x uint8 -> int32 is exact: k_score_term_mma) instead of  */
                                      /* IDP4A on the CUDA cores.  Bit-identical results; measured slower on B200 (16.2 vs 13.9 ms */
                                      /* per 500-query batch at 8.8M docs: the tail scatter dominates), so opt-in.   */
typedef struct gs_search_opts {
    int32_t algo;             /* gs_algo_t                                                              */
    uint32_t flags;
    int32_t query_group;      /* term-parallel: (doc tile, query) cell rows = warps per CTA, 1..8 (0 = 2)  */
    int32_t doc_query_tile;   /* doc-parallel: queries per pass over the forward index (0 = auto)       */
    int32_t sample_shift;     /* threshold sample = 1/2^shift of the doc tiles (0 = auto)               */
} gs_search_opts_t;

/* Counters of the last search that used a workspace (read back with gs_search_stats). */
typedef struct gs_stats {
    int64_t candidates;        /* (query, doc) cells that passed the threshold filter                  */
    int32_t overflow_queries;  /* queries whose candidate list overflowed (exact only after gs_search_finish) */
    int32_t launches;          /* kernels launched by the call (host-side count)                       */
    int32_t algo_used;         /* gs_algo_t actually run                                               */
    int32_t sample_tiles;      /* doc tiles scored densely to obtain the thresholds                    */
    int32_t doc_query_tile;    /* doc-parallel: queries per pass over the forward index (0 otherwise)  */
    int32_t doc_passes;        /* doc-parallel: passes over the forward index per full-collection launch */
    int32_t query_group;       /* term-parallel: cell rows (warps) per CTA                             */
} gs_stats_t;

/* ------------------------------------------------------------------------------------------------
 * Index (§3).
 * gs_index_build: docs->indptr/term_ids/weights are DEVICE pointers; they may be released once the
 * call returns (the call synchronises `stream`).  Builds (i) the inverted index: per-term posting
 * lists sorted by doc id, padded to 32 with (-1, 0) sentinels, plus offsets/lengths; (ii) the CSR
 * forward index; (iii) the per-(term, doc-tile) segment table; (iv) dense strips for the densest
 * lists.  Errors: see gs_status_t; on error *out is NULL and nothing is leaked.
 * ---------------------------------------------------------------------------------------------- */
GS_API gs_status_t gs_index_build(const gs_csr_t* docs, int32_t vocab_size, const gs_build_opts_t* opts,
                           const gs_alloc_t* alloc, gs_stream_t stream, gs_index_t** out);
GS_API gs_status_t gs_index_info(const gs_index_t* index, gs_info_t* out);
GS_API void gs_index_free(gs_index_t* index);

/* Inspection (tests of Eq. 2/3): copy per-term metadata / one padded posting list to HOST buffers.
 * host_offsets [V+1] int64 (padded start of each list), host_lengths [V] int32 (true |PL(t)|). */
GS_API gs_status_t gs_index_copy_meta(const gs_index_t* index, int64_t* host_offsets, int32_t* host_lengths);
/* Copies min(capacity, padded_length(term)) entries; host_weights is float[] or uint8_t[] per wtype. */
GS_API gs_status_t gs_index_copy_list(const gs_index_t* index, int32_t term, int64_t capacity,
                               int32_t* host_doc_ids, void* host_weights, int64_t* out_padded_length);

/* The terms whose posting lists are also stored as dense strips, densest first: writes
 * min(capacity, head_terms) term ids to host_terms and the total to *out_count. */
GS_API gs_status_t gs_index_copy_head_terms(const gs_index_t* index, int32_t capacity, int32_t* host_terms,
                                     int32_t* out_count);

/* Cost model behind GS_ALGO_AUTO.  PAPER.md L176-181 (§5.3) states the trade-off: the term-parallel scatter touches
 * q̄·L̄ postings per query, the document-parallel kernel streams all N·k̄ postings per pass, and the crossover is where the
 * work ratio meets the ratio of the effective rates.  On B200 both sides were measured over N in {20K .. 1M} documents,
 * B in {1 .. 256} queries of 25 .. 4000 terms (profiles/r02_dispatch_sweep.md); the forms below predict
 * the faster path on 63 of the 64 grid points (the miss costs 6 %):
 *   term: 0.10 ms + max(1, B*tiles / 9472 warp slots) * (nnz/B) * 0.6 us * (1 + 1.8*min(1, N/1e6))
 *         (a cell row costs ~0.6 us per query term: one segment-table probe per (query, term, doc tile));
 *   doc : 0.13 ms + ceil(B/QT) * stream_bytes / 4.7 TB/s + nnz * 0.1 us * (1 + 2.7*N/1e6)
 *         (one pass over the forward index per tile of QT = 8 (B <= 8) or 16 queries, plus the hit walk).
 * Host arithmetic only (no device call, no handle): num_docs, tile_docs and stream_bytes (forward index + head strips,
 * gs_info_t.bytes_forward + the head share of bytes_head) describe the index; B and nnz the query batch.  Returns
 * GS_ALGO_TERM_PARALLEL or GS_ALGO_DOC_PARALLEL; the two estimates (milliseconds) go to out_term_ms / out_doc_ms when
 * non-null.  Document-parallel wins for one or two long queries (B = 1, >= ~200 terms); term-parallel everywhere else. */
GS_API int32_t gs_dispatch_model(int64_t num_docs, int32_t tile_docs, int64_t stream_bytes, int64_t B, int64_t nnz,
                                 double* out_term_ms, double* out_doc_ms);

/* ------------------------------------------------------------------------------------------------
 * Search (§4-§5).
 * gs_search: queries and outputs are DEVICE pointers.  ASYNCHRONOUS on `stream`: the call only enqueues work (no
 * synchronisation, no allocation, no host read-back), so it can be captured into a CUDA graph and is re-entrant on
 * different streams with different workspaces (document-parallel searches of one device are serialised among
 * themselves: they share one constant-memory query tile).  The one exception is GS_FLAG_VALIDATE_QUERIES, which
 * synchronises to return the validation status.
 * out_doc_ids [B*k] int32, out_scores [B*k] float (GS_W_F32) or int32_t (GS_W_U8), row-major, each row sorted by
 * (score desc, doc id asc).  If k > N, slots >= N hold id -1 and score -inf / INT32_MIN.  Query term ids outside
 * [0,V) are ignored unless validation is on.  B == 0 is legal (nothing is written; the output pointers may then be
 * NULL).  Limits: B <= 65535 queries per call, k <= GS_MAX_K, a query row holds fewer than 2^19 terms (longer rows are
 * treated as empty and reported as GS_ERR_OUT_OF_RANGE under GS_FLAG_VALIDATE_QUERIES).
 * workspace: >= gs_search_workspace_bytes(...) bytes, 256-byte aligned; it must stay untouched until the search (and
 * its gs_search_finish) is done.
 *
 * Exactness and gs_search_finish.  The search filters every (query, doc) cell against a per-query lower bound of the
 * k-th best score taken from a sample of the doc tiles, and keeps the survivors in a candidate list of fixed capacity
 * (8x the expected size).  A query whose list overflows (documents ordered so that the sample is unrepresentative) is
 * counted in gs_stats_t.overflow_queries and its output row is NOT yet exact.  gs_search_finish synchronises `stream`,
 * reads that count and re-runs exactly those queries through the dense path (every score materialised, exact), then
 * synchronises again; with no overflow it costs one stream synchronisation and a 64-byte read-back.  Pass the same
 * arguments as to gs_search.  *out_resolved (may be NULL) receives the number of queries re-run.  A caller that
 * skips gs_search_finish (e.g. inside a captured graph) must check overflow_queries == 0 through gs_search_stats.
 * gs_search_host calls it internally.
 * ---------------------------------------------------------------------------------------------- */
GS_API gs_status_t gs_search_workspace_bytes(const gs_index_t* index, int64_t num_queries, int64_t query_nnz,
                                      int32_t k, const gs_search_opts_t* opts, size_t* out_bytes);
GS_API gs_status_t gs_search(const gs_index_t* index, const gs_csr_t* queries, int32_t k,
                      const gs_search_opts_t* opts, int32_t* out_doc_ids, void* out_scores,
                      void* workspace, size_t workspace_bytes, gs_stream_t stream);
GS_API gs_status_t gs_search_finish(const gs_index_t* index, const gs_csr_t* queries, int32_t k,
                             const gs_search_opts_t* opts, int32_t* out_doc_ids, void* out_scores,
                             void* workspace, size_t workspace_bytes, gs_stream_t stream, int32_t* out_resolved);

/* Same search with HOST buffers: queries->* and the outputs are HOST pointers (pinned memory makes
 * the copies asynchronous).  Copies H2D, searches, copies D2H, synchronises `stream`.  Uses a
 * workspace owned by the handle (grown on demand, hence NOT re-entrant for one handle). */
GS_API gs_status_t gs_search_host(gs_index_t* index, const gs_csr_t* host_queries, int32_t k,
                           const gs_search_opts_t* opts, int32_t* host_doc_ids, void* host_scores,
                           gs_stream_t stream);

/* Synchronises `stream` and copies the counters of the last gs_search on `workspace` to *out. */
GS_API gs_status_t gs_search_stats(const void* workspace, gs_stream_t stream, gs_stats_t* out);

/* Scores only (no top-k): out_scores [B][ld] float|int32 DEVICE, ld >= N.  Element (b,d) is Eq. (4).
 * Used for element-by-element parity of either scoring kernel (algo must not be AUTO). */
GS_API gs_status_t gs_score_dense(const gs_index_t* index, const gs_csr_t* queries, const gs_search_opts_t* opts,
                           void* out_scores, int64_t ld, void* workspace, size_t workspace_bytes,
                           gs_stream_t stream);

/* Top-k alone: rows of a dense DEVICE score matrix [B][ld] (float or int32 per
 * wtype) -> the k best (score desc, id asc) of columns [0,N).  -0.0 ranks equal to +0.0. */
GS_API gs_status_t gs_topk_workspace_bytes(int64_t num_rows, int64_t n, int32_t k, size_t* out_bytes);
GS_API gs_status_t gs_topk_dense(const void* scores, int32_t wtype, int64_t num_rows, int64_t n, int64_t ld,
                          int32_t k, int32_t* out_ids, void* out_scores, void* workspace,
                          size_t workspace_bytes, gs_stream_t stream);

/* gs_topk_dense without a workspace argument and without any allocation, for callers that cannot call cudaMalloc
 * (code under CUDA graph capture, tight serving loops, harnesses that forbid it): the select's scratch lives in a
 * static device array of GS_TOPK_STATIC_SCRATCH_BYTES inside the library (every GPU that loads the library holds it
 * until the process exits).  Same arguments, results and errors as gs_topk_dense, plus: GS_ERR_OUT_OF_RANGE when the
 * call's scratch need — gs_topk_workspace_bytes(num_rows, n, k) — exceeds GS_TOPK_STATIC_SCRATCH_BYTES (2.5 MiB: up to
 * 64 rows at k = GS_MAX_K, 256 rows at k <= 64).  All calls share the array: calls that overlap on
 * the GPU (different streams, or unordered threads) race; order them on one stream.  Asynchronous on `stream`; calls no
 * cudaMalloc, cudaFree or allocating library routine. */
#define GS_TOPK_STATIC_SCRATCH_BYTES 2624000   /* = gs_topk_workspace_bytes(64, n, 4096) */
GS_API gs_status_t gs_topk_dense_static(const void* scores, int32_t wtype, int64_t num_rows, int64_t n, int64_t ld,
                                 int32_t k, int32_t* out_ids, void* out_scores, gs_stream_t stream);

/* Exact merge of partial top-k lists (document sharding; §6.7 L322-324 merges on
 * the host, L430 asks for a device-side merge).  `ids` [n_lists][B][k_in] int32 and `scores` [n_lists][B][k_in]
 * (float | int32 per wtype) are DEVICE arrays: list l holds, for every query, the top-k_in of shard l as returned by
 * gs_search (shard-local doc ids, -1 in unused slots).  `list_doc_base` [n_lists] is a HOST array (or NULL = zeros):
 * the global id of shard l's document 0.  Output: the k_out best of the union per query under (score desc, global
 * doc id asc), rows padded with (-1, -inf | INT32_MIN) when the union is smaller.  Global ids must be distinct and
 * < 2^32 - 1.  n_lists <= GS_MERGE_MAX_LISTS, k_out <= GS_MAX_K.  Asynchronous on `stream`, never allocates. */
#define GS_MERGE_MAX_LISTS 64
GS_API gs_status_t gs_merge_topk_workspace_bytes(int32_t n_lists, int64_t num_queries, int32_t k_in, int32_t k_out,
                                                 size_t* out_bytes);
GS_API gs_status_t gs_merge_topk(int32_t wtype, int32_t n_lists, int64_t num_queries, int32_t k_in, int32_t k_out,
                                 const int32_t* ids, const void* scores, const int64_t* list_doc_base,
                                 int32_t* out_doc_ids, void* out_scores, void* workspace, size_t workspace_bytes,
                                 gs_stream_t stream);

/* ------------------------------------------------------------------------------------------------
 * Kernel timing (SURVEY §8d measurement): when enabled on the calling thread, every kernel launch of
 * the following gs_search / gs_score_dense / gs_topk_dense calls is bracketed by CUDA events on the
 * call's stream; gs_profile_read synchronises those events, returns launch counts and summed device
 * milliseconds per kernel class, and clears the record.  Off by default (no events are recorded).
 * ---------------------------------------------------------------------------------------------- */
#define GS_PROF_CLASSES 8
typedef enum gs_kclass {
    GS_K_INGEST = 0,       /* S1  query ingest                                            */
    GS_K_SCORE_TERM = 1,   /* S2a term-parallel tiled scatter-add (+ head strips)          */
    GS_K_SCORE_DOC = 2,    /* S2b document-parallel forward-index streaming                */
    GS_K_QTILE = 3,        /* S1  transposed query tiles of the document-parallel kernel   */
    GS_K_SELECT = 4,       /* S3  radix select (histogram / scan / collect)                */
    GS_K_SORT = 5,         /* S3  bitonic finish + decode                                  */
    GS_K_MISC = 6          /* zeroing, statistics                                          */
} gs_kclass_t;
typedef struct gs_profile {
    int32_t launches[GS_PROF_CLASSES];
    float ms[GS_PROF_CLASSES];
} gs_profile_t;
GS_API void gs_profile_enable(int32_t on);
GS_API gs_status_t gs_profile_read(gs_profile_t* out);
GS_API const char* gs_kclass_name(int32_t kclass);

GS_API const char* gs_strerror(gs_status_t status);
GS_API const char* gs_version(void);
GS_API int32_t gs_abi_version(void);
GS_API int32_t gs_last_cuda_error(void);    /* cudaError_t of the last GS_ERR_CUDA on this thread */
GS_API int32_t gs_last_launch_count(void);  /* kernels launched by the last search/score/topk call on this thread */

#ifdef __cplusplus
}
#endif
#endif /* GPUSPARSE_H */
