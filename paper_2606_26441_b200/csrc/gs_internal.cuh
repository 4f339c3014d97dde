// gs_internal.cuh — internal declarations shared by the CUDA translation units of libgpusparse.
// Nothing here is visible through the C ABI (include/gpusparse.h).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/gpusparse.h"

#define GS_STRIP_MAX 64         // dense strips kept by the index
#define GS_HEAD_MAX GS_STRIP_MAX // entries of a query's compact head list (one per strip at most)
#define GS_HOT_STRIPS 32        // the densest strips: kept in tensor memory by the fp32 batch kernel
#define GS_XSTRIP_MAX 128      // second tier of strips: the next 128 lists ...
#define GS_XDENS 0.05f         // ... of density >= 0.05 (sweep: 64 lists 16.3 ms, 128 15.4, 192 15.3, 384 15.9 per batch)
// GS_XSTRIP_MAX: second tier of dense strips, read from global memory by the term-parallel kernels only
#define GS_MMA_K 192            // strips (head + second tier) of the tensor-core head contraction = K of the integer MMA
#define GS_FWD_DOC_SHIFT 27     // forward term word = term id | (doc id & 31) << 27   (V < 2^27)
#define GS_FWD_CHUNK 128        // a 32-document block of the forward index is padded to a multiple of this many postings
#define GS_TAIL32 32            // tail terms of a query kept in the fixed-stride prefetch table
#define GS_SEL_BINS 2048        // radix-select digit: 11 bits
#define GS_SEL_BITS 11

void gs_set_cuda_error(cudaError_t e);
// Raises a kernel's dynamic shared-memory limit to the device's opt-in maximum, once per (kernel, device): launches then pass
// their actual size, and concurrent callers never see a limit smaller than what they launch with.
cudaError_t gs_optin_smem_impl(const void* kern);
template <typename K> inline cudaError_t gs_optin_smem(K kern) { return gs_optin_smem_impl(reinterpret_cast<const void*>(kern)); }
#define GS_CUDA(call)                                   \
    do {                                                \
        cudaError_t e__ = (call);                       \
        if (e__ != cudaSuccess) {                       \
            gs_set_cuda_error(e__);                     \
            return GS_ERR_CUDA;                         \
        }                                               \
    } while (0)
#define GS_TRY(call)                                    \
    do {                                                \
        gs_status_t s__ = (call);                       \
        if (s__ != GS_OK) return s__;                   \
    } while (0)

// Per-term entry of the tile-segment tables (16 bytes: one 128-bit load).  "Which slots of PL(t) hold documents of doc tile
// j?" is answered in one of two ways, chosen per term at build time:
//   mode GS_SEG_FULL   (len >= ntiles / 2: a posting in every other doc tile or more): seg_tab[tab_off + j] = number of postings of t
//                      with doc tile < j, j in [0, ntiles] — two adjacent loads give the slot range;
//   mode GS_SEG_SPARSE (rare terms, empty in most tiles): seg_l1[tab_off + (j >> 5)] = (bit mask of the non-empty tiles of
//                      the 32-tile group, index into seg_l2 of the group's first non-empty tile); seg_l2[i] = list position
//                      where that tile's postings start, seg_l2[i + 1] = where they end (next non-empty tile, or len).
//                      An empty (term, tile) costs ONE 8-byte load from a table of V * ntiles / 4 bytes (cache resident for
//                      a query's terms); the tables cost O(postings) + V * ntiles / 4 bytes instead of 12 * V * ntiles.
#define GS_SEG_FULL 0u
#define GS_SEG_SPARSE 1u
struct __align__(16) gs_term_meta {
    uint32_t tab_off;     // first entry of the term in seg_tab (full) / seg_l1 (sparse)
    uint32_t mode;        // GS_SEG_FULL | GS_SEG_SPARSE
    uint32_t list_blk;    // start of the term's padded posting list / 32 (lists are padded to 32 slots)
    uint32_t len;         // true list length
};

// ------------------------------------------------------------------------------------------------
// The index handle.  All pointers are device pointers owned by the handle.
// ------------------------------------------------------------------------------------------------
struct gs_index {
    int64_t N = 0;            // documents
    int32_t V = 0;            // vocabulary
    int32_t wtype = 0;        // gs_weight_t
    int64_t P = 0;            // postings
    int64_t P_pad = 0;        // sum of padded lengths (Eq. 2)
    int64_t nonempty = 0;
    int32_t Ts = 512;         // docs per accumulator tile
    int32_t ntiles = 0;       // ceil(N / Ts)
    int64_t N_pad = 0;        // ntiles * Ts
    // forward (doc-major) index — PAPER.md L174.  Hybrid layout: the H strip terms of a document live in the
    // dense strips below (column-major, 0 = absent); every other posting lives in this "tail" block CSR: one
    // row pointer per aligned block of 32 documents, each block's range padded to GS_FWD_CHUNK postings.
    int64_t* fwd_blk = nullptr;      // [n_blk+1] start of each block's range (multiple of GS_FWD_CHUNK)
    uint32_t* fwd_terms = nullptr;   // [P_fwd] term id | (doc & 31) << GS_FWD_DOC_SHIFT; padding = V | 31 << shift
    void* fwd_w = nullptr;           // [P_fwd] float | uint8 (0 in the padding)
    int64_t n_blk = 0;               // ceil(N / 32)
    int64_t P_tail = 0;              // postings of the terms without a strip
    int64_t P_fwd = 0;               // P_tail + block padding
    // inverted index — PAPER.md L79-90
    int64_t* inv_off = nullptr;      // [V+1] start of each padded list (multiple of 32)
    int32_t* inv_len = nullptr;      // [V]   true list length
    int32_t* inv_doc = nullptr;      // [P_pad] doc ids, ascending within a list, -1 in the padding
    void* inv_w = nullptr;           // [P_pad] float | uint8, 0 in the padding
    // compressed postings, integer-impact mode (gs_build_opts_t.pack_postings): when inv_packed, the two arrays above are
    // replaced by ONE word per posting, doc id | impact << 24 (N < 2^24; padding 0xFFFFFFFF); when fwd_packed, fwd_w is
    // gone and a forward term word is term | impact << 19 | (doc & 31) << 27 (V < 2^19)
    uint32_t* inv_pk = nullptr;      // [P_pad]
    bool inv_packed = false, fwd_packed = false;
    // tile-segment tables (see gs_term_meta)
    gs_term_meta* term_meta = nullptr;   // [V]
    uint32_t* seg_tab = nullptr;         // full-mode terms: [n_full][ntiles + 1]
    uint2* seg_l1 = nullptr;             // sparse-mode terms: [n_sparse][ceil(ntiles / 32)] (mask, seg_l2 index)
    uint32_t* seg_l2 = nullptr;          // sparse-mode terms: segment starts of the non-empty (term, tile) pairs + one end per term
    int64_t seg_entries = 0;             // entries of seg_tab
    int64_t seg_l1_entries = 0, seg_l2_entries = 0;
    // dense strips of the densest lists ("head" terms)
    int32_t H = 0;                   // strips (<= GS_STRIP_MAX), densest list first
    int32_t head_terms_host[GS_STRIP_MAX];
    int16_t* head_slot = nullptr;    // [V]: strip number of a term or -1
    void* head_strip = nullptr;      // [H][N_pad] float | uint8 (0 where the doc is not in the list)
    // second tier ("x strips"): the next densest lists (up to 128 of density >= 0.05), a dense copy used by the term-parallel kernels
    // only — there they replace the scatter of a 50-130-posting segment per doc tile by four 128-bit loads and eight
    // FFMA2; the lists stay tail terms everywhere else (forward index, document-parallel kernel)
    int32_t HX = 0;
    int16_t* xslot = nullptr;        // [V]: x-strip number of a term or -1
    void* xstrip = nullptr;          // [HX][N_pad]
    // Integer-impact mode, 512-doc tiles: the strips once more, as the A operand of the tensor-core head contraction
    // (k_score_term_mma).  Per doc tile 4 sub-tiles of 128 documents; a sub-tile is a 128 x GS_MMA_K matrix of
    // uint8 (row = document, column = strip: head strips in columns 0..63, second-tier strips in 64..191, 0 where there is no
    // strip) in the K-major no-swizzle core-matrix layout tcgen05.mma reads from shared memory: [K/16][128/8][8 rows][16 B],
    // so a sub-tile is ONE contiguous block of 24 KB and a doc tile one 1-D TMA bulk copy of 96 KB.
    uint8_t* mma_strips = nullptr;   // [ntiles][4][GS_MMA_K/16][16][8][16]
    // allocator
    gs_alloc_t alloc{};
    bool has_alloc = false;
    // workspace owned by the handle for gs_search_host
    void* host_ws = nullptr;
    size_t host_ws_bytes = 0;
    void* host_stage = nullptr;      // device staging for queries and outputs
    size_t host_stage_bytes = 0;
    int64_t bytes_inverted = 0, bytes_meta = 0, bytes_forward = 0, bytes_head = 0;
};

void* gs_dev_alloc(const gs_index* ix, size_t bytes, cudaStream_t s);
void gs_dev_free(const gs_index* ix, void* p, cudaStream_t s);

// ------------------------------------------------------------------------------------------------
// Order-preserving keys.  A 64-bit composite key makes the order (score desc, doc id asc) a strict
// total order on distinct documents: key = ord(score) << 32 | (0xFFFFFFFF - doc id).
// ------------------------------------------------------------------------------------------------
__host__ __device__ __forceinline__ uint32_t gs_ord_f32(uint32_t bits) {
    if (bits == 0x80000000u) bits = 0u;                      // -0.0 ranks equal to +0.0
    return (bits & 0x80000000u) ? ~bits : (bits | 0x80000000u);
}
__host__ __device__ __forceinline__ uint32_t gs_unord_f32(uint32_t o) {
    return (o & 0x80000000u) ? (o & 0x7FFFFFFFu) : ~o;
}
__host__ __device__ __forceinline__ uint32_t gs_ord_i32(uint32_t bits) { return bits ^ 0x80000000u; }
__host__ __device__ __forceinline__ uint64_t gs_make_key(uint32_t ord, uint32_t doc) {
    return ((uint64_t)ord << 32) | (uint64_t)(0xFFFFFFFFu - doc);
}
template <int WT>
__device__ __forceinline__ uint32_t gs_ord_bits(uint32_t bits) {
    return WT == GS_W_F32 ? gs_ord_f32(bits) : gs_ord_i32(bits);
}

// ------------------------------------------------------------------------------------------------
// Query batch after ingest (S1): per-query compact head-term lists + compacted tail term lists.
// Accumulator type: float (GS_W_F32) or int32 (GS_W_U8), both 4 bytes, stored as uint32 bit patterns.
// ------------------------------------------------------------------------------------------------
struct gs_qbatch {
    int64_t B = 0;
    int64_t nnz = 0;
    const int64_t* indptr = nullptr;   // caller's CSR indptr (device)
    uint2* head_pair = nullptr;        // [B][GS_HEAD_MAX] compact (strip number, accumulator-typed weight bits): the "hot" strips
                                       // (number < GS_HOT_STRIPS) from entry 0 upwards, the others from the last entry downwards
    int32_t* head_cnt = nullptr;       // [B] head terms of the query | hot ones << 8
    uint2* xpair = nullptr;            // [B][GS_XSTRIP_MAX] compact (x-strip number, weight bits); used when x_on
    int32_t* xcnt = nullptr;           // [B]
    bool x_on = false;                 // the batch's x-strip terms are in xpair (and NOT in the tail lists)
    uint4* tail_desc = nullptr;        // [nnz] compacted at indptr[b] .. indptr[b]+tail_cnt[b]: per tail term
                                       // (accumulator-typed weight bits, segment-table offset, segment-table mode, list start / 32)
    int32_t* tail_cnt = nullptr;       // [B]
    uint4* tail32 = nullptr;           // [B][32] the first 32 tail terms, same entries (mode = 0xFFFFFFFF: no term): a
                                       // fixed-stride copy the batch kernel can prefetch without reading indptr first
    int32_t* status = nullptr;         // device status word: first validation error (gs_status_t) or 0
};

// Where a scoring kernel puts its results.
//   dense : scores[(b - q0) * ld + col] for the doc tiles it was given (col = compact tile index * Ts + d)
//   filter: append key64 to cand[b * cand_cap + n] when key >= thr[b]
struct gs_tileset {
    int32_t first = 0;       // first doc tile
    int32_t stride = 1;      // tile j of the set is doc tile first + j*stride
    int32_t count = 0;       // number of tiles in the set
};
// Candidate counters sit one per 128-byte line.  A document-parallel pass adds to the counters of its 16 queries once per
// passing cell (2 M atomics per pass at 8.8M docs): packed into one line they all queue at one L2 slice, and the pass time
// then depended on where the workspace happened to lie (15.0 vs 20.3 ms per 128-query search for workspaces 2 MB apart).
#define GS_CNT_STRIDE 32
struct gs_sink {
    uint32_t* dense = nullptr;
    int64_t ld = 0;
    const uint64_t* thr = nullptr;       // [B] threshold keys (filter mode when non-null)
    uint64_t* cand = nullptr;            // [B][cand_cap]
    uint32_t* cand_cnt = nullptr;        // [B * GS_CNT_STRIDE]: query b's counter is cand_cnt[b * GS_CNT_STRIDE]
    int64_t cand_cap = 0;
};

// ------------------------------------------------------------------------------------------------
// Launchers (one per translation unit).  Each returns GS_OK or GS_ERR_CUDA and counts its launches.
// ------------------------------------------------------------------------------------------------
extern thread_local int32_t gs_tls_launches;

// Brackets the launches issued during its lifetime with CUDA events when gs_profile_enable(1) is set
// on the calling thread (no-op otherwise).  `n` = kernels launched inside the scope.
struct GsProfScope {
    GsProfScope(int kclass, cudaStream_t s, int n = 1);
    ~GsProfScope();
    GsProfScope(const GsProfScope&) = delete;
    GsProfScope& operator=(const GsProfScope&) = delete;
    int slot = -1;
    cudaStream_t stream = nullptr;
};

gs_status_t gs_launch_ingest(const gs_index* ix, const gs_csr_t* q, bool validate, bool use_head, bool use_x,
                             gs_qbatch* qb, cudaStream_t s);
bool gs_score_term_wants_x(const gs_index* ix, int64_t nq, int group, bool use_head);   // the batch kernel will run

gs_status_t gs_launch_score_term(const gs_index* ix, const gs_qbatch& qb, int64_t q0, int64_t nq, int group,
                                 bool use_head, bool use_mma, const gs_tileset& ts, const gs_sink& sink, cudaStream_t s);

int gs_score_term_group(const gs_index* ix, int64_t nq, int group, bool use_head);   // cell rows (warps) per CTA actually used
int gs_score_doc_qtile(int qtile);                                    // queries per pass actually used

// doc-parallel: scratch holds the transposed query tile(s)
size_t gs_score_doc_scratch_bytes_ex(const gs_index* ix, int qtile, int64_t nq, int64_t q_nnz);
gs_status_t gs_launch_score_doc(const gs_index* ix, const gs_csr_t* q, const gs_qbatch& qb, int64_t q0, int64_t nq,
                                int qtile, const gs_tileset& ts, const gs_sink& sink, void* scratch,
                                cudaStream_t s);

// top-k selection (S3).  Source = dense score rows or candidate key lists.
struct gs_sel_src {
    // dense
    const uint32_t* dense = nullptr;
    int64_t ld = 0;
    int64_t n_cols = 0;        // columns per row (compact); column c maps to doc via tileset/Ts
    int64_t n_docs = 0;        // columns whose doc id >= n_docs are ignored
    gs_tileset ts{};
    int32_t Ts = 0;            // 0: column == doc id
    // list
    const uint64_t* keys = nullptr;
    int64_t cap = 0;
    const uint32_t* counts = nullptr;
    int32_t cnt_stride = 1;    // row b's count is counts[b * cnt_stride]
    int32_t wtype = 0;
};
size_t gs_select_scratch_bytes(int64_t rows, int32_t k);
// Selects the k best of every row; writes sorted results to out_ids/out_scores (row stride k) when
// non-null, and the k-th key (threshold) of each row to out_thr when non-null.  When out_keys is
// non-null the selected (unsorted) keys are ALSO appended to out_keys[b*out_cap + ..] / out_cnt[b].
gs_status_t gs_launch_select(const gs_sel_src& src, int64_t rows, int32_t k, int32_t* out_ids, void* out_scores,
                             uint64_t* out_thr, uint64_t* out_keys, uint32_t* out_cnt, int64_t out_cap,
                             void* scratch, cudaStream_t s);

// k-way merge of partial top-k lists (merge.cu)
size_t gs_merge_scratch_bytes(int32_t n_lists, int64_t B, int32_t k_in, int32_t k_out);
gs_status_t gs_launch_merge(int32_t wtype, int32_t n_lists, int64_t B, int32_t k_in, int32_t k_out, const int32_t* ids,
                            const void* scores, const int64_t* base, int32_t* out_ids, void* out_scores, void* scratch,
                            cudaStream_t s);
