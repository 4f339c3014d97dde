// ingest.cu — S1: validate and reorganise the CSR query batch for the scoring kernels.
//
// The paper pads queries to a [B, M] matrix of (term id, weight) in Python (PAPER.md L120-123,
// L146-152).  Here one warp per query splits its terms into
//   * head terms (the H densest lists, kept as dense strips): compact list head_pair[b][..] of (strip number, weight), the
//     "hot" strips (the GS_HOT_STRIPS densest, held in tensor memory by the fp32 batch kernel) from the front, the others
//     from the back;
//   * tail terms: compacted (row b starts at indptr[b]) into tail_desc: weight converted to the accumulator type (float,
//     or int32 for uint8 impacts) + the term's entry of the compact tile-segment table (table offset, table mode, list start),
//     looked up HERE once per (query, term) instead of once per (query, term, doc tile); the first 32 of them are also
//     written to the fixed-stride table tail32[b][32], which the batch kernel prefetches two rows ahead.
// Term ids outside [0,V) are dropped (memory safety); with validation on, the first error
// (out of range / duplicate / non-finite) is recorded in a status word the host reads back.
#include "gs_internal.cuh"

namespace {

template <int WT>
__global__ void k_ingest(const int64_t* __restrict__ indptr, const int32_t* __restrict__ terms,
                         const void* __restrict__ weights, int64_t B, int32_t V, const int16_t* __restrict__ head_slot,
                         int h_term, const int16_t* __restrict__ xslot, int h_x, uint2* __restrict__ xpair,
                         int32_t* __restrict__ xcnt, int validate, uint2* __restrict__ head_pair,
                         int32_t* __restrict__ head_cnt,
                         const gs_term_meta* __restrict__ term_meta, uint4* __restrict__ tail_desc,
                         int32_t* __restrict__ tail_cnt, uint4* __restrict__ tail32,
                         int32_t* __restrict__ status, int64_t nnz) {
    const int lane = threadIdx.x & 31;
    const int64_t b = (blockIdx.x * (int64_t)blockDim.x + threadIdx.x) >> 5;
    if (b >= B) return;
    int64_t a = indptr[b], e = indptr[b + 1];
    // memory safety: the row's range must lie inside the nnz-sized arrays (always checked); a bad row is treated as empty
    // and reported as GS_ERR_OUT_OF_RANGE (returned to the caller when validation is on)
    if (a < 0 || e < a || e > nnz || (b == 0 && a != 0) || e - a >= (1 << 19)) {      // rows of >= 2^19 terms: not supported
        if (lane == 0) atomicCAS(status, 0, (int)GS_ERR_OUT_OF_RANGE);
        a = e = 0;
    }
    int32_t n_tail = 0, n_hot = 0, n_cold = 0, n_x = 0;
    tail32[b * GS_TAIL32 + lane] = make_uint4(0u, 0u, 0xFFFFFFFFu, 0u);
    __syncwarp();
    for (int64_t i0 = a; i0 < e; i0 += 32) {
        const int64_t i = i0 + lane;
        int32_t t = -1;
        uint32_t w = 0;
        bool ok = false;
        if (i < e) {
            t = terms[i];
            ok = t >= 0 && t < V;
            if (WT == GS_W_F32) {
                float x = ((const float*)weights)[i];
                w = __float_as_uint(x);
                if (validate && !isfinite(x)) atomicCAS(status, 0, (int)GS_ERR_NONFINITE);
            } else {
                w = (uint32_t)((const uint8_t*)weights)[i];
            }
            if (validate && !ok) atomicCAS(status, 0, (int)GS_ERR_OUT_OF_RANGE);
            if (validate && ok) {   // duplicates: compare with every earlier entry of the row
                for (int64_t j = a; j < i; ++j)
                    if (terms[j] == t) { atomicCAS(status, 0, (int)GS_ERR_DUPLICATE_TERM); break; }
            }
        }
        int slot = (ok && h_term > 0) ? (int)head_slot[t] : -1;
        if (slot >= h_term) slot = -1;
        // a valid row holds each head term at most once, so the two ends of the list never meet; the bounds only protect
        // memory when a (non-validated) row repeats a term — entries beyond them are dropped and flagged
        const bool is_hot = ok && slot >= 0 && slot < GS_HOT_STRIPS, is_cold = ok && slot >= GS_HOT_STRIPS;
        const unsigned mhot = __ballot_sync(0xFFFFFFFFu, is_hot), mcold = __ballot_sync(0xFFFFFFFFu, is_cold);
        if (is_hot) {
            const int dst = n_hot + __popc(mhot & ((1u << lane) - 1u));
            if (dst < GS_HOT_STRIPS) head_pair[b * GS_HEAD_MAX + dst] = make_uint2((uint32_t)slot, w);
            else atomicCAS(status, 0, (int)GS_ERR_DUPLICATE_TERM);
        }
        if (is_cold) {
            const int dst = n_cold + __popc(mcold & ((1u << lane) - 1u));
            if (dst < GS_HEAD_MAX - GS_HOT_STRIPS) head_pair[b * GS_HEAD_MAX + (GS_HEAD_MAX - 1 - dst)] = make_uint2((uint32_t)slot, w);
            else atomicCAS(status, 0, (int)GS_ERR_DUPLICATE_TERM);
        }
        n_hot = min(GS_HOT_STRIPS, n_hot + __popc(mhot));
        n_cold = min(GS_HEAD_MAX - GS_HOT_STRIPS, n_cold + __popc(mcold));
        // second-tier strips (term-parallel batch searches): their own compact list, not the tail
        int xs = (ok && slot < 0 && h_x > 0) ? (int)xslot[t] : -1;
        if (xs >= h_x) xs = -1;
        const unsigned mx = __ballot_sync(0xFFFFFFFFu, xs >= 0);
        if (xs >= 0) {
            const int dst = n_x + __popc(mx & ((1u << lane) - 1u));
            if (dst < GS_XSTRIP_MAX) xpair[b * GS_XSTRIP_MAX + dst] = make_uint2((uint32_t)xs, w);
            else atomicCAS(status, 0, (int)GS_ERR_DUPLICATE_TERM);
        }
        n_x = min(GS_XSTRIP_MAX, n_x + __popc(mx));
        const bool is_tail = ok && slot < 0 && xs < 0;
        const unsigned m = __ballot_sync(0xFFFFFFFFu, is_tail);
        if (is_tail) {
            const int64_t dst = a + n_tail + __popc(m & ((1u << lane) - 1u));
            const gs_term_meta tm = term_meta[t];
            const uint4 d = make_uint4(w, tm.tab_off, tm.mode, tm.list_blk);
            tail_desc[dst] = d;
            if (dst - a < GS_TAIL32) tail32[b * GS_TAIL32 + (dst - a)] = d;
        }
        n_tail += __popc(m);
        __syncwarp();
    }
    if (lane == 0) { tail_cnt[b] = n_tail; head_cnt[b] = (n_hot + n_cold) | (n_hot << 8); xcnt[b] = n_x; }
    // fourth word of the lane's tail32 entry: the query's counts, so that the batch kernels get them with the term in one
    // 16-byte load: tail terms (19 bits) | cold head terms << 19 (6 bits) | hot head terms << 25 (6 bits) | bit 31: the
    // lane's own term is a sparse-mode list (second-level segment lookup)
    {
        uint4* e = tail32 + b * GS_TAIL32 + lane;
        const uint32_t mode = e->z;                 // written above, possibly by another lane (ordered by the __syncwarp)
        e->w = (uint32_t)n_tail | ((uint32_t)n_cold << 19) | ((uint32_t)n_hot << 25) | (mode == GS_SEG_SPARSE ? 0x80000000u : 0u);
    }
}

}  // namespace

gs_status_t gs_launch_ingest(const gs_index* ix, const gs_csr_t* q, bool validate, bool use_head, bool use_x,
                             gs_qbatch* qb, cudaStream_t s) {
    const int64_t B = q->rows;
    const int h_x = (use_head && use_x && ix->HX > 0) ? ix->HX : 0;
    qb->x_on = h_x > 0;
    GS_CUDA(cudaMemsetAsync(qb->status, 0, sizeof(int32_t), s));
    if (B == 0) return GS_OK;
    const int threads = 128;
    const unsigned grid = (unsigned)((B * 32 + threads - 1) / threads);
    GsProfScope ps(GS_K_INGEST, s);
    if (ix->wtype == GS_W_F32)
        k_ingest<GS_W_F32><<<grid, threads, 0, s>>>(q->indptr, q->term_ids, q->weights, B, ix->V, ix->head_slot,
                                                   use_head ? ix->H : 0, ix->xslot, h_x, qb->xpair, qb->xcnt, validate, qb->head_pair, qb->head_cnt, ix->term_meta,
                                                   qb->tail_desc, qb->tail_cnt, qb->tail32, qb->status, q->nnz);
    else
        k_ingest<GS_W_U8><<<grid, threads, 0, s>>>(q->indptr, q->term_ids, q->weights, B, ix->V, ix->head_slot,
                                                  use_head ? ix->H : 0, ix->xslot, h_x, qb->xpair, qb->xcnt, validate, qb->head_pair, qb->head_cnt, ix->term_meta,
                                                  qb->tail_desc, qb->tail_cnt, qb->tail32, qb->status, q->nnz);
    ++gs_tls_launches;
    GS_CUDA(cudaGetLastError());
    return GS_OK;
}
