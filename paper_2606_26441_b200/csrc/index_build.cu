// index_build.cu — S0: doc CSR -> GPU-resident inverted index + forward index + tile segments + head strips.
//
// PAPER.md §3 (L67-100): two flat arrays doc_ids(int32)/scores(fp32) with per-term offsets/lengths
// (L79-84); every list padded to a multiple of W=32 with (doc_id=-1, score=0) and sorted by doc id
// (Eq. 2); no delta coding (L75).  Additions of this build: a per-(term, doc
// tile) segment table so a kernel can find the slice of a list inside a doc-id range without
// searching, and dense strips for the few lists that cover >= half the collection.
//
// Because CSR rows arrive in doc order, a STABLE sort of the postings by term id yields doc-id-sorted
// lists directly.  The sort is cub::DeviceRadixSort (a library primitive; the build is not on the
// timed path).
#include <cub/device/device_radix_sort.cuh>
#include <cub/device/device_scan.cuh>

#include <algorithm>
#include <vector>

#include "gs_internal.cuh"

namespace {

constexpr int kThreads = 256;

// err[0] = first error code seen
__global__ void k_check_indptr(const int64_t* __restrict__ indptr, int64_t rows, int* err) {
    int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (i < rows && indptr[i + 1] < indptr[i]) atomicCAS(err, 0, (int)GS_ERR_OUT_OF_RANGE);
}

template <int WT>
__global__ void k_check_entries(const int32_t* __restrict__ terms, const void* __restrict__ w, int64_t nnz, int32_t V,
                                int* err) {
    int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (i >= nnz) return;
    int32_t t = terms[i];
    if (t < 0 || t >= V) atomicCAS(err, 0, (int)GS_ERR_OUT_OF_RANGE);
    if (WT == GS_W_F32) {
        float x = ((const float*)w)[i];
        if (!isfinite(x)) atomicCAS(err, 0, (int)GS_ERR_NONFINITE);
    }
}

// term histogram with a full-vocabulary shared-memory privatised copy when it fits
__global__ void k_term_hist(const int32_t* __restrict__ terms, int64_t nnz, int32_t V, int32_t* __restrict__ counts,
                            int use_smem) {
    extern __shared__ int32_t sh[];
    if (use_smem) {
        for (int i = threadIdx.x; i < V; i += blockDim.x) sh[i] = 0;
        __syncthreads();
    }
    for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < nnz; i += (int64_t)gridDim.x * blockDim.x) {
        int32_t t = terms[i];
        if (t < 0 || t >= V) continue;
        if (use_smem) atomicAdd(&sh[t], 1);
        else atomicAdd(&counts[t], 1);
    }
    if (use_smem) {
        __syncthreads();
        for (int i = threadIdx.x; i < V; i += blockDim.x)
            if (sh[i]) atomicAdd(&counts[i], sh[i]);
    }
}

__global__ void k_iota(uint32_t* __restrict__ v, int64_t n) {
    int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (i < n) v[i] = (uint32_t)i;
}

// one warp per document: write the doc id over its posting range
__global__ void k_expand_rows(const int64_t* __restrict__ indptr, int64_t rows, int32_t* __restrict__ rowid) {
    int64_t warp = (blockIdx.x * (int64_t)blockDim.x + threadIdx.x) >> 5;
    int lane = threadIdx.x & 31;
    if (warp >= rows) return;
    int64_t a = indptr[warp], b = indptr[warp + 1];
    for (int64_t i = a + lane; i < b; i += 32) rowid[i] = (int32_t)warp;
}

// sorted position j (term-major, stable) -> padded slot
template <typename W>
__global__ void k_scatter_padded(const int32_t* __restrict__ sorted_terms, const uint32_t* __restrict__ sorted_src,
                                 const int32_t* __restrict__ rowid, const W* __restrict__ w_in,
                                 const int64_t* __restrict__ cnt_scan, const int64_t* __restrict__ inv_off,
                                 int64_t nnz, int32_t* __restrict__ inv_doc, W* __restrict__ inv_w) {
    int64_t j = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (j >= nnz) return;
    int32_t t = sorted_terms[j];
    uint32_t src = sorted_src[j];
    int64_t pos = inv_off[t] + (j - cnt_scan[t]);
    inv_doc[pos] = rowid[src];
    inv_w[pos] = w_in[src];
}

__device__ __forceinline__ int32_t term_of_slot(const int64_t* __restrict__ inv_off, int32_t V, int64_t pos) {
    // largest t with inv_off[t] <= pos
    int32_t lo = 0, hi = V;   // answer in [lo, hi)
    while (hi - lo > 1) {
        int32_t mid = (lo + hi) >> 1;
        if (inv_off[mid] <= pos) lo = mid; else hi = mid;
    }
    return lo;
}

// Per padded slot: duplicate detection (equal neighbours inside a list) + the tile-segment tables (gs_term_meta).
// Full mode: the posting at list position i in doc tile j writes i into the entries (tile of its predecessor, j]; the last
// posting fills the rest with len.  Sparse mode, pass 0: the first posting of a tile sets the tile's bit in its 32-tile group;
// pass 1 (after the prefix sums over the masks): it writes its list position into the tile's seg_l2 entry, and the last
// posting of the list writes the closing entry (len).
__global__ void k_segments(const int64_t* __restrict__ inv_off, const int32_t* __restrict__ inv_len,
                           const int32_t* __restrict__ inv_doc, int32_t V, int64_t P_pad, int32_t Ts, int32_t ntiles,
                           const gs_term_meta* __restrict__ meta, uint32_t* __restrict__ tab, uint2* __restrict__ l1,
                           uint32_t* __restrict__ l2, const uint32_t* __restrict__ l2_end, int pass, int* err) {
    int64_t pos = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (pos >= P_pad) return;
    int32_t t = term_of_slot(inv_off, V, pos);
    int32_t i = (int32_t)(pos - inv_off[t]);
    int32_t len = inv_len[t];
    if (i >= len) return;                       // padding slot
    const gs_term_meta m = meta[t];
    const uint32_t abs0 = (uint32_t)inv_off[t];          // the tables hold absolute posting slots (P_pad < 2^32)
    int32_t doc = inv_doc[pos];
    int32_t tile_cur = doc / Ts;
    int32_t tile_prev = -1;
    if (i > 0) {
        int32_t prev = inv_doc[pos - 1];
        if (prev == doc && pass == 0) atomicCAS(err, 0, (int)GS_ERR_DUPLICATE_TERM);
        tile_prev = prev / Ts;
    }
    if (m.mode == GS_SEG_FULL) {
        if (pass != 0) return;
        uint32_t* row = tab + m.tab_off;
        for (int32_t j = tile_prev + 1; j <= tile_cur; ++j) row[j] = abs0 + (uint32_t)i;
        if (i == len - 1)
            for (int32_t j = tile_cur + 1; j <= ntiles; ++j) row[j] = abs0 + (uint32_t)len;
        return;
    }
    uint2* g = l1 + m.tab_off + (tile_cur >> 5);
    if (pass == 0) {
        if (tile_cur != tile_prev) atomicOr(&g->x, 1u << (tile_cur & 31));
        return;
    }
    if (tile_cur != tile_prev) {
        const uint2 e = *g;
        l2[e.y + (uint32_t)__popc(e.x & ((1u << (tile_cur & 31)) - 1u))] = abs0 + (uint32_t)i;
    }
    if (i == len - 1) l2[l2_end[t]] = abs0 + (uint32_t)len;
}

// Sparse-mode terms, one warp per term: running count of the non-empty tiles before each 32-tile group -> l1[g].y
// (relative to the term), count of the term's non-empty tiles + 1 (the closing entry) -> cnt[t]; 0 for the other terms.
__global__ void k_l1_count(const gs_term_meta* __restrict__ meta, int32_t V, int32_t n_grp, uint2* __restrict__ l1,
                           uint32_t* __restrict__ cnt) {
    const int64_t t = (blockIdx.x * (int64_t)blockDim.x + threadIdx.x) >> 5;
    const int lane = threadIdx.x & 31;
    if (t >= V) return;
    const gs_term_meta m = meta[t];
    if (m.mode != GS_SEG_SPARSE || m.len == 0) { if (lane == 0) cnt[t] = 0u; return; }
    uint32_t run = 0;
    for (int32_t g0 = 0; g0 < n_grp; g0 += 32) {
        const int32_t g = g0 + lane;
        const uint32_t c = g < n_grp ? (uint32_t)__popc(l1[m.tab_off + g].x) : 0u;
        uint32_t incl = c;
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t v = __shfl_up_sync(0xFFFFFFFFu, incl, o);
            if (lane >= o) incl += v;
        }
        if (g < n_grp) l1[m.tab_off + g].y = run + incl - c;
        run += __shfl_sync(0xFFFFFFFFu, incl, 31);
    }
    if (lane == 0) cnt[t] = run + 1u;
}

// l1[g].y += start of the term's entries in seg_l2; l2_end[t] = index of the term's closing entry
__global__ void k_l1_rebase(const gs_term_meta* __restrict__ meta, int32_t V, int32_t n_grp, const uint32_t* __restrict__ cnt,
                            const uint32_t* __restrict__ base, uint2* __restrict__ l1, uint32_t* __restrict__ l2_end) {
    const int64_t t = (blockIdx.x * (int64_t)blockDim.x + threadIdx.x) >> 5;
    const int lane = threadIdx.x & 31;
    if (t >= V) return;
    const gs_term_meta m = meta[t];
    if (cnt[t] == 0u) { if (lane == 0) l2_end[t] = 0u; return; }
    const uint32_t b = base[t];
    for (int32_t g = lane; g < n_grp; g += 32) l1[m.tab_off + g].y += b;
    if (lane == 0) l2_end[t] = b + cnt[t] - 1u;
}

template <typename W>
__global__ void k_fill_strip(const int32_t* __restrict__ inv_doc, const W* __restrict__ inv_w, int64_t off, int32_t len,
                             W* __restrict__ strip) {
    int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (i < len) strip[inv_doc[off + i]] = inv_w[off + i];
}

// forward "tail" index: the postings of a document whose term has no dense strip, in the row's order, stored per
// aligned block of 32 documents as ONE flat range padded to a multiple of GS_FWD_CHUNK postings.  The term word also
// carries the document's position inside its block (bits 27..31), so a warp that streams a block's range with
// 128-bit loads knows the owner of each posting without a search; padding slots hold the term id V (never a query
// term) at position 31 with weight 0.  One warp per document counts, one warp per block lays the block out, one
// warp per document writes.
__global__ void k_tail_count(const int64_t* __restrict__ indptr, const int32_t* __restrict__ terms,
                             const int16_t* __restrict__ head_slot, int64_t rows, int32_t V, int32_t* __restrict__ cnt) {
    const int64_t warp = (blockIdx.x * (int64_t)blockDim.x + threadIdx.x) >> 5;
    const int lane = threadIdx.x & 31;
    if (warp >= rows) return;
    const int64_t a = indptr[warp], b = indptr[warp + 1];
    int n = 0;
    for (int64_t i = a + lane; i < b; i += 32) {
        const int32_t t = terms[i];
        n += (t >= 0 && t < V && head_slot[t] < 0) ? 1 : 0;
    }
    for (int o = 16; o > 0; o >>= 1) n += __shfl_xor_sync(0xFFFFFFFFu, n, o);
    if (lane == 0) cnt[warp] = n;
}

// lane = document of the block: start of the document inside the block, padded size of the block
__global__ void k_blk_layout(const int32_t* __restrict__ cnt, int64_t rows, int64_t nblk, int32_t* __restrict__ doc_rel,
                             int64_t* __restrict__ blk_cnt, unsigned long long* __restrict__ true_total) {
    const int64_t blk = (blockIdx.x * (int64_t)blockDim.x + threadIdx.x) >> 5;
    const int lane = threadIdx.x & 31;
    if (blk >= nblk) return;
    const int64_t doc = blk * 32 + lane;
    const int c = doc < rows ? cnt[doc] : 0;
    int incl = c;
    for (int o = 1; o < 32; o <<= 1) {
        const int v = __shfl_up_sync(0xFFFFFFFFu, incl, o);
        if (lane >= o) incl += v;
    }
    if (doc < rows) doc_rel[doc] = incl - c;
    if (lane == 31) {
        blk_cnt[blk] = ((int64_t)incl + GS_FWD_CHUNK - 1) / GS_FWD_CHUNK * GS_FWD_CHUNK;
        atomicAdd(true_total, (unsigned long long)incl);
    }
}

__global__ void k_fill_u32(uint32_t* __restrict__ p, int64_t n, uint32_t v) {
    for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) p[i] = v;
}

template <typename W>
__global__ void k_tail_fill(const int64_t* __restrict__ indptr, const int32_t* __restrict__ terms, const W* __restrict__ w,
                            const int16_t* __restrict__ head_slot, int64_t rows, int32_t V,
                            const int64_t* __restrict__ fwd_blk, const int32_t* __restrict__ doc_rel,
                            uint32_t* __restrict__ out_terms, W* __restrict__ out_w) {
    const int64_t warp = (blockIdx.x * (int64_t)blockDim.x + threadIdx.x) >> 5;
    const int lane = threadIdx.x & 31;
    if (warp >= rows) return;
    const int64_t a = indptr[warp], b = indptr[warp + 1];
    int64_t dst = fwd_blk[warp >> 5] + doc_rel[warp];
    for (int64_t i0 = a; i0 < b; i0 += 32) {
        const int64_t i = i0 + lane;
        int32_t t = -1;
        bool keep = false;
        if (i < b) {
            t = terms[i];
            keep = t >= 0 && t < V && head_slot[t] < 0;
        }
        const unsigned m = __ballot_sync(0xFFFFFFFFu, keep);
        if (keep) {
            const int64_t o = dst + __popc(m & ((1u << lane) - 1u));
            out_terms[o] = (uint32_t)t | ((uint32_t)(warp & 31) << GS_FWD_DOC_SHIFT);
            out_w[o] = w[i];
        }
        dst += __popc(m);
    }
}

// integer-impact mode, compressed postings: (doc id, impact) -> doc | impact << 24; the padding (doc -1) -> 0xFFFFFFFF
__global__ void k_pack_inv(const int32_t* __restrict__ doc, const uint8_t* __restrict__ w, int64_t n, uint32_t* __restrict__ pk) {
    for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
        const int32_t d = doc[i];
        pk[i] = d < 0 ? 0xFFFFFFFFu : ((uint32_t)d | ((uint32_t)w[i] << 24));
    }
}
// forward term word (term | doc-in-block << 27) takes the impact into bits 19..26 (V < 2^19)
__global__ void k_pack_fwd(uint32_t* __restrict__ terms, const uint8_t* __restrict__ w, int64_t n) {
    for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x)
        terms[i] |= (uint32_t)w[i] << 19;
}

// A operand of the tensor-core head contraction (gs_index::mma_strips): one thread per 16-byte unit = (doc, 16 strips)
__global__ void k_build_mma_strips(const uint8_t* __restrict__ head, int H, const uint8_t* __restrict__ xs, int HX, int64_t N_pad,
                                   int32_t ntiles, uint8_t* __restrict__ out) {
    constexpr int KC = GS_MMA_K / 16;
    const int64_t u = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;           // unit = ((tile*4 + s)*KC + kc)*128 + row
    if (u >= (int64_t)ntiles * 4 * KC * 128) return;
    const int row = (int)(u & 127);
    const int kc = (int)((u >> 7) % KC);
    const int64_t ts = (u >> 7) / KC;                                           // tile*4 + s
    const int64_t doc = ts * 128 + row;
    uint32_t w[4] = {0u, 0u, 0u, 0u};
#pragma unroll
    for (int kb = 0; kb < 16; ++kb) {
        const int k = kc * 16 + kb;
        uint32_t v = 0u;
        if (k < GS_STRIP_MAX) { if (k < H) v = head[(size_t)k * N_pad + doc]; }
        else if (k - GS_STRIP_MAX < HX) v = xs[(size_t)(k - GS_STRIP_MAX) * N_pad + doc];
        w[kb >> 2] |= v << (8 * (kb & 3));
    }
    // core matrix (kc, rg = row/8): 8 rows of 16 bytes
    uint4* dst = reinterpret_cast<uint4*>(out + (size_t)ts * (KC * 2048) + (size_t)(kc * 16 + (row >> 3)) * 128 + (row & 7) * 16);
    *dst = make_uint4(w[0], w[1], w[2], w[3]);
}

inline unsigned grid_for(int64_t n, int threads = kThreads) { return (unsigned)((n + threads - 1) / threads); }

}  // namespace

void* gs_dev_alloc(const gs_index* ix, size_t bytes, cudaStream_t s) {
    if (bytes == 0) bytes = 256;
    if (ix && ix->has_alloc) return ix->alloc.alloc(bytes, (gs_stream_t)s, ix->alloc.user);
    void* p = nullptr;
    if (cudaMalloc(&p, bytes) != cudaSuccess) { cudaGetLastError(); return nullptr; }
    return p;
}
void gs_dev_free(const gs_index* ix, void* p, cudaStream_t s) {
    if (!p) return;
    if (ix && ix->has_alloc) ix->alloc.free(p, (gs_stream_t)s, ix->alloc.user);
    else cudaFree(p);
}

namespace {
struct Temp {   // frees build temporaries on every exit path
    const gs_index* ix; cudaStream_t s; std::vector<void*> ptrs;
    void* get(size_t bytes) { void* p = gs_dev_alloc(ix, bytes, s); if (p) ptrs.push_back(p); return p; }
    ~Temp() { cudaStreamSynchronize(s); for (void* p : ptrs) gs_dev_free(ix, p, s); }
};

template <typename W>
gs_status_t build_typed(gs_index* ix, const gs_csr_t* docs, const gs_build_opts_t& o, cudaStream_t s) {
    const int64_t N = ix->N, P = ix->P;
    const int32_t V = ix->V;
    constexpr int WT = sizeof(W) == 4 ? GS_W_F32 : GS_W_U8;
    Temp tmp{ix, s, {}};
    int* d_err = (int*)tmp.get(sizeof(int));
    if (!d_err) return GS_ERR_OOM;
    GS_CUDA(cudaMemsetAsync(d_err, 0, sizeof(int), s));

    if (N > 0) k_check_indptr<<<grid_for(N), kThreads, 0, s>>>(docs->indptr, N, d_err);
    if (o.validate && P > 0)
        k_check_entries<WT><<<grid_for(P), kThreads, 0, s>>>(docs->term_ids, docs->weights, P, V, d_err);
    int h_err = 0;
    GS_CUDA(cudaMemcpyAsync(&h_err, d_err, sizeof(int), cudaMemcpyDeviceToHost, s));
    GS_CUDA(cudaStreamSynchronize(s));
    if (h_err) return (gs_status_t)h_err;

    // ---- list lengths
    ix->inv_len = (int32_t*)gs_dev_alloc(ix, sizeof(int32_t) * (size_t)V, s);
    ix->inv_off = (int64_t*)gs_dev_alloc(ix, sizeof(int64_t) * (size_t)(V + 1), s);
    if (!ix->inv_len || !ix->inv_off) return GS_ERR_OOM;
    GS_CUDA(cudaMemsetAsync(ix->inv_len, 0, sizeof(int32_t) * (size_t)V, s));
    if (P > 0) {
        int dev = 0, smem_max = 0, sms = 0;
        cudaGetDevice(&dev);
        cudaDeviceGetAttribute(&smem_max, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
        size_t need = sizeof(int32_t) * (size_t)V;
        int use_smem = need <= (size_t)smem_max;
        if (use_smem) GS_CUDA(cudaFuncSetAttribute(k_term_hist, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)need));
        k_term_hist<<<sms * 2, 512, use_smem ? need : 0, s>>>(docs->term_ids, P, V, ix->inv_len, use_smem);
    }
    std::vector<int32_t> h_len(V);
    GS_CUDA(cudaMemcpyAsync(h_len.data(), ix->inv_len, sizeof(int32_t) * (size_t)V, cudaMemcpyDeviceToHost, s));
    GS_CUDA(cudaStreamSynchronize(s));

    // ---- host: padded offsets (Eq. 2), unpadded scan, head selection
    std::vector<int64_t> h_off(V + 1), h_scan(V + 1);
    int64_t acc = 0, accp = 0, nonempty = 0;
    for (int32_t t = 0; t < V; ++t) {
        h_scan[t] = acc;
        h_off[t] = accp;
        acc += h_len[t];
        accp += ((int64_t)h_len[t] + GS_WARP_BLOCK - 1) / GS_WARP_BLOCK * GS_WARP_BLOCK;
        nonempty += h_len[t] > 0;
    }
    h_scan[V] = acc;
    h_off[V] = accp;
    if (acc != P) return GS_ERR_OUT_OF_RANGE;   // some term id was outside [0,V) (validate off)
    ix->P_pad = accp;
    ix->nonempty = nonempty;
    if (accp >= 0xFFFFFFF0LL) return GS_ERR_OUT_OF_RANGE;      // posting slots are 32-bit in the segment tables and kernels
    GS_CUDA(cudaMemcpyAsync(ix->inv_off, h_off.data(), sizeof(int64_t) * (size_t)(V + 1), cudaMemcpyHostToDevice, s));

    std::vector<int32_t> order;
    int hmax = o.head_max < 0 ? 0 : (o.head_max == 0 ? GS_STRIP_MAX : std::min(o.head_max, GS_STRIP_MAX));
    float dens = o.head_density > 0.f ? o.head_density : 0.25f;
    for (int32_t t = 0; t < V; ++t)
        if (N > 0 && (double)h_len[t] >= (double)dens * (double)N && h_len[t] > 0) order.push_back(t);
    std::stable_sort(order.begin(), order.end(), [&](int32_t a, int32_t b) { return h_len[a] > h_len[b]; });
    if ((int)order.size() > hmax) order.resize(hmax);
    ix->H = (int32_t)order.size();
    std::vector<int16_t> h_slot(V, (int16_t)-1);
    for (int h = 0; h < GS_STRIP_MAX; ++h) ix->head_terms_host[h] = h < ix->H ? order[h] : -1;
    for (int h = 0; h < ix->H; ++h) h_slot[order[h]] = (int16_t)h;
    ix->head_slot = (int16_t*)gs_dev_alloc(ix, sizeof(int16_t) * (size_t)V, s);
    if (!ix->head_slot) return GS_ERR_OOM;
    GS_CUDA(cudaMemcpyAsync(ix->head_slot, h_slot.data(), sizeof(int16_t) * (size_t)V, cudaMemcpyHostToDevice, s));

    // ---- second tier of strips for the term-parallel kernels (512-doc tiles only: the batch kernel is their user)
    std::vector<int32_t> xorder;
    if (o.head_max >= 0 && ix->Ts == 512 && N > 0) {
        const float xdens = std::min(dens, GS_XDENS);
        for (int32_t t = 0; t < V; ++t)
            if (h_slot[t] < 0 && h_len[t] > 0 && (double)h_len[t] >= (double)xdens * (double)N) xorder.push_back(t);
        std::stable_sort(xorder.begin(), xorder.end(), [&](int32_t a, int32_t b) { return h_len[a] > h_len[b]; });
        if ((int)xorder.size() > GS_XSTRIP_MAX) xorder.resize(GS_XSTRIP_MAX);
    }
    ix->HX = (int32_t)xorder.size();
    if (ix->HX > 0) {
        std::vector<int16_t> x_slot(V, (int16_t)-1);
        for (int h = 0; h < ix->HX; ++h) x_slot[xorder[h]] = (int16_t)h;
        ix->xslot = (int16_t*)gs_dev_alloc(ix, sizeof(int16_t) * (size_t)V, s);
        if (!ix->xslot) return GS_ERR_OOM;
        GS_CUDA(cudaMemcpyAsync(ix->xslot, x_slot.data(), sizeof(int16_t) * (size_t)V, cudaMemcpyHostToDevice, s));
        GS_CUDA(cudaStreamSynchronize(s));        // x_slot is a local
    }

    // ---- forward index, hybrid: strips for the H densest lists + a block CSR of every other posting
    {
        int64_t p_tail = P;
        for (int h = 0; h < ix->H; ++h) p_tail -= h_len[order[h]];
        ix->P_tail = p_tail;
        const int64_t nblk = (N + 31) / 32;
        ix->n_blk = nblk;
        ix->fwd_blk = (int64_t*)gs_dev_alloc(ix, sizeof(int64_t) * (size_t)(nblk + 1), s);
        if (!ix->fwd_blk) return GS_ERR_OOM;
        int32_t* d_cnt = (int32_t*)tmp.get(sizeof(int32_t) * (size_t)std::max<int64_t>(N, 1));
        int32_t* d_rel = (int32_t*)tmp.get(sizeof(int32_t) * (size_t)std::max<int64_t>(N, 1));
        int64_t* d_blk_cnt = (int64_t*)tmp.get(sizeof(int64_t) * (size_t)(nblk + 1));
        unsigned long long* d_true = (unsigned long long*)tmp.get(sizeof(unsigned long long));
        if (!d_cnt || !d_rel || !d_blk_cnt || !d_true) return GS_ERR_OOM;
        GS_CUDA(cudaMemsetAsync(d_blk_cnt, 0, sizeof(int64_t) * (size_t)(nblk + 1), s));
        GS_CUDA(cudaMemsetAsync(d_true, 0, sizeof(unsigned long long), s));
        if (N > 0) {
            k_tail_count<<<grid_for(N * 32), kThreads, 0, s>>>(docs->indptr, docs->term_ids, ix->head_slot, N, V, d_cnt);
            k_blk_layout<<<grid_for(nblk * 32), kThreads, 0, s>>>(d_cnt, N, nblk, d_rel, d_blk_cnt, d_true);
        }
        if (nblk + 1 > 0x7FFFFFFFLL) return GS_ERR_OUT_OF_RANGE;
        size_t scan_bytes = 0;
        GS_CUDA(cub::DeviceScan::ExclusiveSum(nullptr, scan_bytes, d_blk_cnt, ix->fwd_blk, (int)(nblk + 1), s));
        void* d_scan_tmp = tmp.get(scan_bytes);
        if (!d_scan_tmp) return GS_ERR_OOM;
        GS_CUDA(cub::DeviceScan::ExclusiveSum(d_scan_tmp, scan_bytes, d_blk_cnt, ix->fwd_blk, (int)(nblk + 1), s));
        int64_t p_fwd = 0;
        unsigned long long true_total = 0;
        GS_CUDA(cudaMemcpyAsync(&p_fwd, ix->fwd_blk + nblk, sizeof(int64_t), cudaMemcpyDeviceToHost, s));
        GS_CUDA(cudaMemcpyAsync(&true_total, d_true, sizeof(unsigned long long), cudaMemcpyDeviceToHost, s));
        GS_CUDA(cudaStreamSynchronize(s));
        if ((int64_t)true_total != p_tail) return GS_ERR_OUT_OF_RANGE;     // some term id was outside [0,V) (validate off)
        ix->P_fwd = p_fwd;
        ix->fwd_terms = (uint32_t*)gs_dev_alloc(ix, sizeof(uint32_t) * (size_t)std::max<int64_t>(p_fwd, 1), s);
        ix->fwd_w = gs_dev_alloc(ix, sizeof(W) * (size_t)std::max<int64_t>(p_fwd, 1), s);
        if (!ix->fwd_terms || !ix->fwd_w) return GS_ERR_OOM;
        if (p_fwd > 0) {
            int dev = 0, sms = 0;
            cudaGetDevice(&dev);
            cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
            k_fill_u32<<<sms * 8, 512, 0, s>>>(ix->fwd_terms, p_fwd, (uint32_t)V | (31u << GS_FWD_DOC_SHIFT));
            GS_CUDA(cudaMemsetAsync(ix->fwd_w, 0, sizeof(W) * (size_t)p_fwd, s));
            k_tail_fill<W><<<grid_for(N * 32), kThreads, 0, s>>>(docs->indptr, docs->term_ids, (const W*)docs->weights,
                                                                ix->head_slot, N, V, ix->fwd_blk, d_rel, ix->fwd_terms,
                                                                (W*)ix->fwd_w);
        }
        ix->bytes_forward = (int64_t)(sizeof(int64_t) * (size_t)(nblk + 1) + (sizeof(uint32_t) + sizeof(W)) * (size_t)p_fwd);
        if (WT == GS_W_U8 && o.pack_postings >= 0 && V < (1 << 19)) {
            if (p_fwd > 0) {
                int dev = 0, sms = 0;
                cudaGetDevice(&dev);
                cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
                k_pack_fwd<<<sms * 8, 512, 0, s>>>(ix->fwd_terms, (const uint8_t*)ix->fwd_w, p_fwd);
                GS_CUDA(cudaStreamSynchronize(s));
                GS_CUDA(cudaGetLastError());
            }
            gs_dev_free(ix, ix->fwd_w, s);
            ix->fwd_w = nullptr;
            ix->fwd_packed = true;
            ix->bytes_forward = (int64_t)(sizeof(int64_t) * (size_t)(nblk + 1) + sizeof(uint32_t) * (size_t)p_fwd);
        }
    }

    // ---- padded inverted arrays, pre-filled with the sentinel (doc_id=-1, score=0), L90
    ix->inv_doc = (int32_t*)gs_dev_alloc(ix, sizeof(int32_t) * (size_t)ix->P_pad, s);
    ix->inv_w = gs_dev_alloc(ix, sizeof(W) * (size_t)ix->P_pad, s);
    if (!ix->inv_doc || !ix->inv_w) return GS_ERR_OOM;
    if (ix->P_pad > 0) {
        GS_CUDA(cudaMemsetAsync(ix->inv_doc, 0xFF, sizeof(int32_t) * (size_t)ix->P_pad, s));
        GS_CUDA(cudaMemsetAsync(ix->inv_w, 0, sizeof(W) * (size_t)ix->P_pad, s));
    }
    ix->bytes_inverted = (int64_t)((sizeof(int32_t) + sizeof(W)) * (size_t)ix->P_pad);

    // ---- tile-segment tables: a full per-tile table for the lists that reach almost every doc tile, the two-level
    // bitmap + segment-start arrays for the others (gs_term_meta)
    const int32_t n_grp = (ix->ntiles + 31) / 32;
    {
        std::vector<gs_term_meta> h_meta((size_t)V);
        int64_t n_ent = 0, n_l1 = 0;
        for (int32_t t = 0; t < V; ++t) {
            // full mode from one posting per two doc tiles on: the two-level lookup of the sparse mode costs a dependent load
            // when the tile is not empty.  Tables: 1.00 GB at a threshold of 2 postings per tile, 1.21 GB at 1/2, 2.10 GB at
            // 1/8 (8.8M docs); same-box A/B of 2 vs 1/2 on the 500-query batch: 16.75 vs 16.6 ms, i.e. within the run-to-run
            // noise (B200 units of the pool differ by ~5 %, which an earlier cross-box comparison mistook for a gain)
            const bool full = (int64_t)h_len[t] * 2 >= (int64_t)ix->ntiles && h_len[t] > 0;
            h_meta[t].mode = full ? GS_SEG_FULL : GS_SEG_SPARSE;
            h_meta[t].tab_off = (uint32_t)(full ? n_ent : n_l1);
            h_meta[t].list_blk = (uint32_t)(h_off[t] / GS_WARP_BLOCK);
            h_meta[t].len = (uint32_t)h_len[t];
            if (full) n_ent += ix->ntiles + 1; else n_l1 += n_grp;
            if (n_ent >= 0xFFFFFFF0LL || n_l1 >= 0xFFFFFFF0LL || h_off[t] / GS_WARP_BLOCK > 0xFFFFFFFFLL) return GS_ERR_OUT_OF_RANGE;
        }
        ix->seg_entries = n_ent;
        ix->seg_l1_entries = n_l1;
        ix->term_meta = (gs_term_meta*)gs_dev_alloc(ix, sizeof(gs_term_meta) * (size_t)V, s);
        ix->seg_tab = (uint32_t*)gs_dev_alloc(ix, sizeof(uint32_t) * (size_t)std::max<int64_t>(n_ent, 1), s);
        ix->seg_l1 = (uint2*)gs_dev_alloc(ix, sizeof(uint2) * (size_t)std::max<int64_t>(n_l1, 1), s);
        if (!ix->term_meta || !ix->seg_tab || !ix->seg_l1) return GS_ERR_OOM;
        GS_CUDA(cudaMemcpyAsync(ix->term_meta, h_meta.data(), sizeof(gs_term_meta) * (size_t)V, cudaMemcpyHostToDevice, s));
        GS_CUDA(cudaMemsetAsync(ix->seg_tab, 0, sizeof(uint32_t) * (size_t)std::max<int64_t>(n_ent, 1), s));
        GS_CUDA(cudaMemsetAsync(ix->seg_l1, 0, sizeof(uint2) * (size_t)std::max<int64_t>(n_l1, 1), s));
        GS_CUDA(cudaStreamSynchronize(s));            // h_meta is a local
    }

    if (P > 0) {
        // ---- stable sort of (term, source position) by term
        int32_t* d_sorted_terms = (int32_t*)tmp.get(sizeof(int32_t) * (size_t)P);
        uint32_t* d_src_in = (uint32_t*)tmp.get(sizeof(uint32_t) * (size_t)P);
        uint32_t* d_src_out = (uint32_t*)tmp.get(sizeof(uint32_t) * (size_t)P);
        int32_t* d_rowid = (int32_t*)tmp.get(sizeof(int32_t) * (size_t)P);
        int64_t* d_scan = (int64_t*)tmp.get(sizeof(int64_t) * (size_t)(V + 1));
        if (!d_sorted_terms || !d_src_in || !d_src_out || !d_rowid || !d_scan) return GS_ERR_OOM;
        GS_CUDA(cudaMemcpyAsync(d_scan, h_scan.data(), sizeof(int64_t) * (size_t)(V + 1), cudaMemcpyHostToDevice, s));
        k_iota<<<grid_for(P), kThreads, 0, s>>>(d_src_in, P);
        k_expand_rows<<<grid_for(N * 32), kThreads, 0, s>>>(docs->indptr, N, d_rowid);
        int end_bit = 1;
        while ((1 << end_bit) < V) ++end_bit;
        size_t cub_bytes = 0;
        if (P > 0x7FFFFFFFLL) return GS_ERR_OUT_OF_RANGE;   // cub item counts are int
        GS_CUDA(cub::DeviceRadixSort::SortPairs(nullptr, cub_bytes, docs->term_ids, d_sorted_terms, d_src_in, d_src_out,
                                                (int)P, 0, end_bit, s));
        void* d_cub = tmp.get(cub_bytes);
        if (!d_cub) return GS_ERR_OOM;
        GS_CUDA(cub::DeviceRadixSort::SortPairs(d_cub, cub_bytes, docs->term_ids, d_sorted_terms, d_src_in, d_src_out,
                                                (int)P, 0, end_bit, s));
        k_scatter_padded<W><<<grid_for(P), kThreads, 0, s>>>(d_sorted_terms, d_src_out, d_rowid, (const W*)docs->weights,
                                                            d_scan, ix->inv_off, P, ix->inv_doc, (W*)ix->inv_w);
        k_segments<<<grid_for(ix->P_pad), kThreads, 0, s>>>(ix->inv_off, ix->inv_len, ix->inv_doc, V, ix->P_pad, ix->Ts,
                                                            ix->ntiles, ix->term_meta, ix->seg_tab, ix->seg_l1, nullptr, nullptr,
                                                            0, d_err);
        GS_CUDA(cudaMemcpyAsync(&h_err, d_err, sizeof(int), cudaMemcpyDeviceToHost, s));
        GS_CUDA(cudaStreamSynchronize(s));
        GS_CUDA(cudaGetLastError());
        if (h_err && o.validate) return (gs_status_t)h_err;
        // sparse-mode terms: prefix sums over the tile masks, then the segment starts
        uint32_t* d_cnt = (uint32_t*)tmp.get(sizeof(uint32_t) * (size_t)(V + 1));
        uint32_t* d_base = (uint32_t*)tmp.get(sizeof(uint32_t) * (size_t)(V + 1));
        uint32_t* d_end = (uint32_t*)tmp.get(sizeof(uint32_t) * (size_t)V);
        if (!d_cnt || !d_base || !d_end) return GS_ERR_OOM;
        GS_CUDA(cudaMemsetAsync(d_cnt, 0, sizeof(uint32_t) * (size_t)(V + 1), s));
        k_l1_count<<<grid_for((int64_t)V * 32), kThreads, 0, s>>>(ix->term_meta, V, n_grp, ix->seg_l1, d_cnt);
        size_t sb = 0;
        GS_CUDA(cub::DeviceScan::ExclusiveSum(nullptr, sb, d_cnt, d_base, V + 1, s));
        void* d_sb = tmp.get(sb);
        if (!d_sb) return GS_ERR_OOM;
        GS_CUDA(cub::DeviceScan::ExclusiveSum(d_sb, sb, d_cnt, d_base, V + 1, s));
        uint32_t n_l2 = 0;
        GS_CUDA(cudaMemcpyAsync(&n_l2, d_base + V, sizeof(uint32_t), cudaMemcpyDeviceToHost, s));
        GS_CUDA(cudaStreamSynchronize(s));
        ix->seg_l2_entries = (int64_t)n_l2;
        ix->seg_l2 = (uint32_t*)gs_dev_alloc(ix, sizeof(uint32_t) * (size_t)std::max<uint32_t>(n_l2, 1u), s);
        if (!ix->seg_l2) return GS_ERR_OOM;
        k_l1_rebase<<<grid_for((int64_t)V * 32), kThreads, 0, s>>>(ix->term_meta, V, n_grp, d_cnt, d_base, ix->seg_l1, d_end);
        k_segments<<<grid_for(ix->P_pad), kThreads, 0, s>>>(ix->inv_off, ix->inv_len, ix->inv_doc, V, ix->P_pad, ix->Ts,
                                                            ix->ntiles, ix->term_meta, ix->seg_tab, ix->seg_l1, ix->seg_l2, d_end,
                                                            1, d_err);
        GS_CUDA(cudaStreamSynchronize(s));
        GS_CUDA(cudaGetLastError());
    }
    ix->bytes_meta = (int64_t)(sizeof(uint32_t) * (size_t)ix->seg_entries + sizeof(uint2) * (size_t)ix->seg_l1_entries +
                               sizeof(uint32_t) * (size_t)ix->seg_l2_entries + sizeof(gs_term_meta) * (size_t)V +
                               sizeof(int64_t) * (size_t)(V + 1) + sizeof(int32_t) * (size_t)V + 2 * sizeof(int16_t) * (size_t)V);
    // ---- dense strips of the head lists
    if (ix->H > 0) {
        size_t strip_bytes = sizeof(W) * (size_t)ix->H * (size_t)ix->N_pad;
        ix->head_strip = gs_dev_alloc(ix, strip_bytes, s);
        if (!ix->head_strip) return GS_ERR_OOM;
        GS_CUDA(cudaMemsetAsync(ix->head_strip, 0, strip_bytes, s));
        for (int h = 0; h < ix->H; ++h) {
            int32_t t = order[h];
            k_fill_strip<W><<<grid_for(h_len[t]), kThreads, 0, s>>>(ix->inv_doc, (const W*)ix->inv_w, h_off[t], h_len[t],
                                                                   (W*)ix->head_strip + (size_t)h * (size_t)ix->N_pad);
        }
        ix->bytes_head = (int64_t)strip_bytes;
    }
    if (ix->HX > 0) {
        size_t xbytes = sizeof(W) * (size_t)ix->HX * (size_t)ix->N_pad;
        ix->xstrip = gs_dev_alloc(ix, xbytes, s);
        if (!ix->xstrip) return GS_ERR_OOM;
        GS_CUDA(cudaMemsetAsync(ix->xstrip, 0, xbytes, s));
        for (int h = 0; h < ix->HX; ++h) {
            int32_t t = xorder[h];
            k_fill_strip<W><<<grid_for(h_len[t]), kThreads, 0, s>>>(ix->inv_doc, (const W*)ix->inv_w, h_off[t], h_len[t],
                                                                   (W*)ix->xstrip + (size_t)h * (size_t)ix->N_pad);
        }
        ix->bytes_head += (int64_t)xbytes;
    }
    GS_CUDA(cudaStreamSynchronize(s));
    GS_CUDA(cudaGetLastError());
    // ---- integer-impact mode: the strips as the A operand of the tensor-core head contraction
    if (WT == GS_W_U8 && ix->Ts == 512 && ix->H > 0 && ix->ntiles > 0) {
        const size_t bytes = (size_t)ix->ntiles * 4 * (GS_MMA_K / 16) * 2048;
        ix->mma_strips = (uint8_t*)gs_dev_alloc(ix, bytes, s);
        if (!ix->mma_strips) return GS_ERR_OOM;
        const int64_t units = (int64_t)ix->ntiles * 4 * (GS_MMA_K / 16) * 128;
        k_build_mma_strips<<<grid_for(units), kThreads, 0, s>>>((const uint8_t*)ix->head_strip, ix->H, (const uint8_t*)ix->xstrip, ix->HX,
                                                              ix->N_pad, ix->ntiles, ix->mma_strips);
        GS_CUDA(cudaStreamSynchronize(s));
        GS_CUDA(cudaGetLastError());
        ix->bytes_head += (int64_t)bytes;
    }
    // ---- compressed postings (integer-impact mode): one word per posting replaces the two arrays
    if (WT == GS_W_U8 && o.pack_postings >= 0 && N < (1 << 24)) {
        ix->inv_pk = (uint32_t*)gs_dev_alloc(ix, sizeof(uint32_t) * (size_t)std::max<int64_t>(ix->P_pad, 1), s);
        if (!ix->inv_pk) return GS_ERR_OOM;
        if (ix->P_pad > 0) {
            int dev = 0, sms = 0;
            cudaGetDevice(&dev);
            cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
            k_pack_inv<<<sms * 8, 512, 0, s>>>(ix->inv_doc, (const uint8_t*)ix->inv_w, ix->P_pad, ix->inv_pk);
            GS_CUDA(cudaStreamSynchronize(s));
            GS_CUDA(cudaGetLastError());
        }
        gs_dev_free(ix, ix->inv_doc, s);
        gs_dev_free(ix, ix->inv_w, s);
        ix->inv_doc = nullptr;
        ix->inv_w = nullptr;
        ix->inv_packed = true;
        ix->bytes_inverted = (int64_t)(sizeof(uint32_t) * (size_t)ix->P_pad);
    }
    return GS_OK;
}
}  // namespace

gs_status_t gs_build_index_impl(gs_index* ix, const gs_csr_t* docs, const gs_build_opts_t& o, cudaStream_t s) {
    return ix->wtype == GS_W_F32 ? build_typed<float>(ix, docs, o, s) : build_typed<uint8_t>(ix, docs, o, s);
}
