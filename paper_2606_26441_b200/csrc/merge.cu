// merge.cu — exact k-way merge of partial top-k lists (document sharding).
//
// PAPER.md §6.7 L322-324 shards the documents over two GPUs and merges the partial top-k lists on the
// HOST (0.6x of one GPU at 100K docs); L430 (future work 4) asks for a device-side merge.  Contiguous
// doc-id ranges are independent: every shard returns its own [B][k] (local doc id, score) under the
// order (score desc, doc id asc); adding the shard's first doc id makes the ids global, and the k
// best of the union under the same order are exactly the k best of the whole collection, ties
// included.  Here: one kernel turns the gathered lists into 64-bit keys (same composite key as the
// search: ord(score) << 32 | ~doc, all distinct), compacted per query (padding entries, id -1, are
// dropped); the radix select of topk.cu picks and sorts the k best.
#include "gs_internal.cuh"

namespace {

struct MergeParams {
    const int32_t* ids; const uint32_t* scores;      // [n_lists][B][k_in]
    int64_t B; int32_t n_lists; int32_t k_in; int32_t wtype;
    int64_t base[GS_MERGE_MAX_LISTS];                // first global doc id of each list's shard
    uint64_t* keys; uint32_t* counts; int64_t cap;   // [B][cap], [B]
};

// one warp per 32 consecutive entries of one (list, query) row: ballot compaction, one atomic per warp
__global__ void k_merge_keys(const MergeParams p) {
    const int lane = threadIdx.x & 31;
    const int64_t warp = (blockIdx.x * (int64_t)blockDim.x + threadIdx.x) >> 5;
    const int chunks = (p.k_in + 31) / 32;
    const int64_t row = warp / chunks;               // list * B + b
    if (row >= (int64_t)p.n_lists * p.B) return;
    const int j = (int)(warp - row * chunks) * 32 + lane;
    const int l = (int)(row / p.B);
    const int64_t b = row - (int64_t)l * p.B;
    int32_t id = -1;
    uint32_t sc = 0;
    if (j < p.k_in) { id = p.ids[row * p.k_in + j]; sc = p.scores[row * p.k_in + j]; }
    const bool ok = id >= 0;
    const unsigned m = __ballot_sync(0xFFFFFFFFu, ok);
    if (m == 0u) return;
    uint32_t pos = 0;
    if (lane == 0) pos = atomicAdd(&p.counts[b], (uint32_t)__popc(m));
    pos = __shfl_sync(0xFFFFFFFFu, pos, 0) + (uint32_t)__popc(m & ((1u << lane) - 1u));
    if (ok) {
        const uint32_t ord = p.wtype == GS_W_F32 ? gs_ord_f32(sc) : gs_ord_i32(sc);
        p.keys[b * p.cap + pos] = gs_make_key(ord, (uint32_t)((int64_t)id + p.base[l]));
    }
}

}  // namespace

size_t gs_merge_scratch_bytes(int32_t n_lists, int64_t B, int32_t k_in, int32_t k_out) {
    auto up = [](size_t x) { return (x + 255) & ~(size_t)255; };
    return up((size_t)B * 4) + up((size_t)B * (size_t)n_lists * (size_t)k_in * 8) + gs_select_scratch_bytes(B, k_out);
}

gs_status_t gs_launch_merge(int32_t wtype, int32_t n_lists, int64_t B, int32_t k_in, int32_t k_out, const int32_t* ids,
                            const void* scores, const int64_t* base, int32_t* out_ids, void* out_scores, void* scratch,
                            cudaStream_t s) {
    auto up = [](size_t x) { return (x + 255) & ~(size_t)255; };
    MergeParams p{};
    p.ids = ids; p.scores = (const uint32_t*)scores; p.B = B; p.n_lists = n_lists; p.k_in = k_in; p.wtype = wtype;
    for (int l = 0; l < n_lists; ++l) p.base[l] = base ? base[l] : 0;
    unsigned char* w = (unsigned char*)scratch;
    p.counts = (uint32_t*)w; w += up((size_t)B * 4);
    p.keys = (uint64_t*)w; w += up((size_t)B * (size_t)n_lists * (size_t)k_in * 8);
    p.cap = (int64_t)n_lists * k_in;
    GS_CUDA(cudaMemsetAsync(p.counts, 0, (size_t)B * 4, s));
    const int64_t warps = (int64_t)n_lists * B * ((k_in + 31) / 32);
    const int threads = 256;
    {
        GsProfScope ps(GS_K_MISC, s);
        k_merge_keys<<<(unsigned)((warps * 32 + threads - 1) / threads), threads, 0, s>>>(p);
        ++gs_tls_launches;
        GS_CUDA(cudaGetLastError());
    }
    gs_sel_src src{};
    src.keys = p.keys; src.cap = p.cap; src.counts = p.counts; src.wtype = wtype;
    return gs_launch_select(src, B, k_out, out_ids, out_scores, nullptr, nullptr, nullptr, 0, w, s);
}
