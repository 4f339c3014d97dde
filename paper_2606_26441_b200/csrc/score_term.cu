// score_term.cu — S2a: term-at-a-time batched scatter-add, tiled by doc-id range (kernel K1').
//
// PAPER.md Eq. (5): scores[d] += w_i * PL(t_i)[d] for all d in PL(t_i), one independent
// scatter per query term; the paper launches one program per (query, term) that atomically adds
// into a global [B,N] buffer (L118-125, L137-172) and names "scattered atomics" as the cost
// (L172, L411).  Here the doc-id axis is cut into tiles of Ts docs; a CTA owns a block of
// (query, doc-tile) cells whose accumulators live in SHARED memory; each cell is owned by exactly
// one warp, so accumulation is plain LDS/FFMA/STS in a fixed order (no atomics, deterministic),
// and the per-(term, tile) segment table turns "the part of PL(t) inside this tile" into two loads.
// Posting slices are read with aligned, coalesced 128-byte warp loads (lists are padded to 32).
//
// Lists stored as dense strips ("head" terms, >= half of all docs) are not scattered: thread d of
// the epilogue keeps the strip values of its document in registers and adds the dot product with
// the query's dense head weights (read through shared-memory broadcasts).
#include <algorithm>

#include "gs_internal.cuh"

namespace {

constexpr int kThreads = 512;
constexpr int kWarps = kThreads / 32;

template <int WT> struct Num;
template <> struct Num<GS_W_F32> {
    using W = float;
    using A = float;
    static __device__ __forceinline__ A qw(uint32_t bits) { return __uint_as_float(bits); }
    static __device__ __forceinline__ A mac(A acc, A q, W w) { return fmaf(q, w, acc); }
    static __device__ __forceinline__ uint32_t bits(A a) { return __float_as_uint(a); }
};
template <> struct Num<GS_W_U8> {
    using W = uint8_t;
    using A = int32_t;
    static __device__ __forceinline__ A qw(uint32_t bits) { return (int32_t)bits; }
    static __device__ __forceinline__ A mac(A acc, A q, W w) { return acc + q * (int32_t)w; }
    static __device__ __forceinline__ uint32_t bits(A a) { return (uint32_t)a; }
};

struct TermParams {
    // index
    const int64_t* inv_off; const int32_t* inv_doc; const void* inv_w; const uint32_t* seg;
    const void* head_strip; int32_t H; int64_t N; int64_t N_pad; int32_t Ts; int32_t ntiles;
    // queries
    const int64_t* q_indptr; const uint32_t* head_w; const int32_t* tail_term; const uint32_t* tail_w;
    const int32_t* tail_cnt;
    int64_t q0; int32_t nq; int32_t G;          // queries [q0, q0+nq), G per CTA
    int32_t n_qgroups;
    // tiles
    gs_tileset ts; int32_t m;                   // m tiles of the set per CTA
    gs_sink sink;
};

template <int WT>
__device__ __forceinline__ void emit(const TermParams& p, int64_t b, int32_t col, int32_t doc,
                                     typename Num<WT>::A s) {
    const uint32_t bits = Num<WT>::bits(s);
    if (p.sink.thr == nullptr) {
        p.sink.dense[(b - p.q0) * p.sink.ld + col] = bits;
    } else {
        const uint64_t key = gs_make_key(gs_ord_bits<WT>(bits), (uint32_t)doc);
        if (key >= p.sink.thr[b]) {
            const uint32_t pos = atomicAdd(&p.sink.cand_cnt[b], 1u);
            if ((int64_t)pos < p.sink.cand_cap) p.sink.cand[b * p.sink.cand_cap + pos] = key;
        }
    }
}

template <int WT, bool HEAD>
__global__ void __launch_bounds__(kThreads, 1) k_score_term(const TermParams p) {
    using W = typename Num<WT>::W;
    using A = typename Num<WT>::A;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    A* acc = reinterpret_cast<A*>(smem_raw);                       // [cells][Ts]
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int qg = blockIdx.x % p.n_qgroups;
    const int tg = blockIdx.x / p.n_qgroups;
    const int g0 = qg * p.G;
    const int Gc = min(p.G, p.nq - g0);                            // queries in this CTA
    const int j0 = tg * p.m;
    const int mc = min(p.m, p.ts.count - j0);                      // tiles in this CTA
    const int ncells = Gc * mc;
    const int Ts = p.Ts;
    A* headq = acc + (size_t)p.G * p.m * Ts;                       // [G][32] dense head weights (HEAD only)

    for (int i = threadIdx.x; i < ncells * Ts; i += kThreads) acc[i] = A(0);
    if (HEAD)
        for (int i = threadIdx.x; i < Gc * GS_HEAD_MAX; i += kThreads)
            headq[i] = Num<WT>::qw(p.head_w[(p.q0 + g0) * GS_HEAD_MAX + i]);
    __syncthreads();

    // ---- scatter phase: warp `warp` owns cells warp, warp+16, ...  (cell = (sub tile, query))
    const W* __restrict__ inv_w = reinterpret_cast<const W*>(p.inv_w);
    for (int c = warp; c < ncells; c += kWarps) {
        const int g = c % Gc, sub = c / Gc;
        const int64_t b = p.q0 + g0 + g;
        const int tile = p.ts.first + (j0 + sub) * p.ts.stride;
        const int32_t base = tile * Ts;
        A* row = acc + (size_t)c * Ts;
        const int64_t qa = p.q_indptr[b];
        const int cnt = p.tail_cnt[b];
        for (int i0 = 0; i0 < cnt; i0 += 32) {
            int64_t off = 0;
            uint32_t lo = 0, hi = 0, wq = 0;
            if (i0 + lane < cnt) {
                const int32_t t = p.tail_term[qa + i0 + lane];
                wq = p.tail_w[qa + i0 + lane];
                const uint32_t* sr = p.seg + (size_t)t * (p.ntiles + 1) + tile;
                lo = sr[0];
                hi = sr[1];
                off = p.inv_off[t];
            }
            const int nt = min(32, cnt - i0);
            for (int j = 0; j < nt; ++j) {
                const uint32_t lo_j = __shfl_sync(0xFFFFFFFFu, lo, j);
                const uint32_t hi_j = __shfl_sync(0xFFFFFFFFu, hi, j);
                if (lo_j >= hi_j) continue;
                const int64_t off_j = __shfl_sync(0xFFFFFFFFu, off, j);
                const A q = Num<WT>::qw(__shfl_sync(0xFFFFFFFFu, wq, j));
                for (uint32_t pp = (lo_j & ~31u) + lane; pp < hi_j; pp += 32) {
                    const int32_t rel = p.inv_doc[off_j + pp] - base;
                    if ((uint32_t)rel < (uint32_t)Ts) row[rel] = Num<WT>::mac(row[rel], q, inv_w[off_j + pp]);
                }
            }
        }
    }
    __syncthreads();

    // ---- epilogue: (+ head dot product) and hand every cell to the sink
    const W* __restrict__ strip = reinterpret_cast<const W*>(p.head_strip);
    for (int sub = 0; sub < mc; ++sub) {
        const int tile = p.ts.first + (j0 + sub) * p.ts.stride;
        for (int d = threadIdx.x; d < Ts; d += kThreads) {
            const int64_t doc = (int64_t)tile * Ts + d;
            const bool live = doc < p.N;
            A dreg[GS_HEAD_MAX];
            if (HEAD) {
#pragma unroll
                for (int h = 0; h < GS_HEAD_MAX; ++h)
                    dreg[h] = (h < p.H && live) ? (A)strip[(size_t)h * p.N_pad + doc] : A(0);
            }
            const int32_t col = (j0 + sub) * Ts + d;
            for (int g = 0; g < Gc; ++g) {
                A s = acc[(size_t)(sub * Gc + g) * Ts + d];
                if (HEAD) {
                    const A* hq = headq + g * GS_HEAD_MAX;
#pragma unroll
                    for (int h = 0; h < GS_HEAD_MAX; ++h) s = Num<WT>::mac(s, hq[h], (W)dreg[h]);
                }
                if (live) emit<WT>(p, p.q0 + g0 + g, col, (int32_t)doc, s);
            }
        }
    }
}

template <int WT, bool HEAD>
gs_status_t launch(const TermParams& p, unsigned grid, size_t smem, cudaStream_t s) {
    GS_CUDA(cudaFuncSetAttribute(k_score_term<WT, HEAD>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    {
        GsProfScope ps(GS_K_SCORE_TERM, s);
        k_score_term<WT, HEAD><<<grid, kThreads, smem, s>>>(p);
    }
    ++gs_tls_launches;
    GS_CUDA(cudaGetLastError());
    return GS_OK;
}

}  // namespace

static int max_cells_for(const gs_index* ix) {
    const size_t budget = 200 * 1024;   // shared memory for accumulators + head weights
    return (int)(budget / ((size_t)ix->Ts * 4 + GS_HEAD_MAX * 4));
}
int gs_score_term_group(const gs_index* ix, int64_t nq, int group) {
    int G = group > 0 ? group : (int)std::min<int64_t>(nq, 1 << 20);
    return (int)std::max<int64_t>(1, std::min<int64_t>(std::min<int64_t>(G, nq), max_cells_for(ix)));
}

gs_status_t gs_launch_score_term(const gs_index* ix, const gs_qbatch& qb, int64_t q0, int64_t nq, int group,
                                 bool use_head, const gs_tileset& ts, const gs_sink& sink, cudaStream_t s) {
    if (nq <= 0 || ts.count <= 0) return GS_OK;
    const bool head = use_head && ix->H > 0;
    // cells per CTA: bounded by shared memory (accumulators + head weights)
    const int max_cells = max_cells_for(ix);
    if (max_cells < 1) return GS_ERR_OOM;
    const int G = gs_score_term_group(ix, nq, group);
    int m = std::max(1, std::min(max_cells / G, kWarps / std::min(G, kWarps)));
    m = std::min(m, ts.count);
    TermParams p{};
    p.inv_off = ix->inv_off; p.inv_doc = ix->inv_doc; p.inv_w = ix->inv_w; p.seg = ix->seg;
    p.head_strip = ix->head_strip; p.H = head ? ix->H : 0; p.N = ix->N; p.N_pad = ix->N_pad; p.Ts = ix->Ts;
    p.ntiles = ix->ntiles;
    p.q_indptr = qb.indptr; p.head_w = qb.head_w; p.tail_term = qb.tail_term; p.tail_w = qb.tail_w;
    p.tail_cnt = qb.tail_cnt;
    p.q0 = q0; p.nq = (int32_t)nq; p.G = G; p.n_qgroups = (int)((nq + G - 1) / G);
    p.ts = ts; p.m = m; p.sink = sink;
    const int n_tgroups = (ts.count + m - 1) / m;
    const int64_t grid = (int64_t)p.n_qgroups * n_tgroups;
    if (grid > 0x7FFFFFFFLL) return GS_ERR_OUT_OF_RANGE;
    const size_t smem = (size_t)G * m * ix->Ts * 4 + (head ? (size_t)G * GS_HEAD_MAX * 4 : 0);
    if (ix->wtype == GS_W_F32)
        return head ? launch<GS_W_F32, true>(p, (unsigned)grid, smem, s) : launch<GS_W_F32, false>(p, (unsigned)grid, smem, s);
    return head ? launch<GS_W_U8, true>(p, (unsigned)grid, smem, s) : launch<GS_W_U8, false>(p, (unsigned)grid, smem, s);
}
