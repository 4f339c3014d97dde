// score_doc.cu — S2b: document-parallel forward-index kernel (kernel K2').
//
// PAPER.md L174 §5.3: "an alternative document-parallel kernel using a CSR index by document.  Each
// program handles one (query, document) pair, iterating over the document's term list and looking up
// query weights from a dense query matrix ... eliminates all atomic operations (each program
// exclusively owns its output cell)".  The paper's kernel re-reads the forward index for every
// query (76.3 GB per 500-query batch at 100K docs, Table 7) and names inner-loop
// instruction overhead as what keeps it at 62.6 % of peak (L179).
//
// Here the forward index is streamed ONCE per tile of QT queries, and it is a hybrid:
//   * the H densest posting lists are dense strips [H][N_pad] (0 = term absent).  For them there is
//     nothing to look up: a thread owns one document, keeps QT accumulators in registers and does
//     x[h][doc] * Q[h][q] with Q broadcast from shared memory — a small dense contraction that carries
//     ~85 % of the multiply-adds of the synthetic MS MARCO stand-in at 1 instruction per 32 of them;
//   * every other posting sits in a "tail" CSR.  A warp reads 32 consecutive postings of a document
//     (coalesced), tests each term against a V-bit bitmap of the tile's tail terms (shared memory),
//     compacts the hits — (row of the transposed query tile, doc weight) — into a small per-warp
//     queue, and then walks the queue with lane = query: one broadcast LDS for the hit, one
//     conflict-free LDS for the 32 query weights of that row, one FMA.  No divergence (the hit test
//     is resolved by the ballot), no shuffles in the inner loop.
// The tail sums pass to the owning thread through a per-warp transposition buffer; each (query, doc)
// cell is produced by exactly one thread in a fixed order — zero atomics, deterministic.
// The query tile (bitmap + popcount prefix = term -> row, compact [rows][QT] weight matrix, head
// weights [H'][QT]) is built once per pass by k_build_qtile and staged into shared memory.
#include <algorithm>

#include "gs_internal.cuh"

namespace {

struct QTileHdr { uint32_t R; uint32_t nh; uint32_t pad[2]; uint32_t hl[GS_STRIP_MAX]; };

__host__ __device__ inline int bm_words(int32_t V) { return ((V + 31) / 32 + 3) / 4 * 4; }
// per-pass scratch: hdr | bitmap[Wd] | prefix[Wd] | Qh[GS_STRIP_MAX][QT] | rows[rows_cap][QT]
__host__ __device__ inline size_t off_bm() { return sizeof(QTileHdr); }
__host__ __device__ inline size_t off_pre(int Wd) { return off_bm() + (size_t)Wd * 4; }
__host__ __device__ inline size_t off_qh(int Wd) { return off_pre(Wd) + (size_t)Wd * 4; }
__host__ __device__ inline size_t off_rows(int Wd, int QT) { return off_qh(Wd) + (size_t)GS_STRIP_MAX * QT * 4; }

// ---- build the transposed query tile of pass `blockIdx.x`
template <int WT>
__global__ void __launch_bounds__(1024) k_build_qtile(const int64_t* __restrict__ indptr, const int32_t* __restrict__ terms,
                                                      const void* __restrict__ weights, const int16_t* __restrict__ head_slot,
                                                      int H, int64_t q0, int64_t nq, int QT, int32_t V, int Wd,
                                                      unsigned char* __restrict__ scratch, size_t tile_bytes,
                                                      int64_t rows_cap) {
    extern __shared__ uint32_t sm[];                  // bitmap[Wd], prefix[Wd]
    __shared__ uint32_t warp_tot[32];
    __shared__ uint32_t s_hmask[2];
    uint32_t* bm = sm;
    uint32_t* pre = sm + Wd;
    const int pass = blockIdx.x;
    const int64_t qa = q0 + (int64_t)pass * QT;
    const int nqt = (int)min((int64_t)QT, q0 + nq - qa);
    unsigned char* base = scratch + (size_t)pass * tile_bytes;
    QTileHdr* hdr = reinterpret_cast<QTileHdr*>(base);
    uint32_t* g_bm = reinterpret_cast<uint32_t*>(base + off_bm());
    uint32_t* g_pre = reinterpret_cast<uint32_t*>(base + off_pre(Wd));
    uint32_t* g_qh = reinterpret_cast<uint32_t*>(base + off_qh(Wd));
    uint32_t* g_rows = reinterpret_cast<uint32_t*>(base + off_rows(Wd, QT));

    for (int i = threadIdx.x; i < Wd; i += blockDim.x) bm[i] = 0;
    if (threadIdx.x < 2) s_hmask[threadIdx.x] = 0;
    __syncthreads();
    const int64_t ea = indptr[qa], eb = indptr[qa + nqt];
    for (int64_t i = ea + threadIdx.x; i < eb; i += blockDim.x) {
        const int32_t t = terms[i];
        if (t < 0 || t >= V) continue;
        const int hs = H > 0 ? (int)head_slot[t] : -1;
        if (hs >= 0) atomicOr(&s_hmask[hs >> 5], 1u << (hs & 31));
        else atomicOr(&bm[t >> 5], 1u << (t & 31));
    }
    __syncthreads();
    // exclusive scan of popc(bitmap word) in chunks of `per` consecutive words per thread
    const int per = (Wd + blockDim.x - 1) / blockDim.x;
    const int w0 = min(Wd, (int)threadIdx.x * per), w1 = min(Wd, w0 + per);
    uint32_t local = 0;
    for (int w = w0; w < w1; ++w) local += __popc(bm[w]);
    uint32_t incl = local;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    for (int o = 1; o < 32; o <<= 1) {
        const uint32_t v = __shfl_up_sync(0xFFFFFFFFu, incl, o);
        if (lane >= o) incl += v;
    }
    if (lane == 31) warp_tot[warp] = incl;
    __syncthreads();
    if (warp == 0) {
        const uint32_t v = warp_tot[lane];
        uint32_t inc2 = v;
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t u = __shfl_up_sync(0xFFFFFFFFu, inc2, o);
            if (lane >= o) inc2 += u;
        }
        warp_tot[lane] = inc2 - v;   // exclusive
        if (lane == 31) hdr->R = min((uint32_t)inc2, (uint32_t)rows_cap - 1);
    }
    __syncthreads();
    uint32_t run = warp_tot[warp] + incl - local;     // rows before this thread's chunk
    for (int w = w0; w < w1; ++w) {
        pre[w] = run;
        run += __popc(bm[w]);
    }
    if (threadIdx.x == 0) {   // compact list of the strips some query of the tile uses, padded to a multiple of 4
        uint32_t n = 0;
        for (int h = 0; h < H; ++h)
            if ((s_hmask[h >> 5] >> (h & 31)) & 1u) hdr->hl[n++] = (uint32_t)h;
        hdr->nh = n;
        while (n & 3u) hdr->hl[n++] = 0u;           // padding rows carry zero weights
    }
    __syncthreads();
    for (int i = threadIdx.x; i < Wd; i += blockDim.x) { g_bm[i] = bm[i]; g_pre[i] = pre[i]; }
    const uint32_t R = hdr->R;
    for (size_t i = threadIdx.x; i < (size_t)(R + 1) * QT; i += blockDim.x) g_rows[i] = 0u;
    for (int i = threadIdx.x; i < GS_STRIP_MAX * QT; i += blockDim.x) g_qh[i] = 0u;
    __syncthreads();
    for (int j = 0; j < nqt; ++j) {
        const int64_t a = indptr[qa + j], e = indptr[qa + j + 1];
        for (int64_t i = a + threadIdx.x; i < e; i += blockDim.x) {
            const int32_t t = terms[i];
            if (t < 0 || t >= V) continue;
            uint32_t w;
            if (WT == GS_W_F32) w = __float_as_uint(((const float*)weights)[i]);
            else w = (uint32_t)((const uint8_t*)weights)[i];
            const int hs = H > 0 ? (int)head_slot[t] : -1;
            if (hs >= 0) {
                const uint32_t below = hs < 32 ? (s_hmask[0] & ((1u << hs) - 1u))
                                               : (s_hmask[1] & ((1u << (hs - 32)) - 1u));
                const int ci = __popc(below) + (hs >= 32 ? __popc(s_hmask[0]) : 0);
                g_qh[(size_t)ci * QT + j] = w;
            } else {
                const uint32_t word = bm[t >> 5];
                const uint32_t r = pre[t >> 5] + __popc(word & ((1u << (t & 31)) - 1u)) + 1u;
                if (r <= R) g_rows[(size_t)r * QT + j] = w;
            }
        }
    }
}

template <int WT> struct NumD;
template <> struct NumD<GS_W_F32> {
    using W = float; using A = float;
    static __device__ __forceinline__ A mac(A acc, A q, A w) { return fmaf(q, w, acc); }
    static __device__ __forceinline__ A widen(W w) { return w; }
    static __device__ __forceinline__ A from_bits(uint32_t b) { return __uint_as_float(b); }
    static __device__ __forceinline__ uint32_t bits(A a) { return __float_as_uint(a); }
    static __device__ __forceinline__ A thr_score(uint32_t ord) { return __uint_as_float(gs_unord_f32(ord)); }  // NaN for 0
};
template <> struct NumD<GS_W_U8> {
    using W = uint8_t; using A = int32_t;
    static __device__ __forceinline__ A mac(A acc, A q, A w) { return acc + q * w; }
    static __device__ __forceinline__ A widen(W w) { return (int32_t)w; }
    static __device__ __forceinline__ A from_bits(uint32_t b) { return (int32_t)b; }
    static __device__ __forceinline__ uint32_t bits(A a) { return (uint32_t)a; }
    static __device__ __forceinline__ A thr_score(uint32_t ord) { return (int32_t)(ord ^ 0x80000000u); }
};

struct DocParams {
    const int64_t* fwd_indptr; const int32_t* fwd_terms; const void* fwd_w;
    const void* strips; int64_t N_pad;
    int64_t N; int32_t V; int32_t Ts; int32_t Wd;
    const unsigned char* scratch; size_t tile_bytes; int32_t rows_cap_smem;
    int64_t q0; int32_t nq;                     // queries [q0, q0+nq) in tiles of QT
    gs_tileset ts;
    gs_sink sink;
    int32_t ctas_per_pass;
};

template <int QT> struct Geo {
    static constexpr int QL = QT < 32 ? QT : 32;       // lanes along the query axis in the hit loop
    static constexpr int DPW = 32 / QL;                // documents walked side by side in the hit loop
    static constexpr int QPL = QT / QL;                // queries per lane
    static constexpr int QCAP = 128 / DPW;             // hit-queue entries per document
    static constexpr int AST = QT + 1;                 // row stride of the transposition buffer (odd: conflict-free)
    static constexpr int NW = QT <= 16 ? 32 : (QT == 32 ? 24 : 16);   // warps per CTA
    static constexpr size_t per_warp = 128 * 8 + (size_t)32 * AST * 4;
    static __host__ __device__ size_t fixed(int Wd) {
        return (size_t)Wd * 8 + (size_t)GS_STRIP_MAX * QT * 4 + (size_t)QT * 8 + (size_t)QT * 4 + GS_STRIP_MAX * 4;
    }
};

template <int WT, int QT>
__global__ void __launch_bounds__(Geo<QT>::NW * 32, 1) k_score_doc(const DocParams p) {
    using W = typename NumD<WT>::W;
    using A = typename NumD<WT>::A;
    using G = Geo<QT>;
    constexpr int QL = G::QL, DPW = G::DPW, QPL = G::QPL, QCAP = G::QCAP, AST = G::AST, NW = G::NW;
    extern __shared__ __align__(16) unsigned char smem[];
    const int Wd = p.Wd;
    // carve: rows first (16-byte aligned), then the fixed part, then the per-warp part
    const int pass = blockIdx.x / p.ctas_per_pass;
    const int cta = blockIdx.x % p.ctas_per_pass;
    const unsigned char* base = p.scratch + (size_t)pass * p.tile_bytes;
    const QTileHdr* hdr = reinterpret_cast<const QTileHdr*>(base);
    const uint32_t R = hdr->R;
    const int nh = (int)hdr->nh;
    const A* g_rows = reinterpret_cast<const A*>(base + off_rows(Wd, QT));
    const bool rows_in_smem = (int)(R + 1) <= p.rows_cap_smem;

    A* s_qh = reinterpret_cast<A*>(smem);                                         // [GS_STRIP_MAX][QT]
    uint64_t* s_thr = reinterpret_cast<uint64_t*>(s_qh + GS_STRIP_MAX * QT);      // [QT]
    A* s_thr_s = reinterpret_cast<A*>(s_thr + QT);                                // [QT]
    uint32_t* s_hl = reinterpret_cast<uint32_t*>(s_thr_s + QT);                   // [GS_STRIP_MAX]
    uint32_t* s_bm = s_hl + GS_STRIP_MAX;                                         // [Wd]
    uint32_t* s_pre = s_bm + Wd;                                                  // [Wd]
    unsigned char* pw = reinterpret_cast<unsigned char*>(s_pre + Wd);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    uint2* queue = reinterpret_cast<uint2*>(pw + (size_t)warp * G::per_warp);     // [DPW][QCAP]
    A* s_acc = reinterpret_cast<A*>(queue + 128);                                 // [32][AST]
    A* s_rows = reinterpret_cast<A*>(pw + (size_t)NW * G::per_warp);              // [R+1][QT] when it fits

    const int64_t qa = p.q0 + (int64_t)pass * QT;
    const int nqt = (int)min((int64_t)QT, p.q0 + p.nq - qa);
    const bool filter = p.sink.thr != nullptr;
    {   // stage the query tile
        const uint32_t* g_bm = reinterpret_cast<const uint32_t*>(base + off_bm());
        for (int i = threadIdx.x; i < 2 * Wd; i += NW * 32) s_bm[i] = g_bm[i];       // bitmap and prefix are adjacent
        const uint4* qs = reinterpret_cast<const uint4*>(base + off_qh(Wd));
        uint4* qd = reinterpret_cast<uint4*>(s_qh);
        const int nh4 = (nh + 3) & ~3;
        for (int i = threadIdx.x; i < nh4 * QT / 4; i += NW * 32) qd[i] = qs[i];
        for (int i = threadIdx.x; i < GS_STRIP_MAX; i += NW * 32) s_hl[i] = hdr->hl[i];
        for (int i = threadIdx.x; i < QT; i += NW * 32) {
            const uint64_t t = (filter && i < nqt) ? p.sink.thr[qa + i] : 0ull;
            s_thr[i] = t;
            s_thr_s[i] = NumD<WT>::thr_score((uint32_t)(t >> 32));
        }
        if (rows_in_smem) {
            const uint4* rs = reinterpret_cast<const uint4*>(g_rows);
            uint4* rd = reinterpret_cast<uint4*>(s_rows);
            for (size_t i = threadIdx.x; i < (size_t)(R + 1) * QT / 4; i += NW * 32) rd[i] = rs[i];
        }
    }
    __syncthreads();

    const W* __restrict__ fw = reinterpret_cast<const W*>(p.fwd_w);
    const W* __restrict__ strips = reinterpret_cast<const W*>(p.strips);
    const unsigned lt = (1u << lane) - 1u;
    const int ds_of_lane = lane / QL, q_of_lane = lane % QL;
    const uint2* myq = queue + ds_of_lane * QCAP;
    const int subs_per_tile = p.Ts >> 5;
    const int64_t n_subs = (int64_t)p.ts.count * subs_per_tile;

    for (int64_t sb = (int64_t)cta * NW + warp; sb < n_subs; sb += (int64_t)p.ctas_per_pass * NW) {
        const int64_t tile = p.ts.first + (sb / subs_per_tile) * (int64_t)p.ts.stride;
        const int64_t doc0 = tile * p.Ts + (sb % subs_per_tile) * 32;
        if (doc0 >= p.N) continue;
        const int nd = (int)min((int64_t)32, p.N - doc0);
        const int64_t my_a = p.fwd_indptr[min(doc0 + lane, p.N)];
        const int64_t my_e = p.fwd_indptr[min(doc0 + lane + 1, p.N)];

        // ---- tail: bitmap filter -> hit queue -> lane = query accumulation
        for (int g = 0; g * DPW < nd; ++g) {
            A acc[QPL];
#pragma unroll
            for (int u = 0; u < QPL; ++u) acc[u] = A(0);
            int cnt[DPW];
#pragma unroll
            for (int ds = 0; ds < DPW; ++ds) cnt[ds] = 0;

            auto flush = [&]() {
                int mx = 0;
#pragma unroll
                for (int ds = 0; ds < DPW; ++ds) mx = max(mx, cnt[ds]);
                const int mx4 = (mx + 3) & ~3;
#pragma unroll
                for (int ds = 0; ds < DPW; ++ds)
                    for (int j = cnt[ds] + lane; j < mx4; j += 32) queue[ds * QCAP + j] = make_uint2(0u, 0u);
                __syncwarp();
                if (rows_in_smem) {
                    for (int j = 0; j < mx4; j += 4) {
#pragma unroll
                        for (int u = 0; u < 4; ++u) {
                            const uint2 e = myq[j + u];
                            const A w = NumD<WT>::from_bits(e.y);
#pragma unroll
                            for (int v = 0; v < QPL; ++v)
                                acc[v] = NumD<WT>::mac(acc[v], s_rows[e.x * QT + q_of_lane + 32 * v], w);
                        }
                    }
                } else {
                    for (int j = 0; j < mx4; j += 4) {
#pragma unroll
                        for (int u = 0; u < 4; ++u) {
                            const uint2 e = myq[j + u];
                            const A w = NumD<WT>::from_bits(e.y);
#pragma unroll
                            for (int v = 0; v < QPL; ++v)
                                acc[v] = NumD<WT>::mac(acc[v], __ldg(g_rows + (size_t)e.x * QT + q_of_lane + 32 * v), w);
                        }
                    }
                }
                __syncwarp();
#pragma unroll
                for (int ds = 0; ds < DPW; ++ds) cnt[ds] = 0;
            };

#pragma unroll
            for (int ds = 0; ds < DPW; ++ds) {
                const int d = g * DPW + ds;
                int64_t a = __shfl_sync(0xFFFFFFFFu, my_a, d & 31);
                int64_t e = __shfl_sync(0xFFFFFFFFu, my_e, d & 31);
                if (d >= nd) e = a;
                for (int64_t i0 = a; i0 < e; i0 += 32) {
                    const int64_t i = i0 + lane;
                    const bool valid = i < e;
                    const int32_t t = valid ? p.fwd_terms[i] : 0;
                    uint32_t wbits = 0u;
                    if (valid) wbits = NumD<WT>::bits(NumD<WT>::widen(fw[i]));
                    const uint32_t word = s_bm[t >> 5];
                    const bool hit = valid && ((word >> (t & 31)) & 1u);
                    const unsigned m = __ballot_sync(0xFFFFFFFFu, hit);
                    if (m == 0u) continue;
                    if (cnt[ds] + 32 > QCAP) flush();
                    if (hit) {
                        const uint32_t r = s_pre[t >> 5] + __popc(word & ((1u << (t & 31)) - 1u)) + 1u;
                        queue[ds * QCAP + cnt[ds] + __popc(m & lt)] = make_uint2(r, wbits);
                    }
                    cnt[ds] += __popc(m);
                }
            }
            flush();
#pragma unroll
            for (int v = 0; v < QPL; ++v) s_acc[(g * DPW + ds_of_lane) * AST + q_of_lane + 32 * v] = acc[v];
        }
        __syncwarp();

        // ---- head strips: thread = document, QT accumulators in registers
        A acc[QT];
#pragma unroll
        for (int q = 0; q < QT; ++q) acc[q] = s_acc[lane * AST + q];
        const int64_t doc = doc0 + lane;
        const W* sp = strips + doc;
        for (int i = 0; i < nh; i += 4) {
            A x[4];
#pragma unroll
            for (int u = 0; u < 4; ++u) x[u] = NumD<WT>::widen(sp[(size_t)s_hl[i + u] * p.N_pad]);
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const A* qrow = s_qh + (i + u) * QT;
#pragma unroll
                for (int q = 0; q < QT; q += 4) {
                    const int4 v = *reinterpret_cast<const int4*>(qrow + q);
                    acc[q + 0] = NumD<WT>::mac(acc[q + 0], NumD<WT>::from_bits((uint32_t)v.x), x[u]);
                    acc[q + 1] = NumD<WT>::mac(acc[q + 1], NumD<WT>::from_bits((uint32_t)v.y), x[u]);
                    acc[q + 2] = NumD<WT>::mac(acc[q + 2], NumD<WT>::from_bits((uint32_t)v.z), x[u]);
                    acc[q + 3] = NumD<WT>::mac(acc[q + 3], NumD<WT>::from_bits((uint32_t)v.w), x[u]);
                }
            }
        }

        // ---- sink: this thread owns the cells (qa + q, doc)
        if (doc < p.N) {
            if (!filter) {
                uint32_t* out = p.sink.dense + (qa - p.q0) * p.sink.ld + sb * 32 + lane;
#pragma unroll
                for (int q = 0; q < QT; ++q)
                    if (q < nqt) out[(int64_t)q * p.sink.ld] = NumD<WT>::bits(acc[q]);
            } else {
#pragma unroll
                for (int q = 0; q < QT; ++q) {
                    if (q < nqt && !(acc[q] < s_thr_s[q])) {
                        const uint64_t key = gs_make_key(gs_ord_bits<WT>(NumD<WT>::bits(acc[q])), (uint32_t)doc);
                        if (key >= s_thr[q]) {
                            const int64_t b = qa + q;
                            const uint32_t pos = atomicAdd(&p.sink.cand_cnt[b], 1u);
                            if ((int64_t)pos < p.sink.cand_cap) p.sink.cand[b * p.sink.cand_cap + pos] = key;
                        }
                    }
                }
            }
        }
        __syncwarp();
    }
}

size_t tile_bytes_for(const gs_index* ix, int QT, int64_t rows_cap) {
    size_t b = off_rows(bm_words(ix->V), QT) + (size_t)rows_cap * QT * 4;
    return (b + 255) / 256 * 256;
}
int norm_qt(int qtile) {
    if (qtile <= 0) return 32;
    int q = 8;
    while (q < qtile && q < 64) q <<= 1;
    return q;
}

template <int WT, int QT>
gs_status_t launch_doc(DocParams p, const gs_index* ix, int64_t n_subs, int n_passes, int sms, int smem_max, cudaStream_t s) {
    using G = Geo<QT>;
    const size_t fixed = G::fixed(p.Wd) + (size_t)G::NW * G::per_warp;
    if (fixed + (size_t)QT * 4 * 2 > (size_t)smem_max) return GS_ERR_OUT_OF_RANGE;     // vocabulary too large for the bitmap
    const size_t smem = (size_t)smem_max;
    p.rows_cap_smem = (int32_t)std::min<size_t>((smem - fixed) / ((size_t)QT * 4), 0x7FFFFFFF);
    p.ctas_per_pass = (int)std::max<int64_t>(1, std::min<int64_t>(sms, (n_subs + G::NW - 1) / G::NW));
    const unsigned grid = (unsigned)(p.ctas_per_pass * n_passes);
    GS_CUDA(cudaFuncSetAttribute(k_score_doc<WT, QT>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    {
        GsProfScope ps(GS_K_SCORE_DOC, s);
        k_score_doc<WT, QT><<<grid, G::NW * 32, smem, s>>>(p);
    }
    ++gs_tls_launches;
    GS_CUDA(cudaGetLastError());
    (void)ix;
    return GS_OK;
}
template <int WT>
gs_status_t launch_doc_qt(int QT, const DocParams& p, const gs_index* ix, int64_t n_subs, int n_passes, int sms,
                          int smem_max, cudaStream_t s) {
    switch (QT) {
        case 8: return launch_doc<WT, 8>(p, ix, n_subs, n_passes, sms, smem_max, s);
        case 16: return launch_doc<WT, 16>(p, ix, n_subs, n_passes, sms, smem_max, s);
        case 32: return launch_doc<WT, 32>(p, ix, n_subs, n_passes, sms, smem_max, s);
        default: return launch_doc<WT, 64>(p, ix, n_subs, n_passes, sms, smem_max, s);
    }
}

}  // namespace

// rows capacity of one scratch tile: every distinct term of the batch could fall in one tile
static int64_t rows_cap_for(const gs_index* ix, int64_t q_nnz) { return std::min<int64_t>(ix->V, q_nnz) + 1; }

int gs_score_doc_qtile(int qtile) { return norm_qt(qtile); }

size_t gs_score_doc_scratch_bytes_ex(const gs_index* ix, int qtile, int64_t nq, int64_t q_nnz) {
    const int QT = norm_qt(qtile);
    const int64_t passes = (nq + QT - 1) / QT;
    return tile_bytes_for(ix, QT, rows_cap_for(ix, q_nnz)) * (size_t)std::max<int64_t>(passes, 1);
}

gs_status_t gs_launch_score_doc(const gs_index* ix, const gs_csr_t* q, const gs_qbatch& qb, int64_t q0, int64_t nq,
                                int qtile, const gs_tileset& ts, const gs_sink& sink, void* scratch, cudaStream_t s) {
    (void)qb;
    if (nq <= 0 || ts.count <= 0) return GS_OK;
    const int QT = norm_qt(qtile);
    const int n_passes = (int)((nq + QT - 1) / QT);
    const int64_t rows_cap = rows_cap_for(ix, q->nnz);
    const size_t tb = tile_bytes_for(ix, QT, rows_cap);
    const int Wd = bm_words(ix->V);
    int dev = 0, sms = 0, smem_max = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    cudaDeviceGetAttribute(&smem_max, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
    {   // build all query tiles of this chunk in one launch
        const size_t bsm = sizeof(uint32_t) * 2 * (size_t)Wd;
        if (bsm > (size_t)smem_max) return GS_ERR_OUT_OF_RANGE;
        GsProfScope ps(GS_K_QTILE, s);
        if (ix->wtype == GS_W_F32) {
            GS_CUDA(cudaFuncSetAttribute(k_build_qtile<GS_W_F32>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bsm));
            k_build_qtile<GS_W_F32><<<n_passes, 1024, bsm, s>>>(q->indptr, q->term_ids, q->weights, ix->head_slot, ix->H, q0, nq,
                                                              QT, ix->V, Wd, (unsigned char*)scratch, tb, rows_cap);
        } else {
            GS_CUDA(cudaFuncSetAttribute(k_build_qtile<GS_W_U8>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bsm));
            k_build_qtile<GS_W_U8><<<n_passes, 1024, bsm, s>>>(q->indptr, q->term_ids, q->weights, ix->head_slot, ix->H, q0, nq,
                                                             QT, ix->V, Wd, (unsigned char*)scratch, tb, rows_cap);
        }
        ++gs_tls_launches;
        GS_CUDA(cudaGetLastError());
    }
    DocParams p{};
    p.fwd_indptr = ix->fwd_indptr; p.fwd_terms = ix->fwd_terms; p.fwd_w = ix->fwd_w;
    p.strips = ix->head_strip; p.N_pad = ix->N_pad;
    p.N = ix->N; p.V = ix->V; p.Ts = ix->Ts; p.Wd = Wd;
    p.scratch = (const unsigned char*)scratch; p.tile_bytes = tb;
    p.q0 = q0; p.nq = (int32_t)nq;
    p.ts = ts; p.sink = sink;
    const int64_t n_subs = (int64_t)ts.count * (ix->Ts / 32);
    return ix->wtype == GS_W_F32 ? launch_doc_qt<GS_W_F32>(QT, p, ix, n_subs, n_passes, sms, smem_max, s)
                                 : launch_doc_qt<GS_W_U8>(QT, p, ix, n_subs, n_passes, sms, smem_max, s);
}
