// score_doc.cu — S2b: document-parallel CSR kernel (kernel K2').
//
// PAPER.md L174 §5.3: "an alternative document-parallel kernel using a CSR index by document.  Each
// program handles one (query, document) pair, iterating over the document's term list and looking up
// query weights from a dense query matrix ... eliminates all atomic operations (each program
// exclusively owns its output cell)".  The paper's kernel re-reads the forward index for every
// query (76.3 GB per 500-query batch at 100K docs, Table 7).
//
// Here the forward index is streamed ONCE per tile of QT queries.  A warp owns one document at a
// time: its lanes read 32 consecutive postings of the row (coalesced), translate each term id
// through a shared-memory slot table (term -> compact row of the transposed query tile, 0 = term
// not in any query of the tile) and accumulate QT partial scores in registers; a transposed
// butterfly reduction leaves score (doc, query j) in one lane, which owns that output cell — zero
// atomics.  The query tile (slot table + compact [rows][QT] weight matrix, transposed so one row
// is contiguous) is built once per pass by k_build_qtile and staged into shared memory.
#include <algorithm>

#include "gs_internal.cuh"

namespace {

constexpr int kThreads = 1024;
constexpr int kWarps = kThreads / 32;
constexpr int kRowPad = 4;    // row stride QT+4 words: 16-byte aligned and spread over the banks

struct QTileHdr { uint32_t R; uint32_t pad[3]; };

__host__ __device__ inline size_t slot_bytes(int32_t V) { return ((size_t)V * 2 + 15) / 16 * 16; }

// ---- build the transposed query tile of pass `blockIdx.x`
template <int WT>
__global__ void __launch_bounds__(1024) k_build_qtile(const int64_t* __restrict__ indptr, const int32_t* __restrict__ terms,
                                                      const void* __restrict__ weights, int64_t q0, int64_t nq, int QT,
                                                      int32_t V, unsigned char* __restrict__ scratch, size_t tile_bytes,
                                                      int64_t rows_cap) {
    extern __shared__ uint32_t map[];                 // [V]
    __shared__ uint32_t warp_tot[32];
    const int pass = blockIdx.x;
    const int64_t qa = q0 + (int64_t)pass * QT;
    const int nqt = (int)min((int64_t)QT, q0 + nq - qa);
    unsigned char* base = scratch + (size_t)pass * tile_bytes;
    QTileHdr* hdr = reinterpret_cast<QTileHdr*>(base);
    uint16_t* slot = reinterpret_cast<uint16_t*>(base + sizeof(QTileHdr));
    uint32_t* rows = reinterpret_cast<uint32_t*>(base + sizeof(QTileHdr) + slot_bytes(V));
    const int QTP = QT + kRowPad;

    for (int t = threadIdx.x; t < V; t += blockDim.x) map[t] = 0;
    __syncthreads();
    const int64_t ea = indptr[qa], eb = indptr[qa + nqt];
    for (int64_t i = ea + threadIdx.x; i < eb; i += blockDim.x) {
        const int32_t t = terms[i];
        if (t >= 0 && t < V) map[t] = 1;
    }
    __syncthreads();
    // exclusive scan over map in chunks of `per` consecutive terms per thread
    const int per = (V + blockDim.x - 1) / blockDim.x;
    const int t0 = threadIdx.x * per, t1 = min(V, t0 + per);
    uint32_t local = 0;
    for (int t = t0; t < t1; ++t) local += map[t];
    uint32_t incl = local;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    for (int o = 1; o < 32; o <<= 1) {
        uint32_t v = __shfl_up_sync(0xFFFFFFFFu, incl, o);
        if (lane >= o) incl += v;
    }
    if (lane == 31) warp_tot[warp] = incl;
    __syncthreads();
    if (warp == 0) {
        uint32_t v = warp_tot[lane], inc2 = v;
        for (int o = 1; o < 32; o <<= 1) {
            uint32_t u = __shfl_up_sync(0xFFFFFFFFu, inc2, o);
            if (lane >= o) inc2 += u;
        }
        warp_tot[lane] = inc2 - v;   // exclusive
        if (lane == 31) hdr->R = min((uint32_t)inc2, (uint32_t)rows_cap - 1);
    }
    __syncthreads();
    uint32_t run = warp_tot[warp] + incl - local;     // rows before this thread's chunk
    for (int t = t0; t < t1; ++t) {
        uint32_t r = 0;
        if (map[t]) r = ++run;
        slot[t] = (uint16_t)r;
        map[t] = r;
    }
    __syncthreads();
    const uint32_t R = hdr->R;
    for (size_t i = threadIdx.x; i < (size_t)(R + 1) * QTP; i += blockDim.x) rows[i] = 0u;
    __syncthreads();
    for (int j = 0; j < nqt; ++j) {
        const int64_t a = indptr[qa + j], e = indptr[qa + j + 1];
        for (int64_t i = a + threadIdx.x; i < e; i += blockDim.x) {
            const int32_t t = terms[i];
            if (t < 0 || t >= V) continue;
            uint32_t w;
            if (WT == GS_W_F32) w = __float_as_uint(((const float*)weights)[i]);
            else w = (uint32_t)((const uint8_t*)weights)[i];
            rows[(size_t)map[t] * QTP + j] = w;
        }
    }
}

template <int WT> struct NumD;
template <> struct NumD<GS_W_F32> {
    using W = float; using A = float;
    static __device__ __forceinline__ A mac(A acc, A q, W w) { return fmaf(q, w, acc); }
    static __device__ __forceinline__ uint32_t bits(A a) { return __float_as_uint(a); }
};
template <> struct NumD<GS_W_U8> {
    using W = uint8_t; using A = int32_t;
    static __device__ __forceinline__ A mac(A acc, A q, W w) { return acc + q * (int32_t)w; }
    static __device__ __forceinline__ uint32_t bits(A a) { return (uint32_t)a; }
};

struct DocParams {
    const int64_t* fwd_indptr; const int32_t* fwd_terms; const void* fwd_w;
    int64_t N; int32_t V; int32_t Ts;
    const unsigned char* scratch; size_t tile_bytes; int64_t rows_cap_smem;
    int64_t q0; int32_t nq; int32_t n_passes;   // queries [q0, q0+nq) in n_passes tiles of QT
    gs_tileset ts;
    gs_sink sink;
    int32_t ctas_per_pass;
};

template <int WT, int QT>
__global__ void __launch_bounds__(kThreads, 1) k_score_doc(const DocParams p) {
    using W = typename NumD<WT>::W;
    using A = typename NumD<WT>::A;
    constexpr int QTP = QT + kRowPad;
    extern __shared__ __align__(16) unsigned char smem[];
    uint16_t* s_slot = reinterpret_cast<uint16_t*>(smem);
    A* s_rows = reinterpret_cast<A*>(smem + slot_bytes(p.V));
    const int pass = blockIdx.x / p.ctas_per_pass;
    const int cta = blockIdx.x % p.ctas_per_pass;
    const unsigned char* base = p.scratch + (size_t)pass * p.tile_bytes;
    const uint32_t R = reinterpret_cast<const QTileHdr*>(base)->R;
    const uint16_t* g_slot = reinterpret_cast<const uint16_t*>(base + sizeof(QTileHdr));
    const A* g_rows = reinterpret_cast<const A*>(base + sizeof(QTileHdr) + slot_bytes(p.V));
    const bool rows_in_smem = (int64_t)(R + 1) <= p.rows_cap_smem;

    {   // stage the query tile: 16-byte copies
        const uint4* src = reinterpret_cast<const uint4*>(g_slot);
        uint4* dst = reinterpret_cast<uint4*>(s_slot);
        for (size_t i = threadIdx.x; i < slot_bytes(p.V) / 16; i += kThreads) dst[i] = src[i];
        if (rows_in_smem) {
            const uint4* rs = reinterpret_cast<const uint4*>(g_rows);
            uint4* rd = reinterpret_cast<uint4*>(s_rows);
            for (size_t i = threadIdx.x; i < (size_t)(R + 1) * QTP / 4; i += kThreads) rd[i] = rs[i];
        }
    }
    __syncthreads();
    const A* rows = rows_in_smem ? s_rows : g_rows;

    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int64_t qa = p.q0 + (int64_t)pass * QT;
    const int nqt = (int)min((int64_t)QT, p.q0 + p.nq - qa);
    const W* __restrict__ fw = reinterpret_cast<const W*>(p.fwd_w);
    constexpr int SH = QT == 32 ? 0 : (QT == 16 ? 1 : (QT == 8 ? 2 : (QT == 4 ? 3 : (QT == 2 ? 4 : 5))));
    const int myq = lane >> SH;               // query (within the tile) whose total ends up in this lane
    const bool owner = (lane & ((1 << SH) - 1)) == 0 && myq < nqt;

    // warps of all CTAs of this pass stride over the docs of the tile set
    const int64_t docs_in_set = (int64_t)p.ts.count * p.Ts;
    for (int64_t c = (int64_t)cta * kWarps + warp; c < docs_in_set; c += (int64_t)p.ctas_per_pass * kWarps) {
        const int64_t tile = p.ts.first + (c / p.Ts) * p.ts.stride;
        const int64_t doc = tile * p.Ts + (c % p.Ts);
        if (doc >= p.N) continue;
        const int64_t a = p.fwd_indptr[doc], e = p.fwd_indptr[doc + 1];
        A acc[QT];
#pragma unroll
        for (int j = 0; j < QT; ++j) acc[j] = A(0);
        for (int64_t i = a + lane; i < e; i += 32) {
            const int32_t t = p.fwd_terms[i];
            const uint32_t r = s_slot[t];
            if (r != 0) {
                const W w = fw[i];
                const A* row = rows + (size_t)r * QTP;
#pragma unroll
                for (int j = 0; j < QT; j += 4) {
                    const int4 v = *reinterpret_cast<const int4*>(row + j);
                    if (WT == GS_W_F32) {
                        acc[j + 0] = NumD<WT>::mac(acc[j + 0], (A)__int_as_float(v.x), w);
                        acc[j + 1] = NumD<WT>::mac(acc[j + 1], (A)__int_as_float(v.y), w);
                        acc[j + 2] = NumD<WT>::mac(acc[j + 2], (A)__int_as_float(v.z), w);
                        acc[j + 3] = NumD<WT>::mac(acc[j + 3], (A)__int_as_float(v.w), w);
                    } else {
                        acc[j + 0] = NumD<WT>::mac(acc[j + 0], (A)v.x, w);
                        acc[j + 1] = NumD<WT>::mac(acc[j + 1], (A)v.y, w);
                        acc[j + 2] = NumD<WT>::mac(acc[j + 2], (A)v.z, w);
                        acc[j + 3] = NumD<WT>::mac(acc[j + 3], (A)v.w, w);
                    }
                }
            }
        }
        // transposed butterfly: halve the register set at each step until one value per lane group
        int n = QT;
#pragma unroll
        for (int step = 16; step >= 1; step >>= 1) {
            if (n > 1) {
                n >>= 1;
                const bool upper = (lane & step) != 0;
#pragma unroll
                for (int j = 0; j < QT / 2; ++j) {
                    if (j < n) {
                        const A send = upper ? acc[j] : acc[j + n];
                        const A keep = upper ? acc[j + n] : acc[j];
                        acc[j] = keep + __shfl_xor_sync(0xFFFFFFFFu, send, step);
                    }
                }
            } else {
                acc[0] += __shfl_xor_sync(0xFFFFFFFFu, acc[0], step);
            }
        }
        if (owner) {
            const int64_t b = qa + myq;
            const uint32_t bits = NumD<WT>::bits(acc[0]);
            if (p.sink.thr == nullptr) {
                p.sink.dense[(b - p.q0) * p.sink.ld + c] = bits;
            } else {
                const uint64_t key = gs_make_key(gs_ord_bits<WT>(bits), (uint32_t)doc);
                if (key >= p.sink.thr[b]) {
                    const uint32_t pos = atomicAdd(&p.sink.cand_cnt[b], 1u);
                    if ((int64_t)pos < p.sink.cand_cap) p.sink.cand[b * p.sink.cand_cap + pos] = key;
                }
            }
        }
    }
}

size_t tile_bytes_for(const gs_index* ix, int QT, int64_t rows_cap) {
    size_t b = sizeof(QTileHdr) + slot_bytes(ix->V) + (size_t)rows_cap * (QT + kRowPad) * 4;
    return (b + 255) / 256 * 256;
}
int norm_qt(int qtile) {
    if (qtile <= 0) return 16;
    int q = 2;
    while (q < qtile && q < 32) q <<= 1;
    return q < 4 ? 4 : q;
}

template <int WT, int QT>
gs_status_t launch_doc(const DocParams& p, unsigned grid, size_t smem, cudaStream_t s) {
    GS_CUDA(cudaFuncSetAttribute(k_score_doc<WT, QT>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    {
        GsProfScope ps(GS_K_SCORE_DOC, s);
        k_score_doc<WT, QT><<<grid, kThreads, smem, s>>>(p);
    }
    ++gs_tls_launches;
    GS_CUDA(cudaGetLastError());
    return GS_OK;
}
template <int WT>
gs_status_t launch_doc_qt(int QT, const DocParams& p, unsigned grid, size_t smem, cudaStream_t s) {
    switch (QT) {
        case 4: return launch_doc<WT, 4>(p, grid, smem, s);
        case 8: return launch_doc<WT, 8>(p, grid, smem, s);
        case 16: return launch_doc<WT, 16>(p, grid, smem, s);
        default: return launch_doc<WT, 32>(p, grid, smem, s);
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
    int dev = 0, sms = 0, smem_max = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    cudaDeviceGetAttribute(&smem_max, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
    {   // build all query tiles of this chunk in one launch
        const size_t bsm = sizeof(uint32_t) * (size_t)ix->V;
        if (bsm > (size_t)smem_max) return GS_ERR_OUT_OF_RANGE;
        GsProfScope ps(GS_K_QTILE, s);
        if (ix->wtype == GS_W_F32) {
            GS_CUDA(cudaFuncSetAttribute(k_build_qtile<GS_W_F32>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bsm));
            k_build_qtile<GS_W_F32><<<n_passes, 1024, bsm, s>>>(q->indptr, q->term_ids, q->weights, q0, nq, QT, ix->V,
                                                              (unsigned char*)scratch, tb, rows_cap);
        } else {
            GS_CUDA(cudaFuncSetAttribute(k_build_qtile<GS_W_U8>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bsm));
            k_build_qtile<GS_W_U8><<<n_passes, 1024, bsm, s>>>(q->indptr, q->term_ids, q->weights, q0, nq, QT, ix->V,
                                                             (unsigned char*)scratch, tb, rows_cap);
        }
        ++gs_tls_launches;
        GS_CUDA(cudaGetLastError());
    }
    const size_t smem = (size_t)smem_max;
    if (slot_bytes(ix->V) + (size_t)(QT + kRowPad) * 4 * 2 > smem) return GS_ERR_OUT_OF_RANGE;
    DocParams p{};
    p.fwd_indptr = ix->fwd_indptr; p.fwd_terms = ix->fwd_terms; p.fwd_w = ix->fwd_w;
    p.N = ix->N; p.V = ix->V; p.Ts = ix->Ts;
    p.scratch = (const unsigned char*)scratch; p.tile_bytes = tb;
    p.rows_cap_smem = (int64_t)((smem - slot_bytes(ix->V)) / ((size_t)(QT + kRowPad) * 4));
    p.q0 = q0; p.nq = (int32_t)nq; p.n_passes = n_passes;
    p.ts = ts; p.sink = sink;
    const int64_t docs_in_set = (int64_t)ts.count * ix->Ts;
    p.ctas_per_pass = (int)std::max<int64_t>(1, std::min<int64_t>(sms, (docs_in_set + kWarps - 1) / kWarps));
    const unsigned grid = (unsigned)(p.ctas_per_pass * n_passes);
    return ix->wtype == GS_W_F32 ? launch_doc_qt<GS_W_F32>(QT, p, grid, smem, s)
                                 : launch_doc_qt<GS_W_U8>(QT, p, grid, smem, s);
}
