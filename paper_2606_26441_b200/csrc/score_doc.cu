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
//   * every other posting sits in a "tail" CSR whose term word also carries the document's position
//     in its aligned block of 32 documents.  A warp owns such a block and streams its postings as ONE
//     flat range (coalesced, 8 independent loads in flight, next chunk prefetched), tests each term
//     against a V-bit bitmap of the tile's tail terms (shared memory) and compacts the hits, in
//     stream order, into a per-warp queue.  Then lane d walks the hits of document d (they are
//     contiguous in the queue: a binary search finds them): term -> row through a popcount prefix,
//     row -> its (query, weight) pairs in a small CSR, accumulate into the lane's own row of a
//     [32][QT+1] shared-memory tile (odd stride: no two lanes share a bank by construction of the
//     row, no atomics, fixed order).
// Each (query, doc) cell is produced by exactly one thread in a fixed order — zero atomics,
// deterministic.  The query tile (bitmap + popcount prefix, row CSR, head weights [H'][QT]) is built
// once per pass by k_build_qtile and staged into shared memory.
#include <algorithm>

#include "gs_internal.cuh"

namespace {

constexpr uint32_t kTermMask = (1u << GS_FWD_DOC_SHIFT) - 1u;

struct QTileHdr {
    uint32_t R;          // distinct tail terms of the tile (rows)
    uint32_t nh;         // strips some query of the tile uses
    uint32_t np;         // (row, query) pairs
    uint32_t row_off;    // this pass's slice of the shared rowptr array
    uint32_t pair_off;   // ... and of the shared pairs array
    uint32_t pad[3];
    uint32_t hl[GS_STRIP_MAX];
};

__host__ __device__ inline int bm_words(int32_t V) { return ((V + 1 + 31) / 32 + 3) / 4 * 4; }
// per-pass scratch block: hdr | bitmap[Wd] | prefix[Wd] | Qh[GS_STRIP_MAX][QT]
__host__ __device__ inline size_t off_bm() { return sizeof(QTileHdr); }
__host__ __device__ inline size_t off_pre(int Wd) { return off_bm() + (size_t)Wd * 4; }
__host__ __device__ inline size_t off_qh(int Wd) { return off_pre(Wd) + (size_t)Wd * 4; }
__host__ __device__ inline size_t pass_bytes(int Wd, int QT) {
    return (off_qh(Wd) + (size_t)GS_STRIP_MAX * QT * 4 + 255) / 256 * 256;
}
// after the pass blocks: rowptr[nnz + passes + 1] | cursor[nnz + passes + 1] | pairs[nnz] (uint2)
struct SharedScratch { uint32_t* rowptr; uint32_t* cursor; uint2* pairs; };
__host__ __device__ inline SharedScratch shared_scratch(unsigned char* scratch, int Wd, int QT, int64_t passes, int64_t nnz) {
    unsigned char* p = scratch + pass_bytes(Wd, QT) * (size_t)passes;
    const size_t n1 = ((size_t)(nnz + passes + 1) * 4 + 255) / 256 * 256;
    SharedScratch s;
    s.rowptr = reinterpret_cast<uint32_t*>(p);
    s.cursor = reinterpret_cast<uint32_t*>(p + n1);
    s.pairs = reinterpret_cast<uint2*>(p + 2 * n1);
    return s;
}

// block-wide exclusive scan helper: every thread passes the sum of its own chunk, gets the sum of
// all earlier threads' chunks; *total receives the grand total (valid after the call for all threads)
__device__ __forceinline__ uint32_t block_excl_scan(uint32_t local, uint32_t* warp_tot, uint32_t* total) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    uint32_t incl = local;
    for (int o = 1; o < 32; o <<= 1) {
        const uint32_t v = __shfl_up_sync(0xFFFFFFFFu, incl, o);
        if (lane >= o) incl += v;
    }
    __syncthreads();                       // warp_tot may still be read from an earlier call
    if (lane == 31) warp_tot[warp] = incl;
    __syncthreads();
    if (warp == 0) {
        const uint32_t v = lane < (int)(blockDim.x >> 5) ? warp_tot[lane] : 0u;
        uint32_t inc2 = v;
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t u = __shfl_up_sync(0xFFFFFFFFu, inc2, o);
            if (lane >= o) inc2 += u;
        }
        warp_tot[lane] = inc2 - v;
        if (lane == 31) *total = inc2;
    }
    __syncthreads();
    return warp_tot[warp] + incl - local;
}

// ---- build the query tile of pass `blockIdx.x` (one CTA of 1024 threads per pass)
template <int WT>
__global__ void __launch_bounds__(1024) k_build_qtile(const int64_t* __restrict__ indptr, const int32_t* __restrict__ terms,
                                                      const void* __restrict__ weights, const int16_t* __restrict__ head_slot,
                                                      int H, int64_t q0, int64_t nq, int QT, int32_t V, int Wd,
                                                      unsigned char* __restrict__ scratch, int64_t n_passes, int64_t nnz_cap) {
    extern __shared__ uint32_t sm[];                  // bitmap[Wd], prefix[Wd]
    __shared__ uint32_t warp_tot[32];
    __shared__ uint32_t s_hmask[2];
    __shared__ uint32_t s_total;
    uint32_t* bm = sm;
    uint32_t* pre = sm + Wd;
    const int pass = blockIdx.x;
    const int64_t qa = q0 + (int64_t)pass * QT;
    const int nqt = (int)min((int64_t)QT, q0 + nq - qa);
    unsigned char* base = scratch + (size_t)pass * pass_bytes(Wd, QT);
    QTileHdr* hdr = reinterpret_cast<QTileHdr*>(base);
    uint32_t* g_bm = reinterpret_cast<uint32_t*>(base + off_bm());
    uint32_t* g_pre = reinterpret_cast<uint32_t*>(base + off_pre(Wd));
    uint32_t* g_qh = reinterpret_cast<uint32_t*>(base + off_qh(Wd));
    const SharedScratch ss = shared_scratch(scratch, Wd, QT, n_passes, nnz_cap);
    const uint32_t pair_off = (uint32_t)(indptr[qa] - indptr[q0]);
    const uint32_t row_off = pair_off + (uint32_t)pass;
    uint32_t* rowptr = ss.rowptr + row_off;
    uint32_t* cursor = ss.cursor + row_off;
    uint2* pairs = ss.pairs + pair_off;

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
    // term -> row: exclusive scan of popc(bitmap word)
    {
        const int per = (Wd + blockDim.x - 1) / blockDim.x;
        const int w0 = min(Wd, (int)threadIdx.x * per), w1 = min(Wd, w0 + per);
        uint32_t local = 0;
        for (int w = w0; w < w1; ++w) local += __popc(bm[w]);
        uint32_t run = block_excl_scan(local, warp_tot, &s_total);
        for (int w = w0; w < w1; ++w) {
            pre[w] = run;
            run += __popc(bm[w]);
        }
    }
    __syncthreads();
    const uint32_t R = s_total;
    if (threadIdx.x == 0) {   // compact list of the strips some query of the tile uses, padded to a multiple of 4
        uint32_t n = 0;
        for (int h = 0; h < H; ++h)
            if ((s_hmask[h >> 5] >> (h & 31)) & 1u) hdr->hl[n++] = (uint32_t)h;
        hdr->nh = n;
        while (n & 3u) hdr->hl[n++] = 0u;           // padding rows carry zero weights
        hdr->R = R;
        hdr->row_off = row_off;
        hdr->pair_off = pair_off;
    }
    for (int i = threadIdx.x; i < Wd; i += blockDim.x) { g_bm[i] = bm[i]; g_pre[i] = pre[i]; }
    for (int i = threadIdx.x; i < GS_STRIP_MAX * QT; i += blockDim.x) g_qh[i] = 0u;
    for (uint32_t i = threadIdx.x; i <= R; i += blockDim.x) cursor[i] = 0u;
    __syncthreads();
    // pairs per row
    for (int64_t i = ea + threadIdx.x; i < eb; i += blockDim.x) {
        const int32_t t = terms[i];
        if (t < 0 || t >= V) continue;
        if (H > 0 && head_slot[t] >= 0) continue;
        const uint32_t word = bm[t >> 5];
        atomicAdd(&cursor[pre[t >> 5] + __popc(word & ((1u << (t & 31)) - 1u))], 1u);
    }
    __syncthreads();
    {
        const uint32_t per = (R + blockDim.x - 1) / blockDim.x;
        const uint32_t r0 = min(R, threadIdx.x * per), r1 = min(R, r0 + per);
        uint32_t local = 0;
        for (uint32_t r = r0; r < r1; ++r) local += cursor[r];
        uint32_t run = block_excl_scan(local, warp_tot, &s_total);
        for (uint32_t r = r0; r < r1; ++r) {
            rowptr[r] = run;
            run += cursor[r];
        }
    }
    __syncthreads();
    if (threadIdx.x == 0) { rowptr[R] = s_total; hdr->np = s_total; }
    for (uint32_t i = threadIdx.x; i <= R; i += blockDim.x) cursor[i] = 0u;
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
                const uint32_t r = pre[t >> 5] + __popc(word & ((1u << (t & 31)) - 1u));
                const uint32_t pos = atomicAdd(&cursor[r], 1u);
                pairs[rowptr[r] + pos] = make_uint2((uint32_t)j, w);
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
    const unsigned char* scratch; const uint32_t* rowptr; const uint2* pairs;   // shared rowptr / pairs arrays
    int32_t sparse_cap_bytes;                   // shared memory left for a pass's row CSR
    int64_t q0; int32_t nq;                     // queries [q0, q0+nq) in tiles of QT
    gs_tileset ts;
    gs_sink sink;
    int32_t ctas_per_pass;
};

template <int QT> struct Geo {
    static constexpr int AST = QT + 1;                 // row stride of the accumulator tile (odd: lane rows hit distinct banks)
    static constexpr int NW = QT <= 16 ? 32 : (QT == 32 ? 20 : 12);              // warps per CTA
    static constexpr int QCAP = QT <= 8 ? 384 : (QT == 16 ? 512 : (QT == 32 ? 640 : 896));   // hit-queue entries per warp
    static constexpr size_t per_warp = (size_t)QCAP * 8 + (size_t)32 * AST * 4;
    static __host__ __device__ size_t fixed(int Wd) {
        return (size_t)GS_STRIP_MAX * QT * 4 + (size_t)QT * 8 + (size_t)QT * 4 + GS_STRIP_MAX * 4 + (size_t)Wd * 8;
    }
};

template <int WT, int QT>
__global__ void __launch_bounds__(Geo<QT>::NW * 32, 1) k_score_doc(const DocParams p) {
    using W = typename NumD<WT>::W;
    using A = typename NumD<WT>::A;
    using G = Geo<QT>;
    constexpr int AST = G::AST, NW = G::NW, QCAP = G::QCAP;
    extern __shared__ __align__(16) unsigned char smem[];
    const int Wd = p.Wd;
    const int pass = blockIdx.x / p.ctas_per_pass;
    const int cta = blockIdx.x % p.ctas_per_pass;
    const unsigned char* base = p.scratch + (size_t)pass * pass_bytes(Wd, QT);
    const QTileHdr* hdr = reinterpret_cast<const QTileHdr*>(base);
    const uint32_t R = hdr->R, np = hdr->np;
    const int nh = (int)hdr->nh;
    const uint32_t* g_rowptr = p.rowptr + hdr->row_off;
    const uint2* g_pairs = p.pairs + hdr->pair_off;
    const bool sparse_in_smem = (size_t)(R + 2) * 4 + (size_t)np * 8 <= (size_t)p.sparse_cap_bytes;

    A* s_qh = reinterpret_cast<A*>(smem);                                         // [GS_STRIP_MAX][QT]
    uint64_t* s_thr = reinterpret_cast<uint64_t*>(s_qh + GS_STRIP_MAX * QT);      // [QT]
    A* s_thr_s = reinterpret_cast<A*>(s_thr + QT);                                // [QT]
    uint32_t* s_hl = reinterpret_cast<uint32_t*>(s_thr_s + QT);                   // [GS_STRIP_MAX]
    uint32_t* s_bm = s_hl + GS_STRIP_MAX;                                         // [Wd]
    uint32_t* s_pre = s_bm + Wd;                                                  // [Wd]
    unsigned char* pw = reinterpret_cast<unsigned char*>(s_pre + Wd);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    uint2* queue = reinterpret_cast<uint2*>(pw + (size_t)warp * G::per_warp);     // [QCAP]
    A* s_acc = reinterpret_cast<A*>(queue + QCAP);                                // [32][AST]
    uint2* s_pairs = reinterpret_cast<uint2*>(pw + (size_t)NW * G::per_warp);     // [np]      when it fits
    uint32_t* s_rowptr = reinterpret_cast<uint32_t*>(s_pairs + np);               // [R+1]

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
        if (sparse_in_smem) {
            for (uint32_t i = threadIdx.x; i < np; i += NW * 32) s_pairs[i] = g_pairs[i];
            for (uint32_t i = threadIdx.x; i <= R; i += NW * 32) s_rowptr[i] = g_rowptr[i];
        }
    }
    __syncthreads();
    const uint32_t* rowptr = sparse_in_smem ? s_rowptr : g_rowptr;      // generic pointers: either space
    const uint2* pairs = sparse_in_smem ? s_pairs : g_pairs;

    const W* __restrict__ fw = reinterpret_cast<const W*>(p.fwd_w);
    const W* __restrict__ strips = reinterpret_cast<const W*>(p.strips);
    const unsigned lt = (1u << lane) - 1u;
    A* myacc = s_acc + lane * AST;
    const int subs_per_tile = p.Ts >> 5;
    const int64_t n_subs = (int64_t)p.ts.count * subs_per_tile;

    // lane d applies the queued hits of document d (contiguous: the queue is in stream order)
    auto walk = [&](int n) {
        __syncwarp();
        int lo = 0, hi = n;
        for (int it = 32 - __clz(n); it > 0; --it) {          // lower bound of the first entry with doc >= lane
            const int mid = (lo + hi) >> 1;
            if (lo < hi) {
                if ((int)(queue[mid].x >> GS_FWD_DOC_SHIFT) < lane) lo = mid + 1; else hi = mid;
            }
        }
        int end = __shfl_down_sync(0xFFFFFFFFu, lo, 1);
        if (lane == 31) end = n;
        for (int j = lo; j < end; ++j) {
            const uint2 e = queue[j];
            const uint32_t t = e.x & kTermMask;
            const A w = NumD<WT>::from_bits(e.y);
            const uint32_t word = s_bm[t >> 5];
            const uint32_t r = s_pre[t >> 5] + __popc(word & ((1u << (t & 31)) - 1u));
            const uint32_t p0 = rowptr[r], p1 = rowptr[r + 1];
            for (uint32_t i = p0; i < p1; ++i) {
                const uint2 pr = pairs[i];
                myacc[pr.x] = NumD<WT>::mac(myacc[pr.x], NumD<WT>::from_bits(pr.y), w);
            }
        }
        __syncwarp();
    };

    for (int64_t sb = (int64_t)cta * NW + warp; sb < n_subs; sb += (int64_t)p.ctas_per_pass * NW) {
        const int64_t tile = p.ts.first + (sb / subs_per_tile) * (int64_t)p.ts.stride;
        const int64_t doc0 = tile * p.Ts + (sb % subs_per_tile) * 32;
        if (doc0 >= p.N) continue;
        for (int i = lane; i < 32 * AST; i += 32) s_acc[i] = A(0);

        // ---- tail: the block's postings as one flat range -> bitmap filter -> hit queue -> per-document walk
        const int64_t A0 = p.fwd_indptr[doc0];
        const int n = (int)(p.fwd_indptr[min(doc0 + 32, p.N)] - A0);
        const int32_t* __restrict__ tp = p.fwd_terms + A0;
        const W* __restrict__ wp = fw + A0;
        int cnt = 0;
        uint32_t tw[4], ww[4];
        auto load_chunk = [&](int cbase, uint32_t (&t4)[4], uint32_t (&w4)[4]) {
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const int idx = cbase + 32 * u + lane;
                const bool valid = idx < n;
                t4[u] = valid ? (uint32_t)tp[idx] : (uint32_t)p.V;            // bit V of the bitmap is never set
                w4[u] = valid ? NumD<WT>::bits(NumD<WT>::widen(wp[idx])) : 0u;
            }
        };
        load_chunk(0, tw, ww);
        for (int cbase = 0; cbase < n; cbase += 128) {
            uint32_t tn[4], wn[4];
            load_chunk(cbase + 128, tn, wn);                                  // prefetch (all-invalid past the end)
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const uint32_t t = tw[u] & kTermMask;
                const bool hit = (s_bm[t >> 5] >> (t & 31)) & 1u;
                const unsigned m = __ballot_sync(0xFFFFFFFFu, hit);
                if (m != 0u) {
                    if (cnt + 32 > QCAP) { walk(cnt); cnt = 0; }
                    if (hit) queue[cnt + __popc(m & lt)] = make_uint2(tw[u], ww[u]);
                    cnt += __popc(m);
                }
            }
#pragma unroll
            for (int u = 0; u < 4; ++u) { tw[u] = tn[u]; ww[u] = wn[u]; }
        }
        walk(cnt);

        // ---- head strips: thread = document, QT accumulators in registers
        A acc[QT];
#pragma unroll
        for (int q = 0; q < QT; ++q) acc[q] = myacc[q];
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

int norm_qt(int qtile) {
    if (qtile <= 0) return 32;
    int q = 8;
    while (q < qtile && q < 64) q <<= 1;
    return q;
}

template <int WT, int QT>
gs_status_t launch_doc(DocParams p, int64_t n_subs, int n_passes, int sms, int smem_max, cudaStream_t s) {
    using G = Geo<QT>;
    const size_t fixed = G::fixed(p.Wd) + (size_t)G::NW * G::per_warp;
    if (fixed > (size_t)smem_max) return GS_ERR_OUT_OF_RANGE;     // vocabulary too large for the shared-memory bitmap
    const size_t smem = (size_t)smem_max;
    p.sparse_cap_bytes = (int32_t)(smem - fixed);
    p.ctas_per_pass = (int)std::max<int64_t>(1, std::min<int64_t>(sms, (n_subs + G::NW - 1) / G::NW));
    const unsigned grid = (unsigned)(p.ctas_per_pass * n_passes);
    GS_CUDA(cudaFuncSetAttribute(k_score_doc<WT, QT>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    {
        GsProfScope ps(GS_K_SCORE_DOC, s);
        k_score_doc<WT, QT><<<grid, G::NW * 32, smem, s>>>(p);
    }
    ++gs_tls_launches;
    GS_CUDA(cudaGetLastError());
    return GS_OK;
}
template <int WT>
gs_status_t launch_doc_qt(int QT, const DocParams& p, int64_t n_subs, int n_passes, int sms, int smem_max, cudaStream_t s) {
    switch (QT) {
        case 8: return launch_doc<WT, 8>(p, n_subs, n_passes, sms, smem_max, s);
        case 16: return launch_doc<WT, 16>(p, n_subs, n_passes, sms, smem_max, s);
        case 32: return launch_doc<WT, 32>(p, n_subs, n_passes, sms, smem_max, s);
        default: return launch_doc<WT, 64>(p, n_subs, n_passes, sms, smem_max, s);
    }
}

}  // namespace

int gs_score_doc_qtile(int qtile) { return norm_qt(qtile); }

size_t gs_score_doc_scratch_bytes_ex(const gs_index* ix, int qtile, int64_t nq, int64_t q_nnz) {
    const int QT = norm_qt(qtile);
    const int64_t passes = std::max<int64_t>((nq + QT - 1) / QT, 1);
    const int Wd = bm_words(ix->V);
    const size_t n1 = ((size_t)(q_nnz + passes + 1) * 4 + 255) / 256 * 256;
    return pass_bytes(Wd, QT) * (size_t)passes + 2 * n1 + ((size_t)q_nnz * 8 + 255) / 256 * 256;
}

gs_status_t gs_launch_score_doc(const gs_index* ix, const gs_csr_t* q, const gs_qbatch& qb, int64_t q0, int64_t nq,
                                int qtile, const gs_tileset& ts, const gs_sink& sink, void* scratch, cudaStream_t s) {
    (void)qb;
    if (nq <= 0 || ts.count <= 0) return GS_OK;
    const int QT = norm_qt(qtile);
    const int n_passes = (int)((nq + QT - 1) / QT);
    // the scratch was sized for the whole batch (q->rows queries): lay the shared arrays out for that many passes
    const int64_t passes_cap = std::max<int64_t>((q->rows + QT - 1) / QT, 1);
    const int Wd = bm_words(ix->V);
    int dev = 0, sms = 0, smem_max = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    cudaDeviceGetAttribute(&smem_max, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
    if (q->nnz + passes_cap + 1 > 0xFFFFFFFFLL) return GS_ERR_OUT_OF_RANGE;
    {   // build all query tiles of this chunk in one launch
        const size_t bsm = sizeof(uint32_t) * 2 * (size_t)Wd;
        if (bsm > (size_t)smem_max) return GS_ERR_OUT_OF_RANGE;
        GsProfScope ps(GS_K_QTILE, s);
        if (ix->wtype == GS_W_F32) {
            GS_CUDA(cudaFuncSetAttribute(k_build_qtile<GS_W_F32>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bsm));
            k_build_qtile<GS_W_F32><<<n_passes, 1024, bsm, s>>>(q->indptr, q->term_ids, q->weights, ix->head_slot, ix->H, q0, nq,
                                                              QT, ix->V, Wd, (unsigned char*)scratch, passes_cap, q->nnz);
        } else {
            GS_CUDA(cudaFuncSetAttribute(k_build_qtile<GS_W_U8>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bsm));
            k_build_qtile<GS_W_U8><<<n_passes, 1024, bsm, s>>>(q->indptr, q->term_ids, q->weights, ix->head_slot, ix->H, q0, nq,
                                                             QT, ix->V, Wd, (unsigned char*)scratch, passes_cap, q->nnz);
        }
        ++gs_tls_launches;
        GS_CUDA(cudaGetLastError());
    }
    const SharedScratch ss = shared_scratch((unsigned char*)scratch, Wd, QT, passes_cap, q->nnz);
    DocParams p{};
    p.fwd_indptr = ix->fwd_indptr; p.fwd_terms = ix->fwd_terms; p.fwd_w = ix->fwd_w;
    p.strips = ix->head_strip; p.N_pad = ix->N_pad;
    p.N = ix->N; p.V = ix->V; p.Ts = ix->Ts; p.Wd = Wd;
    p.scratch = (const unsigned char*)scratch; p.rowptr = ss.rowptr; p.pairs = ss.pairs;
    p.q0 = q0; p.nq = (int32_t)nq;
    p.ts = ts; p.sink = sink;
    const int64_t n_subs = (int64_t)ts.count * (ix->Ts / 32);
    return ix->wtype == GS_W_F32 ? launch_doc_qt<GS_W_F32>(QT, p, n_subs, n_passes, sms, smem_max, s)
                                 : launch_doc_qt<GS_W_U8>(QT, p, n_subs, n_passes, sms, smem_max, s);
}
