// score_term.cu — S2a: term-at-a-time batched scatter-add, tiled by doc-id range (kernel K1').
//
// PAPER.md Eq. (5): scores[d] += w_i * PL(t_i)[d] for all d in PL(t_i), one independent
// scatter per query term; the paper launches one program per (query, term) that atomically adds
// into a global [B,N] buffer (L118-125, L137-172) and names "scattered atomics" as the cost
// (L172, L411).  Here the doc-id axis is cut into tiles of Ts docs and ONE WARP owns the Ts
// accumulators of one query in one doc tile ("cell row", 2 KB of shared memory at Ts = 512); a CTA
// is a handful of such warps working on consecutive queries of the same tile, several CTAs per SM:
//
//   1. zero the row;
//   2. scatter the query's "tail" lists: the per-(term, tile) segment table turns "the part of
//      PL(t) inside this tile" into two loads, probed for 32 query terms at once (one per lane,
//      the weights travel by warp shuffle); only non-empty segments are visited, each streamed
//      with coalesced loads, several independent 32-posting chunks in flight.  The row is only
//      ever touched by its warp: plain LDS/FFMA/STS, no atomics, fixed order;
//   3. add the query's "head" terms — the densest lists, stored as dense strips — straight from
//      the global strips (128-bit loads, a lane owns 4 consecutive documents; the warps of a CTA
//      share a tile, so the strips come out of L1), through the query's compact (strip, weight) list;
//   4. hand the finished cells to the sink: dense score matrix, or threshold filter -> candidate
//      list, where the warp reserves its slice of the list with ONE atomic.
//
// An earlier version gave a CTA a group of 64 queries and staged the tile's strips in shared memory;
// measured on B200 it was slower at every batch size (barrier stalls, idle warps, strips nobody
// used): DESIGN.md §7.
#include <algorithm>

#include "gs_internal.cuh"

namespace {

template <int WT> struct Num;
template <> struct Num<GS_W_F32> {
    using W = float;
    using A = float;
    static __device__ __forceinline__ A qw(uint32_t bits) { return __uint_as_float(bits); }
    static __device__ __forceinline__ A from_bits(int bits) { return __int_as_float(bits); }
    static __device__ __forceinline__ A mac(A acc, A q, A w) { return fmaf(q, w, acc); }
    static __device__ __forceinline__ A widen(W w) { return w; }
    static __device__ __forceinline__ uint32_t bits(A a) { return __float_as_uint(a); }
    static __device__ __forceinline__ A lowest() { return __uint_as_float(0xFF800000u); }      // -inf
};
template <> struct Num<GS_W_U8> {
    using W = uint8_t;
    using A = int32_t;
    static __device__ __forceinline__ A qw(uint32_t bits) { return (int32_t)bits; }
    static __device__ __forceinline__ A from_bits(int bits) { return bits; }
    static __device__ __forceinline__ A mac(A acc, A q, A w) { return acc + q * w; }
    static __device__ __forceinline__ A widen(W w) { return (int32_t)w; }
    static __device__ __forceinline__ uint32_t bits(A a) { return (uint32_t)a; }
    static __device__ __forceinline__ A lowest() { return (int32_t)0x80000000; }
};

struct TermParams {
    // index
    const int64_t* inv_off; const int32_t* inv_doc; const void* inv_w; const uint32_t* seg;
    const void* head_strip; int32_t H; int64_t N; int64_t N_pad; int32_t Ts; int32_t ntiles;
    // queries
    const int64_t* q_indptr; const uint2* head_pair; const int32_t* head_cnt; const int32_t* tail_term;
    const uint32_t* tail_w; const int32_t* tail_cnt;
    int64_t q0; int32_t nq;                     // queries [q0, q0+nq)
    int32_t warps;                              // cell rows (warps) per CTA (small-batch kernel)
    int32_t chunk, n_chunks;                    // staged kernel: queries per CTA, CTAs per doc tile
    gs_tileset ts;
    gs_sink sink;
    int32_t vec4;                               // dense sink rows are 16-byte aligned
};

// one posting-list segment [dp, dp+n) applied to one accumulator row
template <int WT>
__device__ __forceinline__ void scatter_segment(const int32_t* __restrict__ dp, const typename Num<WT>::W* __restrict__ wp,
                                                int n, typename Num<WT>::A q, typename Num<WT>::A* row, int32_t base,
                                                int32_t Ts, int lane) {
    using A = typename Num<WT>::A;
    if (n <= 32) {
        if (lane < n) {
            const int32_t rel = dp[lane] - base;
            const A w = Num<WT>::widen(wp[lane]);
            if ((uint32_t)rel < (uint32_t)Ts) row[rel] = Num<WT>::mac(row[rel], q, w);
        }
        return;
    }
    for (int c = lane; c < n; c += 128) {
        int32_t rel[4];
        A w[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const int i = c + 32 * u;
            const bool ok = i < n;
            rel[u] = ok ? dp[i] - base : -1;
            w[u] = ok ? Num<WT>::widen(wp[i]) : A(0);
        }
#pragma unroll
        for (int u = 0; u < 4; ++u)
            if ((uint32_t)rel[u] < (uint32_t)Ts) row[rel[u]] = Num<WT>::mac(row[rel[u]], q, w[u]);
    }
}

// dense sink: the finished cells (query b, docs doc0 .. doc0+3) go to the score matrix
template <int WT>
__device__ __forceinline__ void store_quad(const TermParams& p, int64_t b, int j, int dq, int64_t doc0,
                                           typename Num<WT>::A s0, typename Num<WT>::A s1, typename Num<WT>::A s2,
                                           typename Num<WT>::A s3) {
    uint32_t* out = p.sink.dense + (b - p.q0) * p.sink.ld + (int64_t)j * p.Ts + 4 * dq;
    if (doc0 + 3 < p.N && p.vec4) {
        *reinterpret_cast<uint4*>(out) = make_uint4(Num<WT>::bits(s0), Num<WT>::bits(s1), Num<WT>::bits(s2), Num<WT>::bits(s3));
    } else {
        if (doc0 + 0 < p.N) out[0] = Num<WT>::bits(s0);
        if (doc0 + 1 < p.N) out[1] = Num<WT>::bits(s1);
        if (doc0 + 2 < p.N) out[2] = Num<WT>::bits(s2);
        if (doc0 + 3 < p.N) out[3] = Num<WT>::bits(s3);
    }
}

constexpr int kWarpsDefault = 2, kWarpsMax = 8;
constexpr int kSegBatch = 2;      // segments whose first 32 postings are loaded together
constexpr int kQuadRounds = 2;    // rounds of 32 quads (128 documents) a lane keeps in registers in the epilogue

// One (doc tile, query) cell row, done by one warp.  STAGED: the tile's strips are in shared memory (s_strip, [H][Ts]);
// otherwise they are read from the global strips.
template <int WT, bool STAGED>
__device__ __forceinline__ void process_item(const TermParams& p, typename Num<WT>::A* row,
                                             const typename Num<WT>::W* s_strip, int j, int64_t b, int lane) {
    using W = typename Num<WT>::W;
    using A = typename Num<WT>::A;
    const int Ts = p.Ts;
    const int tile = p.ts.first + j * p.ts.stride;
    const int32_t base = tile * Ts;
    const int quads = Ts >> 2;
    for (int dq = lane; dq < quads; dq += 32) reinterpret_cast<int4*>(row)[dq] = make_int4(0, 0, 0, 0);
    __syncwarp();

    // scatter the tail lists of the query: segment of each list inside this tile, 32 terms probed at once.  The
    // non-empty segments are applied one after the other (two lists may hit the same document), but the first 32
    // postings of kSegBatch segments are LOADED together, so their latencies overlap.
    const W* __restrict__ inv_w = reinterpret_cast<const W*>(p.inv_w);
    const int64_t qa = p.q_indptr[b];
    const int cnt = p.tail_cnt[b];
    for (int i0 = 0; i0 < cnt; i0 += 32) {
        int64_t start = 0;
        int n = 0;
        uint32_t wq = 0;
        if (i0 + lane < cnt) {
            const int32_t t = p.tail_term[qa + i0 + lane];
            wq = p.tail_w[qa + i0 + lane];
            const uint32_t* sr = p.seg + (size_t)t * (p.ntiles + 1) + tile;
            const uint32_t lo = sr[0], hi = sr[1];
            n = (int)(hi - lo);
            start = p.inv_off[t] + lo;
        }
        unsigned m = __ballot_sync(0xFFFFFFFFu, n > 0);
        while (m) {
            int n_j[kSegBatch];
            int64_t start_j[kSegBatch];
            A q_j[kSegBatch], w_j[kSegBatch];
            int32_t rel_j[kSegBatch];
#pragma unroll
            for (int u = 0; u < kSegBatch; ++u) {
                n_j[u] = 0;
                if (m) {                                    // uniform
                    const int src = __ffs(m) - 1;
                    m &= m - 1;
                    n_j[u] = __shfl_sync(0xFFFFFFFFu, n, src);
                    start_j[u] = __shfl_sync(0xFFFFFFFFu, start, src);
                    q_j[u] = Num<WT>::qw(__shfl_sync(0xFFFFFFFFu, wq, src));
                    const bool ok = lane < n_j[u];
                    rel_j[u] = ok ? p.inv_doc[start_j[u] + lane] - base : -1;
                    w_j[u] = ok ? Num<WT>::widen(inv_w[start_j[u] + lane]) : A(0);
                }
            }
#pragma unroll
            for (int u = 0; u < kSegBatch; ++u) {
                if (n_j[u] > 0) {                           // uniform
                    if ((uint32_t)rel_j[u] < (uint32_t)Ts) row[rel_j[u]] = Num<WT>::mac(row[rel_j[u]], q_j[u], w_j[u]);
                    if (n_j[u] > 32)
                        scatter_segment<WT>(p.inv_doc + start_j[u] + 32, inv_w + start_j[u] + 32, n_j[u] - 32, q_j[u], row, base, Ts, lane);
                    __syncwarp();                           // two lists may hit the same document
                }
            }
        }
    }
    __syncwarp();

    // head strips + sink.  A lane owns 4 consecutive documents ("quad") in each of up to kQuadRounds rounds of 32
    // quads; the strip loop is the OUTER loop, so one (strip, weight) entry feeds kQuadRounds independent 128-bit
    // strip loads.  Filter mode makes two passes over the row so that a warp reserves its slice of the query's
    // candidate list with ONE atomic: pass 1 finishes the scores in place and counts the cells that pass the
    // threshold, pass 2 writes their keys.
    const int nh = p.H > 0 ? p.head_cnt[b] : 0;
    const uint2* hl = p.head_pair + b * GS_HEAD_MAX;
    const W* __restrict__ gstrip = STAGED ? s_strip : reinterpret_cast<const W*>(p.head_strip) + base;
    const size_t strip_ld = STAGED ? (size_t)Ts : (size_t)p.N_pad;
    const bool filter = p.sink.thr != nullptr;
    const uint64_t thr = filter ? p.sink.thr[b] : 0ull;
    // Score and doc id of the threshold key: key >= threshold key  <=>  score > its score, or equal and doc id <= its doc
    // id (two or three compares per cell instead of building the 64-bit key).  Threshold key 0 = accept everything.
    const A thr_s = thr == 0ull ? Num<WT>::lowest()
                                : Num<WT>::from_bits((int)(WT == GS_W_F32 ? gs_unord_f32((uint32_t)(thr >> 32))
                                                                          : ((uint32_t)(thr >> 32) ^ 0x80000000u)));
    const int n_live = (int)min((int64_t)Ts, p.N - (int64_t)base);      // documents of this tile that exist
    const int64_t thr_cell = (int64_t)(0xFFFFFFFFu - (uint32_t)thr) - (int64_t)base;   // threshold doc as a cell of this tile
    const int tie_cells = (int)max((int64_t)-1, min((int64_t)Ts, thr_cell));           // cells <= this index win a score tie
    uint64_t* cand = filter ? p.sink.cand + b * p.sink.cand_cap : nullptr;
    for (int dq0 = 0; dq0 < quads; dq0 += 32 * kQuadRounds) {
        const bool whole = dq0 + 32 * kQuadRounds <= quads;             // uniform: no quad of this chunk is out of range
        A sc[kQuadRounds][4];
#pragma unroll
        for (int r = 0; r < kQuadRounds; ++r) {
            const int dq = dq0 + 32 * r + lane;
            const int4 a4 = (whole || dq < quads) ? reinterpret_cast<const int4*>(row)[dq] : make_int4(0, 0, 0, 0);
            sc[r][0] = Num<WT>::from_bits(a4.x); sc[r][1] = Num<WT>::from_bits(a4.y);
            sc[r][2] = Num<WT>::from_bits(a4.z); sc[r][3] = Num<WT>::from_bits(a4.w);
        }
        for (int i = 0; i < nh; ++i) {
            const uint2 e = __ldg(hl + i);
            const A q = Num<WT>::qw(e.y);
            const W* src = gstrip + (size_t)e.x * strip_ld + 4 * (dq0 + lane);
            int4 v[kQuadRounds];
#pragma unroll
            for (int r = 0; r < kQuadRounds; ++r) {
                if (whole || dq0 + 32 * r + lane < quads) {
                    if (WT == GS_W_F32) {
                        v[r] = STAGED ? *reinterpret_cast<const int4*>(src + 128 * r) : __ldg(reinterpret_cast<const int4*>(src + 128 * r));
                    } else {
                        const uchar4 u = STAGED ? *reinterpret_cast<const uchar4*>(src + 128 * r)
                                                : __ldg(reinterpret_cast<const uchar4*>(src + 128 * r));
                        v[r] = make_int4(u.x, u.y, u.z, u.w);
                    }
                } else {
                    v[r] = make_int4(0, 0, 0, 0);
                }
            }
#pragma unroll
            for (int r = 0; r < kQuadRounds; ++r) {
                sc[r][0] = Num<WT>::mac(sc[r][0], q, Num<WT>::from_bits(v[r].x));
                sc[r][1] = Num<WT>::mac(sc[r][1], q, Num<WT>::from_bits(v[r].y));
                sc[r][2] = Num<WT>::mac(sc[r][2], q, Num<WT>::from_bits(v[r].z));
                sc[r][3] = Num<WT>::mac(sc[r][3], q, Num<WT>::from_bits(v[r].w));
            }
        }
        if (!filter) {
#pragma unroll
            for (int r = 0; r < kQuadRounds; ++r) {
                const int dq = dq0 + 32 * r + lane;
                if (whole || dq < quads) store_quad<WT>(p, b, j, dq, (int64_t)base + 4 * dq, sc[r][0], sc[r][1], sc[r][2], sc[r][3]);
            }
            continue;
        }
        // filter: bit (4r + u) of `mask` = cell u of the lane's quad in round r passes; the finished scores go back to the row
        uint32_t mask = 0;
#pragma unroll
        for (int r = 0; r < kQuadRounds; ++r) {
            const int dq = dq0 + 32 * r + lane;
            if (whole || dq < quads) {
                reinterpret_cast<uint4*>(row)[dq] = make_uint4(Num<WT>::bits(sc[r][0]), Num<WT>::bits(sc[r][1]),
                                                               Num<WT>::bits(sc[r][2]), Num<WT>::bits(sc[r][3]));
#pragma unroll
                for (int u = 0; u < 4; ++u)
                    if ((sc[r][u] > thr_s || (sc[r][u] == thr_s && 4 * dq + u <= tie_cells)) && 4 * dq + u < n_live)
                        mask |= 1u << (4 * r + u);
            }
        }
        if (__ballot_sync(0xFFFFFFFFu, mask != 0u) == 0u) continue;     // no candidate in this chunk (the common case)
        // the warp reserves its slice of the query's candidate list with ONE atomic
        const uint32_t mine = (uint32_t)__popc(mask);
        uint32_t incl = mine;
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t v = __shfl_up_sync(0xFFFFFFFFu, incl, o);
            if (lane >= o) incl += v;
        }
        const uint32_t total = __shfl_sync(0xFFFFFFFFu, incl, 31);
        uint32_t pos = 0;
        if (lane == 0) pos = atomicAdd(&p.sink.cand_cnt[b], total);
        pos = __shfl_sync(0xFFFFFFFFu, pos, 0) + incl - mine;
        while (mask) {
            const int bit = __ffs(mask) - 1;
            mask &= mask - 1;
            const int cell = 4 * (dq0 + 32 * (bit >> 2) + lane) + (bit & 3);
            if ((int64_t)pos < p.sink.cand_cap)
                cand[pos] = gs_make_key(gs_ord_bits<WT>(Num<WT>::bits(row[cell])), (uint32_t)(base + cell));
            ++pos;
        }
    }
}

// small batches: a warp takes ONE cell row; consecutive warps take consecutive queries of the same tile
template <int WT>
__global__ void __launch_bounds__(kWarpsMax * 32) k_score_term(const TermParams p) {
    using A = typename Num<WT>::A;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int64_t item = (int64_t)blockIdx.x * p.warps + warp;
    if (item >= (int64_t)p.ts.count * p.nq) return;
    const int j = (int)(item / p.nq);                       // position in the tile set
    const int64_t b = p.q0 + (item - (int64_t)j * p.nq);
    A* row = reinterpret_cast<A*>(smem_raw) + (size_t)warp * p.Ts;
    process_item<WT, false>(p, row, nullptr, j, b, lane);
}

// batches: a CTA of kWarpsStaged warps takes ONE doc tile and a chunk of up to p.chunk queries; it stages the tile's
// strips in shared memory once (without this every cell row re-reads its strips from L2: CTAs of one tile land on
// different SMs, so L1 does not help — measured 191 GB of L2 reads per batch), then every warp walks its share of the
// chunk's queries on its own, with no barrier after the staging.
constexpr int kWarpsStaged = 32;

template <int WT>
__global__ void __launch_bounds__(kWarpsStaged * 32, 1) k_score_term_staged(const TermParams p) {
    using W = typename Num<WT>::W;
    using A = typename Num<WT>::A;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int Ts = p.Ts;
    const int j = (int)(blockIdx.x / p.n_chunks);
    const int chunk = (int)(blockIdx.x - (unsigned)j * p.n_chunks);
    A* rows = reinterpret_cast<A*>(smem_raw);                                   // [kWarpsStaged][Ts]
    W* s_strip = reinterpret_cast<W*>(rows + (size_t)kWarpsStaged * Ts);         // [H][Ts]
    {
        const int tile = p.ts.first + j * p.ts.stride;
        const W* __restrict__ g = reinterpret_cast<const W*>(p.head_strip) + (size_t)tile * Ts;
        const int per = Ts / (16 / (int)sizeof(W));                            // 16-byte pieces per strip (Ts % 32 == 0)
        for (int i = threadIdx.x; i < p.H * per; i += kWarpsStaged * 32) {
            const int h = i / per, c = i - h * per;
            reinterpret_cast<int4*>(s_strip + (size_t)h * Ts)[c] =
                __ldg(reinterpret_cast<const int4*>(g + (size_t)h * p.N_pad) + c);
        }
    }
    __syncthreads();
    const int q_end = min(p.nq, (chunk + 1) * p.chunk);
    for (int q = chunk * p.chunk + warp; q < q_end; q += kWarpsStaged)
        process_item<WT, true>(p, rows + (size_t)warp * Ts, s_strip, j, p.q0 + q, lane);
}

int norm_warps(int w) { return w <= 0 ? kWarpsDefault : std::min(w, kWarpsMax); }

template <int WT>
gs_status_t launch(const TermParams& p, unsigned grid, size_t smem, bool staged, cudaStream_t s) {
    if (staged) {
        GS_CUDA(cudaFuncSetAttribute(k_score_term_staged<WT>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        GsProfScope ps(GS_K_SCORE_TERM, s);
        k_score_term_staged<WT><<<grid, kWarpsStaged * 32, smem, s>>>(p);
    } else {
        GS_CUDA(cudaFuncSetAttribute(k_score_term<WT>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        GsProfScope ps(GS_K_SCORE_TERM, s);
        k_score_term<WT><<<grid, p.warps * 32, smem, s>>>(p);
    }
    ++gs_tls_launches;
    GS_CUDA(cudaGetLastError());
    return GS_OK;
}

constexpr int kStagedMinQueries = 64;     // below this the warp-per-row shape is as fast or faster (measured batch sweep)
constexpr int kStagedChunk = 512;         // queries per CTA of the staged kernel

}  // namespace

int gs_score_term_group(const gs_index* ix, int64_t nq, int group, bool use_head) {
    if (group <= 0 && nq >= kStagedMinQueries && use_head && ix->H > 0) return kWarpsStaged;
    return norm_warps(group);
}

gs_status_t gs_launch_score_term(const gs_index* ix, const gs_qbatch& qb, int64_t q0, int64_t nq, int group,
                                 bool use_head, const gs_tileset& ts, const gs_sink& sink, cudaStream_t s) {
    if (nq <= 0 || ts.count <= 0) return GS_OK;
    TermParams p{};
    p.inv_off = ix->inv_off; p.inv_doc = ix->inv_doc; p.inv_w = ix->inv_w; p.seg = ix->seg;
    p.head_strip = ix->head_strip; p.H = use_head ? ix->H : 0; p.N = ix->N; p.N_pad = ix->N_pad; p.Ts = ix->Ts;
    p.ntiles = ix->ntiles;
    p.q_indptr = qb.indptr; p.head_pair = qb.head_pair; p.head_cnt = qb.head_cnt; p.tail_term = qb.tail_term;
    p.tail_w = qb.tail_w; p.tail_cnt = qb.tail_cnt;
    p.q0 = q0; p.nq = (int32_t)nq;
    p.warps = norm_warps(group);
    p.ts = ts; p.sink = sink;
    p.vec4 = sink.dense && (((uintptr_t)sink.dense | (uintptr_t)(sink.ld * 4)) & 15) == 0;
    int dev = 0, smem_max = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&smem_max, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
    const size_t wbytes = ix->wtype == GS_W_F32 ? 4 : 1;
    const size_t smem_staged = (size_t)kWarpsStaged * ix->Ts * 4 + (size_t)p.H * ix->Ts * wbytes;
    // query_group > 0 pins the small-batch kernel (that many cell rows per CTA)
    if (group <= 0 && nq >= kStagedMinQueries && p.H > 0 && smem_staged <= (size_t)smem_max) {
        p.chunk = kStagedChunk;
        p.n_chunks = (int32_t)((nq + p.chunk - 1) / p.chunk);
        const int64_t grid = (int64_t)ts.count * p.n_chunks;
        if (grid > 0x7FFFFFFFLL) return GS_ERR_OUT_OF_RANGE;
        return ix->wtype == GS_W_F32 ? launch<GS_W_F32>(p, (unsigned)grid, smem_staged, true, s)
                                     : launch<GS_W_U8>(p, (unsigned)grid, smem_staged, true, s);
    }
    while (p.warps > 1 && (size_t)p.warps * ix->Ts * 4 > (size_t)smem_max) p.warps >>= 1;
    const size_t smem = (size_t)p.warps * ix->Ts * 4;
    if (smem > (size_t)smem_max) return GS_ERR_OOM;                 // one accumulator row does not fit: tile_docs too large
    const int64_t grid = ((int64_t)ts.count * nq + p.warps - 1) / p.warps;
    if (grid > 0x7FFFFFFFLL) return GS_ERR_OUT_OF_RANGE;
    return ix->wtype == GS_W_F32 ? launch<GS_W_F32>(p, (unsigned)grid, smem, false, s)
                                 : launch<GS_W_U8>(p, (unsigned)grid, smem, false, s);
}
