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
// Three kernels share this ownership rule: k_score_term (small batches, a warp per cell row, strips from
// global memory), k_score_term_staged (batches, any tile size: persistent CTA per doc tile, strips staged in
// shared memory) and k_score_term_batch (batches, 512-doc tiles: the same CTA shape with the tail walked as one
// flat posting stream, FFMA2 strips and a shared-memory candidate buffer — see its own comment).
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
    const int32_t* inv_doc; const void* inv_w;
    const uint32_t* inv_pk;                      // integer-impact mode, compressed postings: doc | impact << 24 (else null)
    const uint32_t* seg_tab; const uint2* seg_l1; const uint32_t* seg_l2;     // tile-segment tables (gs_term_meta), absolute slots
    const void* head_strip; int32_t H; int64_t N; int64_t N_pad; int32_t Ts; int32_t ntiles;
    // queries
    const int64_t* q_indptr; const uint2* head_pair; const int32_t* head_cnt; const uint4* tail_desc;
    const int32_t* tail_cnt; const uint4* tail32;
    const void* xstrip; const uint2* xpair; const int32_t* xcnt;      // second-tier strips (null when the batch has none)
    const uint8_t* mma_strips;                  // integer mode: the strips as the A operand of k_score_term_mma (else null)
    int64_t q0; int32_t nq;                     // queries [q0, q0+nq)
    int32_t warps;                              // cell rows (warps) per CTA (small-batch kernel)
    int32_t chunk, n_chunks;                    // staged kernel: queries per CTA, CTAs per doc tile
    gs_tileset ts;
    gs_sink sink;
    int32_t vec4;                               // dense sink rows are 16-byte aligned
    int32_t pf_rows;                            // small-batch kernel: few rows in flight -> each asks the L2 for its strips at its start
};

// Slot range [lo, hi) of the postings of a tail term (descriptor d: weight bits, table offset, table mode, -) inside doc
// tile `tile`.  Full mode: two adjacent table entries.  Sparse mode: one (mask, index) entry per 32 tiles; an empty
// (term, tile) pair stops there.
__device__ __forceinline__ void probe_range(const TermParams& p, const uint4& d, int tile, uint32_t& lo, uint32_t& hi) {
    lo = hi = 0u;
    if (d.z == GS_SEG_FULL) {
        lo = __ldg(p.seg_tab + d.y + tile);
        hi = __ldg(p.seg_tab + d.y + tile + 1);
    } else if (d.z == GS_SEG_SPARSE) {
        const uint2 e = __ldg(p.seg_l1 + d.y + (tile >> 5));
        const uint32_t bit = 1u << (tile & 31);
        if (e.x & bit) {
            const uint32_t idx = e.y + (uint32_t)__popc(e.x & (bit - 1u));
            lo = __ldg(p.seg_l2 + idx);
            hi = __ldg(p.seg_l2 + idx + 1);
        }
    }
}
// entry i of a query's compact head list: the hot strips from the front, the others from the back (ingest.cu)
__device__ __forceinline__ uint2 head_entry(const uint2* hl, int i, int n_hot) {
    return __ldg(hl + (i < n_hot ? i : GS_HEAD_MAX - 1 - (i - n_hot)));
}

// Posting at slot idx of the inverted index: (doc id, weight widened to the accumulator type).  Integer-impact mode with
// compressed postings reads ONE word (doc | impact << 24), otherwise the two arrays of PAPER.md L79-84.
template <int WT>
__device__ __forceinline__ void load_posting(const TermParams& p, uint32_t idx, int32_t& doc, typename Num<WT>::A& w) {
    using W = typename Num<WT>::W;
    if (WT == GS_W_U8 && p.inv_pk != nullptr) {
        const uint32_t pk = __ldg(p.inv_pk + idx);
        doc = (int32_t)(pk & 0xFFFFFFu);
        w = Num<WT>::from_bits((int)(pk >> 24));
    } else {
        doc = __ldg(p.inv_doc + idx);
        w = Num<WT>::widen(__ldg(reinterpret_cast<const W*>(p.inv_w) + idx));
    }
}

// one posting-list segment (slots [start, start+n)) applied to one accumulator row
template <int WT>
__device__ __forceinline__ void scatter_segment(const TermParams& p, uint32_t start, int n, typename Num<WT>::A q,
                                                typename Num<WT>::A* row, int32_t base, int32_t Ts, int lane) {
    using A = typename Num<WT>::A;
    if (n <= 32) {
        if (lane < n) {
            int32_t doc;
            A w;
            load_posting<WT>(p, start + lane, doc, w);
            const int32_t rel = doc - base;
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
            rel[u] = -1;
            w[u] = A(0);
            if (i < n) { load_posting<WT>(p, start + i, rel[u], w[u]); rel[u] -= base; }
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
template <int WT, bool STAGED, bool XS>
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
    if (!STAGED && p.pf_rows) {
        // A launch of few rows (the threshold sample of a small batch: 136 rows at B = 1) is pure latency: the head phase
        // below reads a row's strip segments strip by strip, ~26 exposed round trips per row.  Ask the L2 for all of
        // them now (one 128-byte line per lane and turn, no registers): they arrive under the tail scatter.  Only for
        // such launches: with thousands of rows in flight (26 KB each) the prefetched lines exceed the L2 and are gone
        // before their use (single-query filter launch: 0.138 -> 0.160 ms, profiles/r02_kernels.md).
        const int L = (Ts * (int)sizeof(W) + 127) >> 7;                    // lines per strip segment
        if ((L & (L - 1)) == 0 && L <= 32) {
            const int sh = 31 - __clz(L), spw = 32 >> sh;                   // strips per warp turn
            const int hc0 = p.H > 0 ? p.head_cnt[b] : 0;
            const int nh0 = hc0 & 0xFF, n_hot0 = hc0 >> 8;
            const uint2* hl0 = p.head_pair + b * GS_HEAD_MAX;
            const char* g0 = reinterpret_cast<const char*>(reinterpret_cast<const W*>(p.head_strip) + base) + ((lane & (L - 1)) << 7);
            for (int s0 = 0; s0 < nh0; s0 += spw) {
                const int si = s0 + (lane >> sh);
                if (si < nh0) {
                    const uint2 e = head_entry(hl0, si, n_hot0);
                    asm volatile("prefetch.global.L2 [%0];" ::"l"(g0 + (size_t)e.x * (size_t)p.N_pad * sizeof(W)));
                }
            }
            if (XS) {
                const int nx0 = p.xcnt[b];
                const uint2* xl0 = p.xpair + b * GS_XSTRIP_MAX;
                const char* x0 = reinterpret_cast<const char*>(reinterpret_cast<const W*>(p.xstrip) + base) + ((lane & (L - 1)) << 7);
                for (int s0 = 0; s0 < nx0; s0 += spw) {
                    const int si = s0 + (lane >> sh);
                    if (si < nx0) {
                        const uint2 e = __ldg(xl0 + si);
                        asm volatile("prefetch.global.L2 [%0];" ::"l"(x0 + (size_t)e.x * (size_t)p.N_pad * sizeof(W)));
                    }
                }
            }
        }
    }

    // scatter the tail lists of the query: segment of each list inside this tile, 32 terms probed at once.  The
    // non-empty segments are applied one after the other (two lists may hit the same document), but the first 32
    // postings of kSegBatch segments are LOADED together, so their latencies overlap.
    const int64_t qa = p.q_indptr[b];
    const int cnt = p.tail_cnt[b];
    for (int i0 = 0; i0 < cnt; i0 += 32) {
        uint32_t start = 0;
        int n = 0;
        uint32_t wq = 0;
        if (i0 + lane < cnt) {
            const uint4 d = __ldg(p.tail_desc + qa + i0 + lane);
            wq = d.x;
            uint32_t hi;
            probe_range(p, d, tile, start, hi);
            n = (int)(hi - start);
        }
        unsigned m = __ballot_sync(0xFFFFFFFFu, n > 0);
        while (m) {
            int n_j[kSegBatch];
            uint32_t start_j[kSegBatch];
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
                    rel_j[u] = -1;
                    w_j[u] = A(0);
                    if (lane < n_j[u]) { load_posting<WT>(p, start_j[u] + lane, rel_j[u], w_j[u]); rel_j[u] -= base; }
                }
            }
#pragma unroll
            for (int u = 0; u < kSegBatch; ++u) {
                if (n_j[u] > 0) {                           // uniform
                    if ((uint32_t)rel_j[u] < (uint32_t)Ts) row[rel_j[u]] = Num<WT>::mac(row[rel_j[u]], q_j[u], w_j[u]);
                    if (n_j[u] > 32)
                        scatter_segment<WT>(p, start_j[u] + 32, n_j[u] - 32, q_j[u], row, base, Ts, lane);
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
    const int hc = p.H > 0 ? p.head_cnt[b] : 0;
    const int nh = hc & 0xFF, n_hot = hc >> 8;
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
            const uint2 e = head_entry(hl, i, n_hot);
            const A q = Num<WT>::qw(e.y);
            const W* src = gstrip + (size_t)e.x * strip_ld + 4 * (dq0 + lane);
            int4 v[kQuadRounds];
#pragma unroll
            for (int r = 0; r < kQuadRounds; ++r) {
                if (whole || dq0 + 32 * r + lane < quads) {
                    if (WT == GS_W_F32) {
                        v[r] = STAGED ? *reinterpret_cast<const int4*>(src + 128 * r) : __ldg(reinterpret_cast<const int4*>(src + 128 * r));
                    } else {
                        // impacts: the four bytes stay packed in v[r].x; one IDP4A per cell below picks its byte
                        v[r].x = (int)(STAGED ? *reinterpret_cast<const uint32_t*>(src + 128 * r)
                                              : __ldg(reinterpret_cast<const uint32_t*>(src + 128 * r)));
                    }
                } else {
                    v[r] = make_int4(0, 0, 0, 0);
                }
            }
#pragma unroll
            for (int r = 0; r < kQuadRounds; ++r) {
                if (WT == GS_W_F32) {
                    sc[r][0] = Num<WT>::mac(sc[r][0], q, Num<WT>::from_bits(v[r].x));
                    sc[r][1] = Num<WT>::mac(sc[r][1], q, Num<WT>::from_bits(v[r].y));
                    sc[r][2] = Num<WT>::mac(sc[r][2], q, Num<WT>::from_bits(v[r].z));
                    sc[r][3] = Num<WT>::mac(sc[r][3], q, Num<WT>::from_bits(v[r].w));
                } else {
#pragma unroll
                    for (int u = 0; u < 4; ++u)
                        sc[r][u] = Num<WT>::from_bits((int)__dp4a((uint32_t)v[r].x, (e.y & 0xFFu) << (8 * u), Num<WT>::bits(sc[r][u])));
                }
            }
        }
        if (XS) {                               // second-tier strips, from global memory
            const int nx = p.xcnt[b];
            const uint2* xl = p.xpair + b * GS_XSTRIP_MAX;
            const W* __restrict__ gx = reinterpret_cast<const W*>(p.xstrip) + base;
            for (int i = 0; i < nx; ++i) {
                const uint2 e = __ldg(xl + i);
                const A q = Num<WT>::qw(e.y);
                const W* src = gx + (size_t)e.x * (size_t)p.N_pad + 4 * (dq0 + lane);
#pragma unroll
                for (int r = 0; r < kQuadRounds; ++r) {
                    if (whole || dq0 + 32 * r + lane < quads) {
                        int4 v;
                        if (WT == GS_W_F32) {
                            v = __ldg(reinterpret_cast<const int4*>(src + 128 * r));
                        } else {
                            const uchar4 u = __ldg(reinterpret_cast<const uchar4*>(src + 128 * r));
                            v = make_int4(u.x, u.y, u.z, u.w);
                        }
                        sc[r][0] = Num<WT>::mac(sc[r][0], q, Num<WT>::from_bits(v.x));
                        sc[r][1] = Num<WT>::mac(sc[r][1], q, Num<WT>::from_bits(v.y));
                        sc[r][2] = Num<WT>::mac(sc[r][2], q, Num<WT>::from_bits(v.z));
                        sc[r][3] = Num<WT>::mac(sc[r][3], q, Num<WT>::from_bits(v.w));
                    }
                }
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
        if (lane == 0) pos = atomicAdd(&p.sink.cand_cnt[b * GS_CNT_STRIDE], total);
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
template <int WT, bool XS>
__global__ void __launch_bounds__(kWarpsMax * 32) k_score_term(const TermParams p) {
    using A = typename Num<WT>::A;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int64_t item = (int64_t)blockIdx.x * p.warps + warp;
    if (item >= (int64_t)p.ts.count * p.nq) return;
    const int j = (int)(item / p.nq);                       // position in the tile set
    const int64_t b = p.q0 + (item - (int64_t)j * p.nq);
    A* row = reinterpret_cast<A*>(smem_raw) + (size_t)warp * p.Ts;
    process_item<WT, false, XS>(p, row, nullptr, j, b, lane);
}

// batches: a CTA of kWarpsStaged warps takes ONE doc tile and a chunk of up to p.chunk queries; it stages the tile's
// strips in shared memory once (without this every cell row re-reads its strips from L2: CTAs of one tile land on
// different SMs, so L1 does not help — measured 191 GB of L2 reads per batch), then every warp walks its share of the
// chunk's queries on its own, with no barrier after the staging.
constexpr int kWarpsStaged = 32;

template <int WT, bool XS>
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
        process_item<WT, true, XS>(p, rows + (size_t)warp * Ts, s_strip, j, p.q0 + q, lane);
}

// ------------------------------------------------------------------------------------------------
// Batch kernel (Ts == 512, >= kStagedMinQueries queries, < 2^32 posting slots): same ownership as above — a persistent
// CTA per doc tile stages the tile's strips once, a warp owns one (query, tile) cell row at a time — with the three
// per-row phases rebuilt around what the ncu source view of the staged kernel showed (profiles/r01d_kernels.md:
// the tail scatter, 8 % of the multiply-adds, took half of the instructions and 57 % of the stall samples):
//   * tail: the row's non-empty segments are FLATTENED into one posting stream.  An exclusive scan of the segment
//     lengths gives every segment its start in the stream; in a round of 32 flat postings a lane finds its segment
//     with one warp OR-reduction (bit i = "a segment starts at flat position f0+i") and a popcount, fetches
//     (segment start - stream start, query weight) from a 32-entry per-warp table in shared memory, and loads its
//     posting: every lane is busy, and the loads of kRounds rounds are in flight together.  The read-modify-writes
//     of a round resolve same-cell conflicts (two lists may hit the same document; one list never does) either list by
//     list (integer mode: the order of the additions into a cell is the query's term order) or, fp32, with one tag byte
//     per cell that picks the lane allowed to update it in this pass (scatter_flat): no atomics, reproducible run to run;
//   * the probes (query terms -> segment table -> list offsets) of the NEXT TWO queries of the warp are prefetched
//     (two-stage software pipeline) from the fixed-stride tail32 table;
//   * head: a lane keeps its 16 documents in registers.  The query's compact strip lists are loaded once, one entry per
//     lane, and broadcast by shuffle.  fp32: the GS_HOT_STRIPS densest strips of the tile live in TENSOR MEMORY (one
//     tcgen05.ld.32x32b.x16 per strip feeds eight FFMA2, see tmem_ld16_wait), the other strips in shared memory (one
//     LDS.128 feeds two FFMA2), the second-tier strips come from global memory.  Integer mode: one IDP4A per cell;
//   * filter: a hit mask over the lane's 16 cells, then a loop over its set bits: a cell that passes goes to the warp's
//     candidate buffer in shared memory.
// Things measured and dropped in round 2 (profiles/r02_kernels.md): a 16-warp x 128-register variant that worked on two
// rows per warp (one per half-warp in the tail phase, strip loads double-buffered) — 20.2 ms against 16.4 ms; L2
// prefetches (next row's posting segments, next doc tile's strips), second-tier strips in the hot strips' staging rows,
// deeper unrolling of the strip loops — each slower or within the noise in a same-unit A/B.
// ------------------------------------------------------------------------------------------------
constexpr int kBT = 512;          // documents per tile
// Values kept after the sweeps of rounds 1 and 2 (profiles/r01d_kernels.md, profiles/r02_kernels.md): 24 warps x 80 registers
// 23.5-25.9 ms, two posting rounds in flight 17.6 vs 16.7 ms (spills), head loop unrolled by 4 16.7 -> 16.3 ms.
constexpr int kBWarps = 32;       // warps (cell rows in flight) per CTA
constexpr int kRounds = 1;        // flat posting rounds whose loads are issued together
constexpr int kHeadUnroll = 4;    // strips of the integer head loop whose loads are issued together

__device__ __forceinline__ unsigned long long pack_f32x2(float lo, float hi) {
    unsigned long long d;
    asm("mov.b64 %0, {%1, %2};" : "=l"(d) : "f"(lo), "f"(hi));
    return d;
}
__device__ __forceinline__ unsigned long long pack_u32x2(uint32_t lo, uint32_t hi) {
    unsigned long long d;
    asm("mov.b64 %0, {%1, %2};" : "=l"(d) : "r"(lo), "r"(hi));
    return d;
}
__device__ __forceinline__ void unpack_f32x2(unsigned long long v, float& lo, float& hi) {
    asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v));
}
// (a.lo * b.lo + c.lo, a.hi * b.hi + c.hi): one FFMA2, each half an IEEE fp32 fma (same result as two fmaf)
__device__ __forceinline__ unsigned long long fma_f32x2(unsigned long long a, unsigned long long b, unsigned long long c) {
    unsigned long long d;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c));
    return d;
}
// ---- tensor memory as a strip store (fp32 batch kernel).  TMEM is 128 lanes x 512 columns of 32 bits per SM; a warp
// reaches the 32 lanes of its quarter (warp % 4).  The GS_HOT_STRIPS densest strips of the doc tile are kept there, every
// lane quarter holding a full copy: lane i, column s*16 + 4r + u = strip s, document 4*(i + 32r) + u of the tile — the 16
// documents lane i of a warp owns in the head phase, so ONE tcgen05.ld.32x32b.x16 replaces the four LDS.128 of a strip.
// Measured on B200: 6.4 SM cycles per (warp, strip) against 16 from shared memory, and the two paths
// overlap, which takes the hot strips off the LSU / shared-memory pipe that bounded the kernel.
// Loads the lane's 16 documents of one strip and waits for them (tcgen05.wait::ld waits for every tensor-memory load of
// the thread).  Load, wait and the packing into eight f32x2 operands are ONE asm block, so the compiler cannot move a use
// of the values above the wait, and ptxas allocates the 16 destination registers as aligned pairs (FFMA2 operands).
__device__ __forceinline__ void tmem_ld16_wait(uint32_t taddr, unsigned long long (&d)[8]) {
    asm volatile(
        "{\n\t.reg .b32 t<16>;\n\t"
        "tcgen05.ld.sync.aligned.32x32b.x16.b32 {t0,t1,t2,t3,t4,t5,t6,t7,t8,t9,t10,t11,t12,t13,t14,t15}, [%8];\n\t"
        "tcgen05.wait::ld.sync.aligned;\n\t"
        "mov.b64 %0, {t0,t1};\n\tmov.b64 %1, {t2,t3};\n\tmov.b64 %2, {t4,t5};\n\tmov.b64 %3, {t6,t7};\n\t"
        "mov.b64 %4, {t8,t9};\n\tmov.b64 %5, {t10,t11};\n\tmov.b64 %6, {t12,t13};\n\tmov.b64 %7, {t14,t15};\n\t}"
        : "=l"(d[0]), "=l"(d[1]), "=l"(d[2]), "=l"(d[3]), "=l"(d[4]), "=l"(d[5]), "=l"(d[6]), "=l"(d[7])
        : "r"(taddr) : "memory");
}

struct Probe1 { uint32_t wq, off, mode, info; };                     // query terms (first 32 tail terms, one per lane)
// + the terms' segments inside the tile.  Full-mode term: slot range [a, b).  Sparse-mode term (bit 31 of info):
// (a, b) = the (mask, seg_l2 index) entry of the tile's 32-tile group, turned into a slot range by resolve_segments (the
// batch kernel: after the previous row's head phase, so the entry's load and then the second-level loads are in flight
// behind other work).  info = the query's counts as ingest packs them into the fourth word of the tail32 entry: tail
// terms (19 bits) | cold head terms << 19 | hot head terms << 25 | the lane's sparse-mode flag << 31 — they come with the
// term in one 16-byte load (separate loads combined at probe time made the warp wait for them at the probe).
struct Probe2 { uint32_t a, b, wq; int32_t info; };

__device__ __forceinline__ Probe1 probe_terms(const TermParams& p, int64_t b, int lane) {
    const uint4 e = __ldg(p.tail32 + b * GS_TAIL32 + lane);
    return Probe1{e.x, e.y, e.z, e.w};
}
__device__ __forceinline__ Probe2 probe_segments(const TermParams& p, const Probe1& t, int tile) {
    Probe2 r;
    r.a = r.b = 0u;
    r.wq = t.wq; r.info = (int32_t)t.info;
    if (t.mode == GS_SEG_FULL) {
        r.a = __ldg(p.seg_tab + t.off + tile);
        r.b = __ldg(p.seg_tab + t.off + tile + 1);
    } else if (t.mode == GS_SEG_SPARSE) {
        const uint2 e = __ldg(p.seg_l1 + t.off + (tile >> 5));
        r.a = e.x; r.b = e.y;
    }
    return r;
}
__device__ __forceinline__ void resolve_segments(const TermParams& p, const Probe2& r, int tile, uint32_t& lo, uint32_t& hi) {
    lo = r.a; hi = r.b;
    if (r.info < 0) {
        const uint32_t bit = 1u << (tile & 31);
        if (lo & bit) {
            const uint32_t idx = hi + (uint32_t)__popc(lo & (bit - 1u));
            lo = __ldg(p.seg_l2 + idx);
            hi = __ldg(p.seg_l2 + idx + 1);
        } else {
            lo = hi = 0u;
        }
    }
}
__device__ __forceinline__ int info_tail(int32_t info) { return info & 0x7FFFF; }
__device__ __forceinline__ int info_cold(int32_t info) { return (info >> 19) & 0x3F; }
__device__ __forceinline__ int info_hot(int32_t info) { return (info >> 25) & 0x3F; }

__device__ __forceinline__ uint2 lds_u2(uint32_t addr) {
    uint2 v;
    asm("ld.shared.v2.u32 {%0, %1}, [%2];" : "=r"(v.x), "=r"(v.y) : "r"(addr));
    return v;
}

// Applies up to 32 posting-list segments (lane s: n postings from slot `start`, query weight bits wq) to `row`.
// `desc_s` = shared-window address of the warp's 32-entry descriptor table.
// `tag` (may be null): 512 bytes of shared memory owned by the warp, one per cell of the row — see the conflict pass below.
template <int WT>
__device__ __forceinline__ void scatter_flat(const TermParams& p, typename Num<WT>::A* row, uint32_t desc_s, int n,
                                             uint32_t start, uint32_t wq, int32_t base, int lane, uint8_t* tag = nullptr) {
    using W = typename Num<WT>::W;
    using A = typename Num<WT>::A;
    int incl = n;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const int v = __shfl_up_sync(0xFFFFFFFFu, incl, o);
        if (lane >= o) incl += v;
    }
    const int T = __shfl_sync(0xFFFFFFFFu, incl, 31);
    if (T == 0) return;
    const int excl = incl - n;
    const unsigned nz = __ballot_sync(0xFFFFFFFFu, n > 0);
    const unsigned lt = (1u << lane) - 1u, le = lt | (1u << lane);
    if (n > 0)
        asm volatile("st.shared.v2.u32 [%0], {%1, %2};" ::"r"(desc_s + 8u * (uint32_t)__popc(nz & lt)), "r"(start - (uint32_t)excl), "r"(wq) : "memory");
    __syncwarp();
    const int last_sg = __popc(nz) - 1;
    const int my_start = n > 0 ? excl : -0x40000000;   // flat position where the lane's segment starts (never matches when empty)
    int c0 = -1;                                   // (segments that start before the current round) - 1
    for (int f0 = 0; f0 < T; f0 += 32 * kRounds) {
        int32_t doc[kRounds];
        A wv[kRounds];
        uint32_t qv[kRounds];
        unsigned sm[kRounds];
        int ord[kRounds];
        // loads of up to kRounds rounds, no use of a loaded value in this loop (their latencies overlap); a lane past the
        // end of the stream re-reads the last posting and is switched off by ord = -1
#pragma unroll
        for (int r = 0; r < kRounds; ++r) {
            const int fr = f0 + 32 * r;
            if (fr < T) {                           // uniform
                const uint32_t d = (uint32_t)(my_start - fr);
                sm[r] = __reduce_or_sync(0xFFFFFFFFu, d < 32u ? (1u << d) : 0u);
                const int o = __popc(sm[r] & le);
                const bool valid = fr + lane < T;
                const int sg = valid ? c0 + o : last_sg;
                const int f = valid ? fr + lane : T - 1;
                ord[r] = valid ? o : -1;
                c0 += __popc(sm[r]);
                const uint2 de = lds_u2(desc_s + 8u * (uint32_t)sg);
                const uint32_t idx = de.x + (uint32_t)f;
                load_posting<WT>(p, idx, doc[r], wv[r]);
                qv[r] = de.y;
            }
        }
#pragma unroll
        for (int r = 0; r < kRounds; ++r) {
            if (f0 + 32 * r < T) {                  // uniform
                A* cell = row + (doc[r] - base);
                const A q = Num<WT>::qw(qv[r]), w = wv[r];
                if (tag != nullptr) {
                    // Two lists may hit the same document in one round (one list never does).  Every lane writes its lane
                    // number to the cell's tag byte; the lane whose number stays there owns the cell in this pass and
                    // does its read-modify-write, the others (rare) go round again.  One pass in the common case instead
                    // of one pass per list of the round.  Which lane a same-address store leaves behind is fixed-function
                    // arbitration: the same lane in every run, so the fp32 sums stay reproducible run to run.
                    uint8_t* tg = tag + (doc[r] - base);
                    bool todo = ord[r] >= 0;
                    while (__any_sync(0xFFFFFFFFu, todo)) {
                        if (todo) *reinterpret_cast<volatile uint8_t*>(tg) = (uint8_t)lane;
                        __syncwarp();
                        if (todo && *reinterpret_cast<volatile uint8_t*>(tg) == (uint8_t)lane) {
                            *cell = Num<WT>::mac(*cell, q, w);
                            todo = false;
                        }
                        __syncwarp();
                    }
                } else {
                    const int o_hi = __popc(sm[r]);
                    // segment by segment: two lists may hit the same document, one list never does
                    for (int o = (int)(sm[r] & 1u); o <= o_hi; ++o) {
                        if (ord[r] == o) *cell = Num<WT>::mac(*cell, q, w);
                        __syncwarp();
                    }
                }
            }
        }
    }
}



constexpr int kWarpBuf = 80;                  // candidate keys a warp collects in shared memory before it appends them
constexpr int kFlushAt = 40;                  // ... which it does at the end of a row once it holds more than this many
constexpr int kCandBuf = kBWarps * kWarpBuf;
// The fp32 batch kernel gives 16 KB of its shared memory to the cell tags of scatter_flat (227 KB per CTA, 192 KB of them rows
// and strips) and keeps a smaller candidate buffer; the integer kernel has room (strips are a quarter of the bytes) but its
// tail is faster with the per-list passes (same-box A/B: 12.44 vs 13.08 ms per batch), so it keeps them and the big buffer.
template <int WT> struct BatchGeo {
    static constexpr bool kTags = WT == GS_W_F32;
    static constexpr int kBuf = kTags ? 32 : kWarpBuf;
    static constexpr int kFlush = kBuf / 2;
    static constexpr size_t kTagBytes = kTags ? (size_t)kBWarps * 512 : 0;
    static constexpr size_t kFixed = (size_t)kBWarps * 32 * 8 + (size_t)kBWarps * kBuf * 10 + (size_t)(kBWarps + 4) * 4 + 32 + 128 + kTagBytes;
};

// ---- cold paths of the batch kernel, kept out of line: the kernel's warps sit in different phases of the row loop, so
// the loop body has to fit the instruction cache (a 116 KB variant of this kernel ran at half the speed of a 45 KB one).

// The warp appends its buffered candidates to the queries' lists (all the atomics of a round in flight together).  The
// buffer holds one run of entries per row the warp has finished: the first lane of a run reserves the whole run in its
// query's list with ONE atomic (same-address atomics of one warp instruction are served one after the other, each a round
// trip: 32 lanes on two or three counters cost tens of microseconds per flush).
__device__ __noinline__ void batch_flush(uint32_t* cand_cnt, uint64_t* cand, int64_t cand_cap, int64_t q0, const uint64_t* w_key,
                                         const uint16_t* w_q, uint32_t* w_cnt, int lane, int wbuf = kWarpBuf) {
    __syncwarp();
    const uint32_t n_buf = min(*reinterpret_cast<volatile uint32_t*>(w_cnt), (uint32_t)wbuf);
    const unsigned le_ = 0xFFFFFFFFu >> (31 - lane);
#pragma unroll 1
    for (uint32_t i0 = 0; i0 < n_buf; i0 += 32) {
        const uint32_t i = i0 + lane;
        const bool valid = i < n_buf;
        const uint32_t qi = valid ? (uint32_t)w_q[i] : 0xFFFFFFFFu;
        const uint32_t prev = __shfl_up_sync(0xFFFFFFFFu, qi, 1);
        const bool head = valid && (lane == 0 || qi != prev);
        const unsigned heads = __ballot_sync(0xFFFFFFFFu, head);
        const int n_valid = __popc(__ballot_sync(0xFFFFFFFFu, valid));
        const int start = 31 - __clz((int)(heads & le_));                 // first lane of this lane's run
        const unsigned later = heads & ~le_;
        const int end = later ? __ffs((int)later) - 1 : n_valid;          // one past the run's last lane
        const int64_t bb = q0 + (valid ? (int64_t)qi : 0);
        uint32_t pos = 0;
        if (head) pos = atomicAdd(&cand_cnt[bb * GS_CNT_STRIDE], (uint32_t)(end - lane));
        pos = __shfl_sync(0xFFFFFFFFu, pos, start & 31) + (uint32_t)(lane - start);
        if (valid && (int64_t)pos < cand_cap) cand[bb * cand_cap + pos] = w_key[i];
    }
    __syncwarp();
    if (lane == 0) *w_cnt = 0u;
    __syncwarp();
}

// One thread: the TMA bulk copies of a work item's strips (one 1-D copy per strip: kBT weights, contiguous in the strip)
// into shared memory, completing on the mbarrier at mbar_s.
// g = the first strip at the item's doc tile, ld = elements between strips
template <typename W>
__device__ __noinline__ void batch_issue_strips(const W* g, int64_t ld, int H, uint32_t strip_s, uint32_t mbar_s) {
    const uint32_t row_bytes = (uint32_t)(kBT * sizeof(W));
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(mbar_s), "r"(row_bytes * (uint32_t)H) : "memory");
#pragma unroll 1
    for (int h = 0; h < H; ++h)
        asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                     ::"r"(strip_s + (uint32_t)h * row_bytes), "l"(g + (size_t)h * ld), "r"(row_bytes), "r"(mbar_s) : "memory");
}

// Waits for a phase of an mbarrier.  The try_wait carries a suspend-time hint and a failed try is followed by a short sleep:
// a bare try_wait loop returned so often that the waiting warps executed 16 % of the kernel's instructions
// (profiles/r02_kernels.md), in issue slots the working warps of the SM need.
__device__ __forceinline__ void mbar_wait(uint32_t mbar_s, uint32_t parity) {
    uint32_t ok = 0;
    for (;;) {
        asm volatile("{ .reg .pred p; mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2, %3; selp.u32 %0, 1, 0, p; }"
                     : "=r"(ok) : "r"(mbar_s), "r"(parity), "r"(2000u) : "memory");
        if (ok) break;
        __nanosleep(200);
    }
}

// Every warp, once per work item, before its first head phase: waits for the item's strips (TMA, first mbarrier).  With
// TMEM: the strips landed, so every warp has left the previous item (its last warp out issued this copy) and tensor memory
// is free.  The first warp here copies the hot strips shared memory -> tensor memory: one tcgen05.cp.32x128b.warpx4 per
// (strip, 128 documents) moves 32 rows of 16 bytes and writes them to all four lane quarters; the copies complete on the
// second mbarrier, which every warp then waits for.  s_tmem: [0] TMEM base, [1..2] copy claimed (per parity).
template <bool TMEM, size_t OFF>
__device__ __noinline__ void batch_wait_strips(uint32_t mbar_s, uint32_t strip_s, uint32_t* s_tmem, int n_hot_strips, int par, int lane) {
    mbar_wait(mbar_s, (uint32_t)par);
    if (TMEM) {
        const uint32_t mbar2_s = mbar_s + 8u;
        uint32_t claimed = 0u;
        if (lane == 0) claimed = atomicExch(s_tmem + 1 + par, 1u) == 0u ? 1u : 0u;
        // The claiming warp runs the copy loop as a whole, every value a broadcast of lane 0's (so the compiler keeps the
        // descriptors in uniform registers: issued from a divergent lane each tcgen05.cp sat in a register-to-uniform
        // "waterfall" loop and the 128 copies took 8.8 K cycles), one elected lane issuing the copies.
        if (__shfl_sync(0xFFFFFFFFu, claimed, 0)) {
            if (lane == 0) s_tmem[1 + (par ^ 1)] = 0u;    // nobody claims the next item before this one's strips have landed
            const uint32_t t0 = __shfl_sync(0xFFFFFFFFu, s_tmem[0], 0);
            extern __shared__ __align__(16) unsigned char smem_raw[];
            const uint32_t ss = (uint32_t)__cvta_generic_to_shared(smem_raw) + (uint32_t)OFF;   // = strip_s, as a constant
            const int nhs = __shfl_sync(0xFFFFFFFFu, n_hot_strips, 0);
            asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
#pragma unroll 1
            for (int h = 0; h < nhs; ++h)
#pragma unroll
                for (int r = 0; r < 4; ++r) {
                    // shared-memory matrix descriptor, no swizzle: start address >> 4, leading byte offset (unused: one
                    // 16-byte column), stride byte offset 128 (8 rows of 16 bytes are contiguous) >> 4, version 1
                    const uint32_t a = ss + (uint32_t)(h * (kBT * 4) + r * 512);
                    const unsigned long long d = (unsigned long long)((a & 0x3FFFFu) >> 4) | (1ull << 16) | (8ull << 32) | (1ull << 46);
                    asm volatile("{ .reg .pred p; elect.sync _|p, 0xFFFFFFFF;\n\t@p tcgen05.cp.cta_group::1.32x128b.warpx4 [%0], %1; }"
                                 ::"r"(t0 + (uint32_t)(h * 16 + r * 4)), "l"(d) : "memory");
                }
            asm volatile("{ .reg .pred p; elect.sync _|p, 0xFFFFFFFF;\n\t@p tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0]; }"
                         ::"r"(mbar2_s) : "memory");
        }
        __syncwarp();
        mbar_wait(mbar2_s, (uint32_t)par);
        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    }
}

template <int WT>
__global__ void __launch_bounds__(kBWarps * 32, 1) k_score_term_batch(const TermParams p) {
    using W = typename Num<WT>::W;
    using A = typename Num<WT>::A;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    // shared memory: rows [kBWarps][kBT] | descriptors [kBWarps][32] uint2 | candidate keys [kBWarps][kWarpBuf] u64 |
    // candidate queries [kBWarps][kWarpBuf] u16 | counters (per-warp candidate counts, query counters and "warps done"
    // counters of the even / odd work items) | mbarrier | strips [H][kBT]
    constexpr size_t kOffDesc = (size_t)kBWarps * kBT * 4;
    constexpr size_t kOffKey = kOffDesc + (size_t)kBWarps * 32 * 8;
    constexpr int WB = BatchGeo<WT>::kBuf;                                   // candidate keys the warp buffers
    constexpr size_t kOffQ = kOffKey + (size_t)kBWarps * WB * 8;
    constexpr size_t kOffCnt = kOffQ + (size_t)kBWarps * WB * 2;
    constexpr size_t kOffBar = kOffCnt + (size_t)(kBWarps + 4) * 4;       // (32 bytes unused: the barriers are static, s_ctl)
    constexpr size_t kOffTag = kOffBar + 32;                                // cell tags
    constexpr size_t kOffStrip = (kOffTag + BatchGeo<WT>::kTagBytes + 127) / 128 * 128;   // [kBWarps][kBT] bytes (scatter_flat, fp32)
    A* row = reinterpret_cast<A*>(smem_raw) + (size_t)warp * kBT;
    const uint32_t desc_s = (uint32_t)__cvta_generic_to_shared(smem_raw + kOffDesc) + (uint32_t)warp * 256u;
    uint64_t* w_key = reinterpret_cast<uint64_t*>(smem_raw + kOffKey) + warp * WB;          // the warp's candidate buffer
    uint16_t* w_q = reinterpret_cast<uint16_t*>(smem_raw + kOffQ) + warp * WB;
    uint32_t* w_cnt = reinterpret_cast<uint32_t*>(smem_raw + kOffCnt) + warp;
    uint8_t* w_tag = BatchGeo<WT>::kTags ? smem_raw + kOffTag + (size_t)warp * kBT : nullptr;
    uint32_t* s_next = reinterpret_cast<uint32_t*>(smem_raw + kOffCnt) + kBWarps;           // [2]
    uint32_t* s_done = s_next + 2;                                                            // [2]
    W* s_strip = reinterpret_cast<W*>(smem_raw + kOffStrip);
    // mbarrier (strip copy) | mbarrier (TMEM copy) | TMEM base address, copy-claimed flags [2].  Static shared memory: with
    // these words in the dynamic block ptxas spilled three more values per row, and a spill reload is an L2 round trip
    // here (227 KB of the SM's 256 KB are shared memory: the streaming loads leave nothing of the L1 for the stack).
    __shared__ __align__(16) unsigned long long s_ctl[4];
    const uint32_t mbar_s = (uint32_t)__cvta_generic_to_shared(s_ctl);
    const uint32_t mbar2_s = mbar_s + 8u;
    uint32_t* s_tmem = reinterpret_cast<uint32_t*>(s_ctl + 2);                     // [0] TMEM base, [1..2] copy claimed (per parity)
    constexpr bool kTmem = WT == GS_W_F32;      // hot strips in tensor memory (fp32; the impact strips are a quarter of the bytes)
    // A work item = (doc tile, chunk of queries).  The CTA is persistent: it takes items blockIdx.x, blockIdx.x + gridDim.x, ...
    // The item's strips come in by TMA: one thread issues a 1-D bulk copy per strip (kBT weights, contiguous in the
    // strip) that completes on an mbarrier (one phase per item); a warp waits for it only before its first head phase.
    // A warp that finds no more rows in the item moves on to the next item's probes and tail scatter at once; the LAST
    // warp out of an item (shared-memory counter) starts the copy of the next item's strips — nobody reads the old ones
    // any more — so the copy, the item prologue and the slow warps' last rows overlap with the other warps' work.
    const int n_items = p.ts.count * p.n_chunks;
    const uint32_t strip_s = (uint32_t)__cvta_generic_to_shared(s_strip);
    auto item_strips = [&](int item) {
        return reinterpret_cast<const W*>(p.head_strip) + (size_t)(p.ts.first + (item / p.n_chunks) * p.ts.stride) * kBT;
    };
    if (lane == 0) *w_cnt = 0u;
    if (threadIdx.x == 0) {
        s_next[0] = s_next[1] = (uint32_t)kBWarps;
        s_done[0] = s_done[1] = 0u;
        asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(mbar_s) : "memory");
        asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(mbar2_s) : "memory");
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        s_tmem[1] = s_tmem[2] = 0u;
    }
    if (kTmem && warp == 0) {                           // the whole tensor memory of the SM (one CTA per SM)
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"((uint32_t)__cvta_generic_to_shared(s_tmem)), "n"(512));
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
    }
    if (kTmem) asm volatile("tcgen05.fence::before_thread_sync;");
    __syncthreads();
    if (kTmem) asm volatile("tcgen05.fence::after_thread_sync;");
    const uint32_t tmem_q = kTmem ? s_tmem[0] + ((uint32_t)(32 * (warp & 3)) << 16) : 0u;     // the warp's lane quarter
    const int n_hot_strips = min(p.H, GS_HOT_STRIPS);
    if (threadIdx.x == 0 && (int)blockIdx.x < n_items) batch_issue_strips<W>(item_strips((int)blockIdx.x), p.N_pad, p.H, strip_s, mbar_s);
    const bool filter = p.sink.thr != nullptr;
    const W* srow = s_strip + 4 * lane;
    int it = 0;
    for (int item = (int)blockIdx.x; item < n_items; item += (int)gridDim.x, ++it) {
    const int par = it & 1;
    const int j = item / p.n_chunks;
    const int chunk = item - j * p.n_chunks;
    const int tile = p.ts.first + j * p.ts.stride;
    const int32_t base = tile * kBT;
    bool strips_ready = false;
    // Queries are handed out dynamically (a row's cost varies with the query's tail lists): a warp starts with query
    // `warp` of the chunk and claims its next one from a shared-memory counter when it starts a row — ONE row ahead: the
    // next row's terms are probed during this row's tail phase, its segments during the head phase.  (Claiming three
    // rows ahead, to have deeper probes, left warps holding up to three unstarted rows at the end of an item while the
    // others waited: 27 K cycles between the first and the last warp out of an item, measured.)
    const int q_end = min(p.nq, (chunk + 1) * p.chunk);
    int q = chunk * p.chunk + warp;             // row being processed
    int q_n1 = q_end;                           // next row
    Probe2 s2{0u, 0u, 0u, 0};
    if (q < q_end) {
        s2 = probe_segments(p, probe_terms(p, p.q0 + q, lane), tile);
        resolve_segments(p, s2, tile, s2.a, s2.b);
    }
    const int n_live = (int)min((int64_t)kBT, p.N - (int64_t)base);                    // documents of this tile that exist
    for (; q < q_end; q = q_n1) {
        const int64_t b = p.q0 + q;
        const Probe2 cur = s2;
        {
            int c = 0;
            if (lane == 0) c = (int)atomicAdd(s_next + par, 1u);
            q_n1 = __shfl_sync(0xFFFFFFFFu, c, 0) + chunk * p.chunk;
        }
        Probe1 s1{0u, 0u, 0xFFFFFFFFu, 0u};
        if (q_n1 < q_end) s1 = probe_terms(p, p.q0 + q_n1, lane);
        const int n_hot = info_hot(cur.info), nh = n_hot + info_cold(cur.info), cnt = info_tail(cur.info);
        const int nx = p.xcnt != nullptr ? __ldg(p.xcnt + b) : 0;      // asked for now, used after the tail and head phases
        const uint64_t thr = filter ? __ldg(p.sink.thr + b) : 0ull;    // asked for now, used by the filter (not carried from row to row: registers)
        // fp32: the query's compact strip lists are loaded once, one entry per lane, and broadcast by shuffle in the head
        // phase (a load per strip put an L1 round trip in front of every strip); asked for now, so that the head phase
        // does not start with a wait for them
        uint2 e_hot = make_uint2(0u, 0u), e_cold = make_uint2(0u, 0u), e_x = make_uint2(0u, 0u);
        if (WT == GS_W_F32) {
            const uint2* hl0 = p.head_pair + b * GS_HEAD_MAX;
            if (lane < n_hot) e_hot = __ldg(hl0 + lane);
            if (lane < nh - n_hot) e_cold = __ldg(hl0 + (GS_HEAD_MAX - 1 - lane));
            if (p.xcnt != nullptr) e_x = __ldg(p.xpair + b * GS_XSTRIP_MAX + lane);    // entries past the query's count: unused
        }

#pragma unroll
        for (int r = 0; r < 4; ++r) reinterpret_cast<int4*>(row)[lane + 32 * r] = make_int4(0, 0, 0, 0);
        __syncwarp();
        scatter_flat<WT>(p, row, desc_s, (int)(cur.b - cur.a), cur.a, cur.wq, base, lane, w_tag);   // [a, b): resolved slot range
        if (cnt > GS_TAIL32) {                      // more than 32 tail terms: probed in line
            const int64_t qa = p.q_indptr[b];
            for (int i0 = GS_TAIL32; i0 < cnt; i0 += 32) {
                __syncwarp();                       // the descriptor table is reused
                uint4 d = make_uint4(0u, 0u, 0xFFFFFFFFu, 0u);
                if (i0 + lane < cnt) d = __ldg(p.tail_desc + qa + i0 + lane);
                uint32_t lo, hi;
                probe_range(p, d, tile, lo, hi);
                scatter_flat<WT>(p, row, desc_s, (int)(hi - lo), lo, d.x, base, lane, w_tag);
            }
        }
        __syncwarp();
        if (q_n1 < q_end) s2 = probe_segments(p, s1, tile);

        if (!strips_ready) {                        // once per warp and item
            batch_wait_strips<kTmem, kOffStrip>(mbar_s, strip_s, s_tmem, n_hot_strips, par, lane);
            strips_ready = true;
        }
        // head strips: the lane's 16 documents (quads lane, lane+32, lane+64, lane+96) stay in registers
        const uint2* hl = p.head_pair + b * GS_HEAD_MAX;
        A sc[4][4];
        if constexpr (WT == GS_W_F32) {
            unsigned long long acc[4][2];
#pragma unroll
            for (int r = 0; r < 4; ++r) {
                const ulonglong2 a2 = reinterpret_cast<const ulonglong2*>(row)[lane + 32 * r];
                acc[r][0] = a2.x; acc[r][1] = a2.y;
            }
            // hot strips: the lane's 16 documents of a strip in one tensor-memory load
#pragma unroll 2
            for (int i = 0; i < n_hot; ++i) {
                const float qf = __uint_as_float(__shfl_sync(0xFFFFFFFFu, e_hot.y, i));
                const unsigned long long q2 = pack_f32x2(qf, qf);
                unsigned long long t[8];
                tmem_ld16_wait(tmem_q + __shfl_sync(0xFFFFFFFFu, e_hot.x, i) * 16u, t);
#pragma unroll
                for (int r = 0; r < 4; ++r) {
                    acc[r][0] = fma_f32x2(t[2 * r], q2, acc[r][0]);
                    acc[r][1] = fma_f32x2(t[2 * r + 1], q2, acc[r][1]);
                }
            }
            // the other strips: shared memory
#pragma unroll 2
            for (int i = 0; i < nh - n_hot; ++i) {
                const float qf = __uint_as_float(__shfl_sync(0xFFFFFFFFu, e_cold.y, i));
                const unsigned long long q2 = pack_f32x2(qf, qf);
                const ulonglong2* src = reinterpret_cast<const ulonglong2*>(srow + (size_t)__shfl_sync(0xFFFFFFFFu, e_cold.x, i) * kBT);
                ulonglong2 v[4];
#pragma unroll
                for (int r = 0; r < 4; ++r) v[r] = src[32 * r];
#pragma unroll
                for (int r = 0; r < 4; ++r) {
                    acc[r][0] = fma_f32x2(v[r].x, q2, acc[r][0]);
                    acc[r][1] = fma_f32x2(v[r].y, q2, acc[r][1]);
                }
            }
            if (nx > 0) {                          // second-tier strips: same contraction, the strip read from global memory
                const uint2* xl = p.xpair + b * GS_XSTRIP_MAX;
                const float* gx = reinterpret_cast<const float*>(p.xstrip) + (size_t)base + 4 * lane;
#pragma unroll 1
                for (int i = 0; i < nx; ++i) {
                    uint2 e;
                    if (i < 32) { e.x = __shfl_sync(0xFFFFFFFFu, e_x.x, i); e.y = __shfl_sync(0xFFFFFFFFu, e_x.y, i); }
                    else e = __ldg(xl + i);
                    const float qf = __uint_as_float(e.y);
                    const unsigned long long q2 = pack_f32x2(qf, qf);
                    const ulonglong2* src = reinterpret_cast<const ulonglong2*>(gx + (size_t)e.x * (size_t)p.N_pad);
                    ulonglong2 v[4];
#pragma unroll
                    for (int r = 0; r < 4; ++r) v[r] = __ldg(src + 32 * r);
#pragma unroll
                    for (int r = 0; r < 4; ++r) {
                        acc[r][0] = fma_f32x2(v[r].x, q2, acc[r][0]);
                        acc[r][1] = fma_f32x2(v[r].y, q2, acc[r][1]);
                    }
                }
            }
#pragma unroll
            for (int r = 0; r < 4; ++r) {
                unpack_f32x2(acc[r][0], sc[r][0], sc[r][1]);
                unpack_f32x2(acc[r][1], sc[r][2], sc[r][3]);
            }
        } else {
#pragma unroll
            for (int r = 0; r < 4; ++r) {
                const int4 a4 = reinterpret_cast<const int4*>(row)[lane + 32 * r];
                sc[r][0] = a4.x; sc[r][1] = a4.y; sc[r][2] = a4.z; sc[r][3] = a4.w;
            }
#pragma unroll kHeadUnroll
            for (int i = 0; i < nh; ++i) {
                const uint2 e = head_entry(hl, i, n_hot);
                // one IDP4A per cell: the impact byte of the query (<= 255) placed in byte u of the second operand picks
                // byte u of the strip word — no unpacking
                const uint32_t qi = e.y & 0xFFu;
                const uint32_t* src = reinterpret_cast<const uint32_t*>(srow + (size_t)e.x * kBT);
                uint32_t v[4];
#pragma unroll
                for (int r = 0; r < 4; ++r) v[r] = src[32 * r];
#pragma unroll
                for (int r = 0; r < 4; ++r)
#pragma unroll
                    for (int u = 0; u < 4; ++u) sc[r][u] = (int32_t)__dp4a(v[r], qi << (8 * u), (uint32_t)sc[r][u]);
            }
            if (nx > 0) {
                const uint2* xl = p.xpair + b * GS_XSTRIP_MAX;
                const uint8_t* gx = reinterpret_cast<const uint8_t*>(p.xstrip) + (size_t)base + 4 * lane;
#pragma unroll 1
                for (int i = 0; i < nx; ++i) {
                    const uint2 e = __ldg(xl + i);
                    const uint32_t qi = e.y & 0xFFu;
                    const uint32_t* src = reinterpret_cast<const uint32_t*>(gx + (size_t)e.x * (size_t)p.N_pad);
                    uint32_t v[4];
#pragma unroll
                    for (int r = 0; r < 4; ++r) v[r] = __ldg(src + 32 * r);
#pragma unroll
                    for (int r = 0; r < 4; ++r)
#pragma unroll
                        for (int u = 0; u < 4; ++u) sc[r][u] = (int32_t)__dp4a(v[r], qi << (8 * u), (uint32_t)sc[r][u]);
                }
            }
        }

        // the next row's sparse-mode entries have arrived during the head phase: their second-level lookups are issued
        // now and land during the filter and the next row's zeroing, so the row starts on resolved slot ranges
        if (q_n1 < q_end) resolve_segments(p, s2, tile, s2.a, s2.b);

        if (!filter) {
#pragma unroll
            for (int r = 0; r < 4; ++r) {
                const int dq = lane + 32 * r;
                store_quad<WT>(p, b, j, dq, (int64_t)base + 4 * dq, sc[r][0], sc[r][1], sc[r][2], sc[r][3]);
            }
            continue;
        }
        // Score and doc id of the threshold key: key >= threshold key  <=>  score > its score, or equal and doc id <= its
        // doc id.  Threshold key 0 = accept everything.  A cell that passes goes to the CTA's candidate buffer in shared
        // memory (one shared-memory atomic per candidate; the global append — an atomic whose result must come back —
        // happens once per CTA, all entries in flight together); when the buffer is full the cell is appended directly.
        const A thr_s = thr == 0ull ? Num<WT>::lowest()
                                    : Num<WT>::from_bits((int)(WT == GS_W_F32 ? gs_unord_f32((uint32_t)(thr >> 32))
                                                                              : ((uint32_t)(thr >> 32) ^ 0x80000000u)));
        const int64_t thr_cell = (int64_t)(0xFFFFFFFFu - (uint32_t)thr) - (int64_t)base;   // threshold doc as a cell of this tile
        const int tie_cells = (int)max((int64_t)-1, min((int64_t)kBT, thr_cell));           // cells <= this index win a score tie
        // bit 4r+u of `hit`: the lane's cell (r, u) reaches the threshold score.  A row has a few such cells, spread over the
        // lanes: testing them one unrolled cell at a time made the warp run the emission body once per distinct (r, u)
        // position with a hit (3.7 times per row); with the mask it runs once per hit of the busiest lane (1-2 times).
        uint32_t hit = 0u;
#pragma unroll
        for (int r = 0; r < 4; ++r)
#pragma unroll
            for (int u = 0; u < 4; ++u) hit |= sc[r][u] >= thr_s ? 1u << (4 * r + u) : 0u;
        if (hit) {
            // the lane's scores go back to its own cells of the row (nobody else reads them) to be picked by index
#pragma unroll
            for (int r = 0; r < 4; ++r)
                reinterpret_cast<uint4*>(row)[lane + 32 * r] = make_uint4(Num<WT>::bits(sc[r][0]), Num<WT>::bits(sc[r][1]),
                                                                         Num<WT>::bits(sc[r][2]), Num<WT>::bits(sc[r][3]));
#pragma unroll 1
            while (hit) {
                const int i = __ffs((int)hit) - 1;
                hit &= hit - 1u;
                const int cell = 4 * (lane + 32 * (i >> 2)) + (i & 3);
                const A v = row[cell];
                if (cell < n_live && (v > thr_s || cell <= tie_cells)) {
                    const uint64_t key = gs_make_key(gs_ord_bits<WT>(Num<WT>::bits(v)), (uint32_t)(base + cell));
                    const uint32_t slot = atomicAdd(w_cnt, 1u);
                    if (slot < (uint32_t)WB) {
                        w_key[slot] = key;
                        w_q[slot] = (uint16_t)q;
                    } else {                                             // buffer full: append directly
                        const uint32_t pos = atomicAdd(&p.sink.cand_cnt[b * GS_CNT_STRIDE], 1u);
                        if ((int64_t)pos < p.sink.cand_cap) p.sink.cand[b * p.sink.cand_cap + pos] = key;
                    }
                }
            }
        }
        __syncwarp();
        if (*reinterpret_cast<volatile uint32_t*>(w_cnt) > (uint32_t)BatchGeo<WT>::kFlush)
            batch_flush(p.sink.cand_cnt, p.sink.cand, p.sink.cand_cap, p.q0, w_key, w_q, w_cnt, lane, WB);
    }
    // out of rows in this item.  Every warp observes every phase of the mbarrier (a warp without rows too: a wait for the
    // NEXT phase issued while this one is still pending would be satisfied at once), then reports itself done.
    if (!strips_ready) batch_wait_strips<kTmem, kOffStrip>(mbar_s, strip_s, s_tmem, n_hot_strips, par, lane);
    __syncwarp();
    if (kTmem) asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");    // the warp's tensor-memory loads are done
    if (lane == 0) {
        __threadfence_block();
        if (atomicAdd(s_done + par, 1u) == (uint32_t)(kBWarps - 1)) {       // last warp out: the strips buffer is free
            s_done[par] = 0u;
            s_next[par] = (uint32_t)kBWarps;                                   // for the item after the next
            if (item + (int)gridDim.x < n_items) batch_issue_strips<W>(item_strips(item + (int)gridDim.x), p.N_pad, p.H, strip_s, mbar_s);
        }
    }
    __syncwarp();
    }
    if (filter) batch_flush(p.sink.cand_cnt, p.sink.cand, p.sink.cand_cap, p.q0, w_key, w_q, w_cnt, lane, WB);
    if (kTmem) {
        asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
        __syncthreads();
        if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(s_tmem[0]), "n"(512));
    }
}

// ------------------------------------------------------------------------------------------------
// Integer-impact mode, batches: the head contraction on the TENSOR CORES.  The strips of a doc tile are a
// genuinely dense block: scores_head[512 docs x B queries] = S[512 x 192 strips] * Q[192 x B], uint8 x uint8 -> int32, which
// tcgen05.mma kind::i8 computes exactly (integer addition is associative: bit-identical to the IDP4A path and to the
// oracle).  The fp32 path does not use this: its products would have to be rounded (PAPER.md keeps fp32, L75/L165).
//
// One persistent CTA of 32 warps per SM walks (doc tile, query chunk) items; inside an item, groups of 32 queries:
//   * A operand: the tile's strips in the K-major core-matrix layout (gs_index::mma_strips), 96 KB, one TMA bulk copy per
//     128-document sub-tile, once per item; B operand: the group's query impacts as a dense 32 x 192 uint8 matrix, built
//     in shared memory from the compact strip lists (double buffered); D: 4 sub-tiles x (128 docs x 32 queries) int32 =
//     128 columns of tensor memory, four groups deep, so the 24 MMAs of group g+1 are issued (by one thread) while the
//     warps still work on group g;
//   * tail: warp w owns the row of query w of the group (shared memory, 2 KB) and scatters the query's tail lists into
//     it with the flat posting stream of the batch kernel (scatter_flat) — no atomics, fixed order;
//   * epilogue (replaces the head phase: ~60 instead of ~300 instructions per row): warp w reads, for its lane quarter
//     (documents 32(w%4) .. +31 of every sub-tile) and its 4 queries (4(w/4) .. +3), the head scores from tensor memory
//     (tcgen05.ld.32x32b.x4: lane = document, columns = queries), adds the tail rows (conflict-free: consecutive lanes are
//     consecutive documents) and hands the cells to the sink (dense store or threshold filter).
// Synchronisation is by TEAMS of four warps: the rows of queries 4t .. 4t+3 are written by warps 4t .. 4t+3 and read by the
// same four warps (one lane quarter each), so two named barriers of 128 threads per group replace CTA barriers and the
// teams drift apart freely (a CTA barrier made every group as slow as its slowest of 32 rows: 19.2 ms per batch against
// 13.9 ms on the CUDA cores).  The B operand of a group is complete when all 32 warps have written their row: the last
// one to arrive (shared-memory counter) issues the group's MMAs.
// ------------------------------------------------------------------------------------------------
constexpr int kMQ = 32;                                     // queries per group = N of the MMA = warps of the CTA
constexpr size_t kMOffDesc = (size_t)kMQ * kBT * 4;         // rows [32][512] int32 | flat-stream descriptors [32][32] uint2
constexpr size_t kMOffKey = kMOffDesc + (size_t)kMQ * 32 * 8;
constexpr size_t kMOffQ = kMOffKey + (size_t)kCandBuf * 8;
constexpr size_t kMOffCnt = kMOffQ + (size_t)kCandBuf * 2;
constexpr size_t kMOffBar = kMOffCnt + (size_t)(kMQ + 4) * 4;   // mbarrier A | mbarrier MMA [4] | tensor-memory base
constexpr size_t kMOffB = (kMOffBar + 64 + 127) / 128 * 128;    // B operand [4][GS_MMA_K/16][4][8][16]
constexpr size_t kMBBytes = (size_t)(GS_MMA_K / 16) * 4 * 128;
constexpr int kMLook = 3;                                       // groups whose B operand and MMAs run ahead of the rows
constexpr size_t kMOffA = kMOffB + 4 * kMBBytes;                // A operand [4][GS_MMA_K/16][16][8][16]
constexpr size_t kMABytes = (size_t)4 * (GS_MMA_K / 16) * 2048;
constexpr size_t kMSmem = kMOffA + kMABytes;
static_assert(kMOffBar % 8 == 0 && kMOffA % 128 == 0, "alignment");

// shared-memory matrix descriptor, K-major, no swizzle: start address >> 4 | leading byte offset (between core matrices
// along K) >> 4 << 16 | stride byte offset (between 8-row groups along M/N) >> 4 << 32 | version 1 << 46
__device__ __forceinline__ unsigned long long umma_desc(uint32_t saddr, uint32_t lbo, uint32_t sbo) {
    return (unsigned long long)((saddr & 0x3FFFFu) >> 4) | ((unsigned long long)(lbo >> 4) << 16) |
           ((unsigned long long)(sbo >> 4) << 32) | (1ull << 46);
}

// One thread: the 24 MMAs of a group, D[sub-tile s] (128 x 32, int32, tensor memory) = A_s (128 x 192) * B^T (32 x 192),
// and the commit that makes their completion arrive on an mbarrier.
__device__ __noinline__ void mma_issue_group(uint32_t a_s, uint32_t b_s, uint32_t d_tmem, uint32_t mbar) {
    // instruction descriptor: D int32 (2 << 4), A and B unsigned 8 bit (0 << 7, 0 << 10), both K-major, N = 32 (>> 3 << 17),
    // M = 128 (>> 4 << 24)
    constexpr uint32_t idesc = (2u << 4) | ((uint32_t)(kMQ >> 3) << 17) | ((uint32_t)(128 >> 4) << 24);
#pragma unroll 1
    for (int s = 0; s < 4; ++s)
#pragma unroll 1
        for (int j = 0; j < GS_MMA_K / 32; ++j) {
            const unsigned long long ad = umma_desc(a_s + (uint32_t)(s * (GS_MMA_K / 16) * 2048 + j * 2 * 2048), 2048u, 128u);
            const unsigned long long bd = umma_desc(b_s + (uint32_t)(j * 2 * 512), 512u, 128u);
            const uint32_t acc = j > 0 ? 1u : 0u;
            asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
                         "tcgen05.mma.cta_group::1.kind::i8 [%0], %1, %2, %3, p;\n\t}"
                         ::"r"(d_tmem + (uint32_t)(s * kMQ)), "l"(ad), "l"(bd), "r"(idesc), "r"(acc) : "memory");
        }
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(mbar) : "memory");
}

// One thread: the item's A operand, one bulk copy per sub-tile
__device__ __noinline__ void mma_issue_a(const uint8_t* g, uint32_t a_s, uint32_t mbar) {
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(mbar), "r"((uint32_t)kMABytes) : "memory");
#pragma unroll 1
    for (int s = 0; s < 4; ++s)
        asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                     ::"r"(a_s + (uint32_t)(s * (kMABytes / 4))), "l"(g + (size_t)s * (kMABytes / 4)), "r"((uint32_t)(kMABytes / 4)), "r"(mbar) : "memory");
}

__global__ void __launch_bounds__(kMQ * 32, 1) k_score_term_mma(const TermParams p) {
    constexpr int WT = GS_W_U8;
    using A = int32_t;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    A* rows = reinterpret_cast<A*>(smem_raw);
    A* row = rows + (size_t)warp * kBT;
    const uint32_t desc_s = (uint32_t)__cvta_generic_to_shared(smem_raw + kMOffDesc) + (uint32_t)warp * 256u;
    uint64_t* w_key = reinterpret_cast<uint64_t*>(smem_raw + kMOffKey) + warp * kWarpBuf;
    uint16_t* w_q = reinterpret_cast<uint16_t*>(smem_raw + kMOffQ) + warp * kWarpBuf;
    uint32_t* w_cnt = reinterpret_cast<uint32_t*>(smem_raw + kMOffCnt) + warp;
    uint32_t* s_bcnt = reinterpret_cast<uint32_t*>(smem_raw + kMOffCnt) + kMQ;       // [4] warps that have written their B row
    const uint32_t mbar_a = (uint32_t)__cvta_generic_to_shared(smem_raw + kMOffBar);
    const uint32_t mbar_m = mbar_a + 8u;                                            // [4]
    uint32_t* s_tmem = reinterpret_cast<uint32_t*>(smem_raw + kMOffBar + 40);
    volatile uint32_t* s_issue = s_tmem + 1;                                         // next group whose MMAs are to be issued
    uint8_t* s_b = smem_raw + kMOffB;
    const uint32_t b_s = (uint32_t)__cvta_generic_to_shared(s_b);
    const uint32_t a_s = (uint32_t)__cvta_generic_to_shared(smem_raw + kMOffA);
    const bool filter = p.sink.thr != nullptr;
    const int n_items = p.ts.count * p.n_chunks;
    auto item_a = [&](int item) {
        return p.mma_strips + (size_t)(p.ts.first + (item / p.n_chunks) * p.ts.stride) * kMABytes;
    };
    if (lane == 0) *w_cnt = 0u;
    if (threadIdx.x == 0) {
        s_bcnt[0] = s_bcnt[1] = s_bcnt[2] = s_bcnt[3] = 0u;
        *s_issue = 0u;
        asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(mbar_a) : "memory");
        for (int i = 0; i < 4; ++i) asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(mbar_m + 8u * i) : "memory");
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == 0) {                                    // the whole tensor memory of the SM (one CTA per SM)
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"((uint32_t)__cvta_generic_to_shared(s_tmem)), "n"(512));
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
    }
    asm volatile("tcgen05.fence::before_thread_sync;");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;");
    const uint32_t tmem0 = s_tmem[0];
    if (threadIdx.x == 0 && (int)blockIdx.x < n_items) mma_issue_a(item_a((int)blockIdx.x), a_s, mbar_a);

    // B operand of the group whose first query is qs: warp w writes row w (query qs + w): zeros, then the query's impacts at
    // the columns of its strips (head strip h -> column h, second-tier strip x -> column 64 + x)
    auto build_b = [&](int qs, int q_end, int buf) {
        uint8_t* bb = s_b + (size_t)buf * kMBBytes + (size_t)(warp >> 3) * 128 + (size_t)(warp & 7) * 16;    // + (k >> 4) * 512 + (k & 15)
        if (lane < GS_MMA_K / 16) *reinterpret_cast<uint4*>(bb + lane * 512) = make_uint4(0u, 0u, 0u, 0u);
        __syncwarp();
        const int q = qs + warp;
        if (q < q_end) {
            const int64_t b = p.q0 + q;
            const int hc = __ldg(p.head_cnt + b);
            const int nh = hc & 0xFF, n_hot = hc >> 8;
            const int nx = p.xcnt != nullptr ? __ldg(p.xcnt + b) : 0;
            const uint2* hl = p.head_pair + b * GS_HEAD_MAX;
            if (lane < n_hot) { const uint2 e = __ldg(hl + lane); bb[(e.x >> 4) * 512 + (e.x & 15)] = (uint8_t)e.y; }
            if (lane < nh - n_hot) { const uint2 e = __ldg(hl + (GS_HEAD_MAX - 1 - lane)); bb[(e.x >> 4) * 512 + (e.x & 15)] = (uint8_t)e.y; }
            for (int i = lane; i < nx; i += 32) {
                const uint2 e = __ldg(p.xpair + b * GS_XSTRIP_MAX + i);
                const uint32_t k = GS_STRIP_MAX + e.x;
                bb[(k >> 4) * 512 + (k & 15)] = (uint8_t)e.y;
            }
        }
    };

    uint32_t G = 0;                                     // groups done by this CTA: tensor-memory buffer G & 3, phase (G >> 2) & 1
    int it = 0;
    for (int item = (int)blockIdx.x; item < n_items; item += (int)gridDim.x, ++it) {
        const int j = item / p.n_chunks;
        const int chunk = item - j * p.n_chunks;
        const int tile = p.ts.first + j * p.ts.stride;
        const int32_t base = tile * kBT;
        const int q_beg = chunk * p.chunk;
        const int q_end = min(p.nq, (chunk + 1) * p.chunk);
        const int n_groups = (q_end - q_beg + kMQ - 1) / kMQ;
        const int n_live = (int)min((int64_t)kBT, p.N - (int64_t)base);
        // B row of the warp's query of group X (first query qs); the last warp to arrive issues the group's MMAs — after
        // the item's strips have landed when X is the item's first group — and, when X is the item's last group, waits
        // for them and starts the copy of the next item's strips (nobody reads the old ones any more)
        auto b_ready = [&](uint32_t X, int qs, bool /*first*/, bool last) {
            build_b(qs, q_end, (int)(X & 3u));
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
            __syncwarp();
            if (lane == 0) {
                __threadfence_block();
                if (atomicAdd(s_bcnt + (X & 3u), 1u) == (uint32_t)(kMQ - 1)) {
                    s_bcnt[X & 3u] = 0u;
                    __threadfence_block();
                    while (*s_issue != X) {}              // groups are issued in order (the strips of the next item follow the last one)
                    mbar_wait(mbar_a, (uint32_t)(it & 1));
                    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
                    mma_issue_group(a_s, b_s + (X & 3u) * (uint32_t)kMBBytes, tmem0 + (X & 3u) * 128u, mbar_m + 8u * (X & 3u));
                    if (last && item + (int)gridDim.x < n_items) {
                        mbar_wait(mbar_m + 8u * (X & 3u), (X >> 2) & 1u);
                        mma_issue_a(item_a(item + (int)gridDim.x), a_s, mbar_a);
                    }
                    __threadfence_block();
                    *s_issue = X + 1u;
                }
            }
            __syncwarp();
        };
        for (int x = 0; x < min(kMLook, n_groups); ++x) b_ready(G + (uint32_t)x, q_beg + x * kMQ, x == 0, x + 1 == n_groups);
        // probes of the warp's query of the first group (terms -> segment tables), the next group's are asked for one group ahead
        Probe2 s2{0u, 0u, 0u, 0};
        if (q_beg + warp < q_end) s2 = probe_segments(p, probe_terms(p, p.q0 + q_beg + warp, lane), tile);
#pragma unroll 1
        for (int g = 0; g < n_groups; ++g, ++G) {
            const int qg = q_beg + g * kMQ;
            const int q = qg + warp;
            const Probe2 cur = s2;
            if (q + kMQ < q_end) s2 = probe_segments(p, probe_terms(p, p.q0 + q + kMQ, lane), tile);
            // ---- tail: the row of query q
#pragma unroll
            for (int r = 0; r < 4; ++r) reinterpret_cast<int4*>(row)[lane + 32 * r] = make_int4(0, 0, 0, 0);
            __syncwarp();
            if (q < q_end) {
                const int cnt = info_tail(cur.info);
                uint32_t lo, hi;
                resolve_segments(p, cur, tile, lo, hi);
                scatter_flat<WT>(p, row, desc_s, (int)(hi - lo), lo, cur.wq, base, lane);
                if (cnt > GS_TAIL32) {                  // more than 32 tail terms: probed in line
                    const int64_t qa = p.q_indptr[p.q0 + q];
                    for (int i0 = GS_TAIL32; i0 < cnt; i0 += 32) {
                        __syncwarp();                   // the descriptor table is reused
                        uint4 d = make_uint4(0u, 0u, 0xFFFFFFFFu, 0u);
                        if (i0 + lane < cnt) d = __ldg(p.tail_desc + qa + i0 + lane);
                        probe_range(p, d, tile, lo, hi);
                        scatter_flat<WT>(p, row, desc_s, (int)(hi - lo), lo, d.x, base, lane);
                    }
                }
            }
            // ---- B of the next group; then the team's four rows are complete
            if (g + kMLook < n_groups) b_ready(G + (uint32_t)kMLook, qg + kMLook * kMQ, false, g + kMLook + 1 == n_groups);
            asm volatile("bar.sync %0, 128;" ::"r"(1 + (warp >> 2)) : "memory");
            // ---- epilogue of group g: head scores from tensor memory + tail rows -> sink
            mbar_wait(mbar_m + 8u * (G & 3u), (G >> 2) & 1u);
            asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
            {
                const int k4 = warp & 3, gq = warp >> 2;
                A thr_s[4];
                int tie[4];
                bool okq[4];
#pragma unroll
                for (int u = 0; u < 4; ++u) {
                    const int qq = qg + 4 * gq + u;
                    okq[u] = qq < q_end;
                    const uint64_t thr = (filter && okq[u]) ? __ldg(p.sink.thr + p.q0 + qq) : 0ull;
                    thr_s[u] = thr == 0ull ? Num<WT>::lowest() : (A)((uint32_t)(thr >> 32) ^ 0x80000000u);
                    const int64_t thr_cell = (int64_t)(0xFFFFFFFFu - (uint32_t)thr) - (int64_t)base;
                    tie[u] = (int)max((int64_t)-1, min((int64_t)kBT, thr_cell));
                }
#pragma unroll 1
                for (int s = 0; s < 4; ++s) {
                    uint32_t v[4];
                    asm volatile("tcgen05.ld.sync.aligned.32x32b.x4.b32 {%0,%1,%2,%3}, [%4];\n\ttcgen05.wait::ld.sync.aligned;"
                                 : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3])
                                 : "r"(tmem0 + ((uint32_t)(32 * k4) << 16) + (G & 3u) * 128u + (uint32_t)(s * kMQ + 4 * gq)) : "memory");
                    const int cell = 128 * s + 32 * k4 + lane;
#pragma unroll
                    for (int u = 0; u < 4; ++u) {
                        if (!okq[u]) continue;
                        const int qq = qg + 4 * gq + u;
                        const A sc = (A)v[u] + rows[(size_t)(4 * gq + u) * kBT + cell];
                        const int64_t b = p.q0 + qq;
                        if (!filter) {
                            if ((int64_t)base + cell < p.N) p.sink.dense[(b - p.q0) * p.sink.ld + (int64_t)j * kBT + cell] = (uint32_t)sc;
                        } else if (sc >= thr_s[u] && cell < n_live && (sc > thr_s[u] || cell <= tie[u])) {
                            const uint64_t key = gs_make_key(gs_ord_bits<WT>((uint32_t)sc), (uint32_t)(base + cell));
                            const uint32_t slot = atomicAdd(w_cnt, 1u);
                            if (slot < (uint32_t)kWarpBuf) {
                                w_key[slot] = key;
                                w_q[slot] = (uint16_t)qq;
                            } else {                                         // buffer full: append directly
                                const uint32_t pos = atomicAdd(&p.sink.cand_cnt[b * GS_CNT_STRIDE], 1u);
                                if ((int64_t)pos < p.sink.cand_cap) p.sink.cand[b * p.sink.cand_cap + pos] = key;
                            }
                        }
                    }
                }
            }
            __syncwarp();
            if (filter && *reinterpret_cast<volatile uint32_t*>(w_cnt) > (uint32_t)kFlushAt)
                batch_flush(p.sink.cand_cnt, p.sink.cand, p.sink.cand_cap, p.q0, w_key, w_q, w_cnt, lane);
            asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
            asm volatile("bar.sync %0, 128;" ::"r"(1 + (warp >> 2)) : "memory");      // the team's rows are free
        }
    }
    if (filter) batch_flush(p.sink.cand_cnt, p.sink.cand, p.sink.cand_cap, p.q0, w_key, w_q, w_cnt, lane);
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem0), "n"(512));
}

// launches of at most this many cell rows prefetch their strips into the L2 at row start (process_item); 1024 and 4096
// measured alike: single-query search 0.1375 -> 0.1336 ms of scoring, Zipf-1.3 collection 0.832 -> 0.811, integer 0.107 -> 0.103
constexpr int64_t kPfRowsMax = 1024;
int norm_warps(int w) { return w <= 0 ? kWarpsDefault : std::min(w, kWarpsMax); }

template <int WT, bool XS>
gs_status_t launch_x(const TermParams& p, unsigned grid, size_t smem, bool staged, cudaStream_t s) {
    if (staged) {
        GS_CUDA(gs_optin_smem(k_score_term_staged<WT, XS>));
        GsProfScope ps(GS_K_SCORE_TERM, s);
        k_score_term_staged<WT, XS><<<grid, kWarpsStaged * 32, smem, s>>>(p);
    } else {
        GS_CUDA(gs_optin_smem(k_score_term<WT, XS>));
        GsProfScope ps(GS_K_SCORE_TERM, s);
        TermParams pp = p;
        pp.pf_rows = (int64_t)p.ts.count * p.nq <= kPfRowsMax ? 1 : 0;
        k_score_term<WT, XS><<<grid, p.warps * 32, smem, s>>>(pp);
    }
    ++gs_tls_launches;
    GS_CUDA(cudaGetLastError());
    return GS_OK;
}
// the second-tier strip loop is compiled in only when the batch carries x lists (it costs the small kernel 16 registers)
template <int WT>
gs_status_t launch(const TermParams& p, unsigned grid, size_t smem, bool staged, cudaStream_t s) {
    return p.xcnt != nullptr ? launch_x<WT, true>(p, grid, smem, staged, s) : launch_x<WT, false>(p, grid, smem, staged, s);
}

// From how many queries on the CTA-per-doc-tile kernels are used.  Batch sweep on B200 (ms per batch, warp-per-row shape vs
// batch kernel): 8.8M docs 48: 3.03 / 3.19, 64: 3.89 / 3.37, 128: 7.25 / 5.51, 256: 13.7 / 9.49, 500: 25.9 / 16.6;
// 1M docs 64: 0.61 / 0.62, 96: 0.84 / 0.88, 128: 1.04 / 0.98, 256: 1.87 / 1.53, 500: 3.41 / 2.59 — the fixed cost of a CTA
// (staging, first-row probes) is amortised over fewer rows when the collection has few doc tiles.
// batches of at least this many queries take the batch / staged kernels (one CTA of 32 warps per doc tile and query chunk);
// measured on B200 after the round-2 cuts of the batch kernel: it wins from one query per warp on, on every collection
// size (8.8M docs: B = 32 1.94 -> 1.77 ms, config 5 B = 32 9.60 -> 8.63 ms; 1M docs B = 64 0.476 -> 0.442 ms), and loses
// below (B = 24: 1.45 vs 1.67 ms)
constexpr int kStagedMinQueries = 32;
constexpr int kStagedChunk = 512;         // most queries per CTA of the staged / batch kernels
constexpr int kChunkWaves = 16;   // CTAs per SM a launch aims for before it stops splitting the queries
static inline bool cta_per_tile(const gs_index* ix, int64_t nq) {
    (void)ix;
    return nq >= kStagedMinQueries;
}

}  // namespace

bool gs_score_term_wants_x(const gs_index* ix, int64_t nq, int group, bool use_head) {
    return group == 0 && cta_per_tile(ix, nq) && use_head && ix->H > 0 && ix->HX > 0 && ix->Ts == kBT;
}

int gs_score_term_group(const gs_index* ix, int64_t nq, int group, bool use_head) {
    if (group == 0 && cta_per_tile(ix, nq) && use_head && ix->H > 0 && ix->Ts == kBT)
        return kBWarps;                                                 // batch kernel
    if (group <= 0 && cta_per_tile(ix, nq) && use_head && ix->H > 0) return kWarpsStaged;
    return norm_warps(group);
}

gs_status_t gs_launch_score_term(const gs_index* ix, const gs_qbatch& qb, int64_t q0, int64_t nq, int group,
                                 bool use_head, bool use_mma, const gs_tileset& ts, const gs_sink& sink, cudaStream_t s) {
    if (nq <= 0 || ts.count <= 0) return GS_OK;
    TermParams p{};
    p.inv_doc = ix->inv_doc; p.inv_w = ix->inv_w; p.inv_pk = ix->inv_packed ? ix->inv_pk : nullptr; p.seg_tab = ix->seg_tab; p.seg_l1 = ix->seg_l1; p.seg_l2 = ix->seg_l2;
    p.head_strip = ix->head_strip; p.H = use_head ? ix->H : 0; p.N = ix->N; p.N_pad = ix->N_pad; p.Ts = ix->Ts;
    p.ntiles = ix->ntiles;
    p.q_indptr = qb.indptr; p.head_pair = qb.head_pair; p.head_cnt = qb.head_cnt; p.tail_desc = qb.tail_desc;
    p.tail_cnt = qb.tail_cnt; p.tail32 = qb.tail32;
    p.xstrip = qb.x_on ? ix->xstrip : nullptr; p.xpair = qb.x_on ? qb.xpair : nullptr; p.xcnt = qb.x_on ? qb.xcnt : nullptr;
    p.q0 = q0; p.nq = (int32_t)nq;
    p.warps = norm_warps(group);
    p.ts = ts; p.sink = sink;
    p.vec4 = sink.dense && (((uintptr_t)sink.dense | (uintptr_t)(sink.ld * 4)) & 15) == 0;
    int dev = 0, smem_max = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&smem_max, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
    const size_t wbytes = ix->wtype == GS_W_F32 ? 4 : 1;
    const size_t smem_staged = (size_t)kWarpsStaged * ix->Ts * 4 + (size_t)p.H * ix->Ts * wbytes;
    // query_group > 0 pins the small-batch kernel (that many cell rows per CTA); -1 pins the generic staged kernel
    if (group <= 0 && cta_per_tile(ix, nq) && p.H > 0 && smem_staged <= (size_t)smem_max) {
        // queries per CTA: all of them (up to kStagedChunk) when the doc tiles alone fill the machine many times over;
        // a launch over few tiles (the threshold sample, a small collection) splits the queries so that the grid still
        // has about kChunkWaves CTAs per SM, down to one cell row per warp
        int sms = 148;
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
        const int64_t want = ((int64_t)kChunkWaves * sms + ts.count - 1) / ts.count;
        const int64_t most = std::max<int64_t>(1, nq / kWarpsStaged);
        int64_t n_chunks = std::max<int64_t>((nq + kStagedChunk - 1) / kStagedChunk, std::min(want, most));
        p.chunk = (int32_t)((nq + n_chunks - 1) / n_chunks);
        p.n_chunks = (int32_t)((nq + p.chunk - 1) / p.chunk);
        const int64_t grid = (int64_t)ts.count * p.n_chunks;
        if (grid > 0x7FFFFFFFLL) return GS_ERR_OUT_OF_RANGE;
        const size_t smem_batch = smem_staged + (ix->wtype == GS_W_F32 ? BatchGeo<GS_W_F32>::kFixed : BatchGeo<GS_W_U8>::kFixed);
        if (group == 0 && ix->Ts == kBT && ix->wtype == GS_W_U8 && use_mma && ix->mma_strips != nullptr &&
            (ix->HX == 0 || qb.x_on) && kMSmem <= (size_t)smem_max && nq <= 65535) {
            // integer impacts: the head contraction on the tensor cores
            p.mma_strips = ix->mma_strips;
            GS_CUDA(gs_optin_smem(k_score_term_mma));
            GsProfScope ps(GS_K_SCORE_TERM, s);
            k_score_term_mma<<<(unsigned)std::min<int64_t>(grid, sms), kMQ * 32, kMSmem, s>>>(p);
            ++gs_tls_launches;
            GS_CUDA(cudaGetLastError());
            return GS_OK;
        }
        if (group == 0 && ix->Ts == kBT && smem_batch <= (size_t)smem_max && nq <= 65535) {
            auto go = [&](auto kern) -> gs_status_t {
                GS_CUDA(gs_optin_smem(kern));
                GsProfScope ps(GS_K_SCORE_TERM, s);
                // persistent: one CTA per SM walks the (doc tile, query chunk) items
                kern<<<(unsigned)std::min<int64_t>(grid, sms), kBWarps * 32, smem_batch, s>>>(p);
                ++gs_tls_launches;
                GS_CUDA(cudaGetLastError());
                return GS_OK;
            };
            return ix->wtype == GS_W_F32 ? go(k_score_term_batch<GS_W_F32>) : go(k_score_term_batch<GS_W_U8>);
        }
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
