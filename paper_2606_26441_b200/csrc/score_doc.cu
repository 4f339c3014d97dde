// score_doc.cu — S2b: document-parallel forward-index kernel (kernel K2').
//
// PAPER.md L174 §5.3: "an alternative document-parallel kernel using a CSR index by document.  Each
// program handles one (query, document) pair, iterating over the document's term list and looking up
// query weights from a dense query matrix ... eliminates all atomic operations (each program
// exclusively owns its output cell)".  The paper's kernel re-reads the forward index for every
// query (76.3 GB per 500-query batch at 100K docs, Table 7) and names inner-loop
// instruction overhead as what keeps it at 62.6 % of peak (L179).
//
// Here the forward index is streamed ONCE per tile of QT queries (one launch per tile = "pass"), and
// it is a hybrid:
//   * the H densest posting lists are dense strips [H][N_pad] (0 = term absent).  For them there is
//     nothing to look up: a thread owns one document, keeps QT accumulators in registers and does
//     acc[q] += x[h][doc] * Q[h][q].  Q, the tile's head weights, is copied into CONSTANT memory
//     before the pass's launch, so every multiplier is a uniform-register operand of the FFMA/IMAD
//     itself: no shared-memory or register traffic for the ~85 % of the multiply-adds the head
//     lists carry (a broadcast LDS.128 feeds only 4 FMAs and costs 4 LSU cycles, which bounds the
//     contraction at a quarter of the FMA rate; measured in DESIGN.md §6);
//   * every other posting sits in a "tail" block CSR: one row pointer per aligned block of 32
//     documents, the block's postings one flat range padded to 128, the term word carrying the
//     document's position in the block.  A warp owns a block and streams its range with 128-bit
//     loads (one 1 KB chunk in flight in registers — the next block's first chunk across the
//     contraction —, the chunk four ahead asked for from the L2 by prefetch.global.L2),
//     tests each term against a V-bit bitmap of the tile's tail terms (shared memory) and compacts
//     the hits, in stream order, into a per-warp queue (one ballot prefix per 128 postings).  Then
//     lane d walks the hits of document d (contiguous in the queue: a binary search finds them) in
//     ONE flattened loop over (hit, pair): term -> row through a popcount prefix, row -> its
//     (query, weight) pairs, accumulate into the lane's own row of a [32][QT+1] shared-memory tile
//     (odd stride: no two lanes share a bank, no atomics, fixed order).
// Each (query, doc) cell is produced by exactly one thread in a fixed order — zero atomics,
// deterministic.  The query tiles (bitmap + popcount prefix, row table, head weights, thresholds)
// are built once per search by k_build_qtile.
//
// What bounds it (profiles/r02_kernels.md, last sections): 32 warps x 64 registers per SM.  A second chunk in
// flight, eight strip values in flight, fewer warps with more registers, batched candidate atomics: each
// measured slower (spills, or too few warps).  The latency the registers cannot cover is covered from the
// L2 instead — prefetches a few microseconds ahead, not a block ahead: at 4.7 TB/s the stream replaces the
// whole 126 MB L2 within one block's time.
#include <algorithm>
#include <cstddef>
#include <mutex>
#include <type_traits>

#include "gs_internal.cuh"


namespace {

constexpr uint32_t kTermMask = (1u << GS_FWD_DOC_SHIFT) - 1u;
constexpr int kMaxQT = 64;
constexpr int kPfDist = 4;   // rolling L2 prefetch of the posting stream: chunks ahead (3, 4, 6 measured alike; 8 and 12 slower)

// What a pass needs with warp-uniform access.  Built in the search workspace by k_build_qtile, copied to
// c_tile before the pass's launch (stream ordered).  qh is last: a pass copies only its [GS_STRIP_MAX][QT] prefix.
struct ConstTile {
    uint32_t nh;                         // strips some query of the tile uses, rounded up to a multiple of 4 (fp32) / 8 (impacts): zero rows
    uint32_t R;                          // distinct tail terms of the tile (rows)
    uint32_t np;                         // (row, query) pairs
    uint32_t row_off;                    // this pass's slice of the shared row array
    uint32_t pair_off;                   // ... and of the shared pairs array
    uint32_t pad[3];
    uint32_t hl[GS_STRIP_MAX];           // compact position -> strip number (0 beyond nh)
    unsigned long long soff[GS_STRIP_MAX]; // ... and the byte offset of that strip's row in the strip array (hl * N_pad * sizeof(W))
    uint32_t thr_s[kMaxQT];              // threshold as a score (accumulator bits); "accept all" = NaN / INT32_MIN
    unsigned long long thr_key[kMaxQT];  // threshold as a key; queries beyond the tile: all ones
    uint32_t qh[GS_STRIP_MAX * kMaxQT];  // f32: [compact strip][QT] head weights, row stride QT; u8: [strip / 4][QT] words of
                                         // four impact bytes (strips 4g .. 4g+3 of query q)
};
__constant__ ConstTile c_tile;

__host__ __device__ inline size_t tile_copy_bytes(int QT) { return offsetof(ConstTile, qh) + (size_t)GS_STRIP_MAX * QT * 4; }
__host__ __device__ inline int bm_words(int32_t V) { return ((V + 1 + 31) / 32 + 3) / 4 * 4; }
// per-pass scratch block: ConstTile | bitmap[Wd] | prefix[Wd]
__host__ __device__ inline size_t off_bm() { return (sizeof(ConstTile) + 255) / 256 * 256; }
__host__ __device__ inline size_t pass_bytes(int Wd) { return (off_bm() + (size_t)Wd * 8 + 255) / 256 * 256; }
// after the pass blocks: rowptr[n1] | cursor[n1] | rows[n1] (uint2: first pair, end pair) | pairs[nnz] (uint2),  n1 = nnz + passes + 1
struct SharedScratch { uint32_t* rowptr; uint32_t* cursor; uint2* rows; uint2* pairs; };
__host__ __device__ inline size_t up256(size_t b) { return (b + 255) / 256 * 256; }
__host__ __device__ inline SharedScratch shared_scratch(unsigned char* scratch, int Wd, int64_t passes, int64_t nnz) {
    unsigned char* p = scratch + pass_bytes(Wd) * (size_t)passes;
    const size_t n1 = (size_t)(nnz + passes + 1);
    SharedScratch s;
    s.rowptr = reinterpret_cast<uint32_t*>(p);
    s.cursor = reinterpret_cast<uint32_t*>(p + up256(n1 * 4));
    s.rows = reinterpret_cast<uint2*>(p + 2 * up256(n1 * 4));
    s.pairs = reinterpret_cast<uint2*>(p + 2 * up256(n1 * 4) + up256(n1 * 8));
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

template <int WT> struct NumD;
template <> struct NumD<GS_W_F32> {
    using W = float; using A = float;
    static __device__ __forceinline__ A mac(A acc, A q, A w) { return fmaf(q, w, acc); }
    static __device__ __forceinline__ A widen(W w) { return w; }
    static __device__ __forceinline__ A from_bits(uint32_t b) { return __uint_as_float(b); }
    static __device__ __forceinline__ uint32_t bits(A a) { return __float_as_uint(a); }
    static __device__ __forceinline__ uint32_t thr_score_bits(uint32_t ord) { return gs_unord_f32(ord); }   // NaN for ord 0
    static __device__ __forceinline__ uint32_t reject_all_bits() { return 0x7F800000u; }                    // +inf
};
template <> struct NumD<GS_W_U8> {
    using W = uint8_t; using A = int32_t;
    static __device__ __forceinline__ A mac(A acc, A q, A w) { return acc + q * w; }
    static __device__ __forceinline__ A widen(W w) { return (int32_t)w; }
    static __device__ __forceinline__ A from_bits(uint32_t b) { return (int32_t)b; }
    static __device__ __forceinline__ uint32_t bits(A a) { return (uint32_t)a; }
    static __device__ __forceinline__ uint32_t thr_score_bits(uint32_t ord) { return ord ^ 0x80000000u; }   // INT32_MIN for ord 0
    static __device__ __forceinline__ uint32_t reject_all_bits() { return 0x7FFFFFFFu; }                    // INT32_MAX
};

// ---- build the query tile of pass `blockIdx.x` (one CTA of 1024 threads per pass)
template <int WT>
__global__ void __launch_bounds__(1024) k_build_qtile(const int64_t* __restrict__ indptr, const int32_t* __restrict__ terms,
                                                      const void* __restrict__ weights, const int16_t* __restrict__ head_slot,
                                                      int H, int64_t q0, int64_t nq, int QT, int32_t V, int Wd,
                                                      const uint64_t* __restrict__ thr, unsigned char* __restrict__ scratch,
                                                      int64_t n_passes, int64_t nnz_cap, const int32_t* __restrict__ status,
                                                      int64_t strip_row_bytes) {
    extern __shared__ uint32_t sm[];                  // bitmap[Wd], prefix[Wd]
    if (*status != 0) return;                         // ingest found a malformed batch (e.g. a non-monotone indptr): nothing is read
    __shared__ uint32_t warp_tot[32];
    __shared__ uint32_t s_hmask[2];
    __shared__ uint32_t s_total;
    uint32_t* bm = sm;
    uint32_t* pre = sm + Wd;
    const int pass = blockIdx.x;
    const int64_t qa = q0 + (int64_t)pass * QT;
    const int nqt = (int)min((int64_t)QT, q0 + nq - qa);
    unsigned char* base = scratch + (size_t)pass * pass_bytes(Wd);
    ConstTile* ct = reinterpret_cast<ConstTile*>(base);
    uint32_t* g_bm = reinterpret_cast<uint32_t*>(base + off_bm());
    uint32_t* g_pre = g_bm + Wd;
    const SharedScratch ss = shared_scratch(scratch, Wd, n_passes, nnz_cap);
    const uint32_t pair_off = (uint32_t)(indptr[qa] - indptr[q0]);
    const uint32_t row_off = pair_off + (uint32_t)pass;
    uint32_t* rowptr = ss.rowptr + row_off;
    uint32_t* cursor = ss.cursor + row_off;
    uint2* rows = ss.rows + row_off;
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
            if ((s_hmask[h >> 5] >> (h & 31)) & 1u) {
                ct->soff[n] = (unsigned long long)h * (unsigned long long)strip_row_bytes;
                ct->hl[n++] = (uint32_t)h;
            }
        const uint32_t n8 = WT == GS_W_F32 ? ((n + 3u) & ~3u) : ((n + 7u) & ~7u);      // strips per turn of the strip contraction
        for (uint32_t i = n; i < GS_STRIP_MAX; ++i) { ct->hl[i] = 0u; ct->soff[i] = 0ull; }      // padding rows carry zero weights
        ct->nh = n8;
        ct->R = R;
        ct->row_off = row_off;
        ct->pair_off = pair_off;
    }
    for (int i = threadIdx.x; i < kMaxQT; i += blockDim.x) {
        // thresholds of the tile's queries (filter phase); without thresholds every cell is accepted
        uint64_t key = ~0ull;
        uint32_t sb = NumD<WT>::reject_all_bits();
        if (i < nqt) {
            key = thr ? thr[qa + i] : 0ull;
            sb = NumD<WT>::thr_score_bits((uint32_t)(key >> 32));
        }
        ct->thr_key[i] = key;
        ct->thr_s[i] = sb;
    }
    for (int i = threadIdx.x; i < Wd; i += blockDim.x) { g_bm[i] = bm[i]; g_pre[i] = pre[i]; }
    for (int i = threadIdx.x; i < GS_STRIP_MAX * QT; i += blockDim.x) ct->qh[i] = 0u;
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
            rows[r] = make_uint2(run, run + cursor[r]);
            run += cursor[r];
        }
    }
    __syncthreads();
    if (threadIdx.x == 0) { rowptr[R] = s_total; ct->np = s_total; }
    for (uint32_t i = threadIdx.x; i <= R; i += blockDim.x) cursor[i] = 0u;
    __syncthreads();
    // queries in order, so the pairs of a row are sorted by query: a fixed accumulation order
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
                if (WT == GS_W_F32) ct->qh[(size_t)ci * QT + j] = w;
                else                                       // impacts: byte (ci & 3) of word [ci / 4][j] — four strips per IDP4A
                    reinterpret_cast<uint8_t*>(ct->qh)[((size_t)(ci >> 2) * QT + j) * 4 + (ci & 3)] = (uint8_t)w;
            } else {
                const uint32_t word = bm[t >> 5];
                const uint32_t r = pre[t >> 5] + __popc(word & ((1u << (t & 31)) - 1u));
                const uint32_t pos = atomicAdd(&cursor[r], 1u);
                pairs[rowptr[r] + pos] = make_uint2((uint32_t)j, w);
            }
        }
        __syncthreads();
    }
}

struct DocParams {
    const int64_t* fwd_blk; const uint32_t* fwd_terms; const void* fwd_w;
    int32_t fwd_packed;                         // integer-impact mode: the term word carries the impact in bits 19..26, no fwd_w
    const void* strips; int64_t N_pad;
    int64_t N; int32_t V; int32_t Ts; int32_t Wd;
    const uint32_t* tile_bm;                    // this pass's bitmap[Wd] | prefix[Wd]
    const uint2* rows; const uint2* pairs;      // shared row / pairs arrays (the pass's slices start at c_tile.row_off / pair_off)
    int32_t sparse_cap_bytes;                   // shared memory left for a pass's row table + pairs
    int64_t qa; int32_t nqt;                    // queries [qa, qa+nqt) of the batch; q_rel = qa - q0 of the launch
    int64_t q_rel;
    const int32_t* status;                      // ingest status word: non-zero = malformed batch, the pass does nothing
    gs_tileset ts;
    gs_sink sink;
};

template <int QT> struct Geo {
    static constexpr int AST = QT + 1;                 // row stride of the accumulator tile (odd: lane rows hit distinct banks)
    static constexpr int NW = QT <= 16 ? 32 : (QT == 32 ? 20 : 12);              // warps per CTA
    // hit-queue entries per warp: a block's hits (281 / 536 / 838 on average at QT = 16 / 32 / 64 on the MS MARCO
    // stand-in) should fit, because a walk over part of a block leaves the lanes of the other documents idle
    static constexpr int QCAP = QT <= 8 ? 640 : (QT == 16 ? 512 : (QT == 32 ? 768 : 1152));
    static constexpr size_t per_warp = (size_t)QCAP * 8 + (size_t)32 * AST * 4;
    static __host__ __device__ size_t fixed(int Wd) { return (size_t)Wd * 8 + (size_t)GS_STRIP_MAX * 8; }   // bitmap, prefix, strip offsets
};

__device__ __forceinline__ uint4 ld_stream4(const uint4* p) { return __ldcs(p); }
__device__ __forceinline__ uint32_t ld_stream1(const uint32_t* p) { return __ldcs(p); }

// Dense strip contraction of one document (thread = document): acc[q] += x[h][doc] * Q[h][q] over the strips the
// tile uses; every weight is fetched by a uniform constant load and used as the uniform operand of the FFMA2 / IDP4A
// itself.  Tiles of up to 16 queries: fully unrolled and in line (strips_body below).  Larger tiles: a separate
// function (strips_call) — compiled on its own, the strip loop's index stays in a uniform register (LDCU
// c[3][UR+imm]), the body (4 x QT multiply-adds) stays small in the instruction cache, and the accumulators travel
// through the lane's own row of the shared-memory tile (conflict-free).
__device__ __forceinline__ unsigned long long fma_f32x2(unsigned long long a, float x, unsigned long long c) {
    // (a.lo * x + c.lo, a.hi * x + c.hi): one FFMA2, each half an IEEE fp32 fma (same result as two fmaf)
    unsigned long long d, xx;
    asm("mov.b64 %0, {%1, %1};" : "=l"(xx) : "f"(x));
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(xx), "l"(c));
    return d;
}

template <int WT, int QT>
__device__ __forceinline__ void strips_body(typename NumD<WT>::A* __restrict__ myacc,
                                          const typename NumD<WT>::W* __restrict__ sp, int64_t N_pad) {
    using A = typename NumD<WT>::A;
    const int nh = (int)c_tile.nh;
    if constexpr (WT == GS_W_F32) {
        // packed pairs of queries: one FFMA2 (uniform-register weight pair x scalar strip value) per two cells
        unsigned long long acc[QT / 2];
#pragma unroll
        for (int q = 0; q < QT / 2; ++q)
            asm("mov.b64 %0, {%1, %2};" : "=l"(acc[q]) : "f"(myacc[2 * q]), "f"(myacc[2 * q + 1]));
        if constexpr (QT <= 16) {
            // Fully unrolled over the (at most GS_STRIP_MAX) compact strips with early exits on nh: every weight offset is a
            // compile-time constant, so the weights arrive by LDCU.128 (four weights = two FFMA2 per uniform load; with a
            // runtime strip index the compiler issued one LDCU.64 per FFMA2) and a strip's address is base + a 64-bit byte
            // offset from the constant tile (no multiply).  Two register groups of kSG strip values alternate: the values of
            // the next group are loaded before the multiply-adds of the current one (a strip value is one DRAM / L2 round
            // trip per block of 32 documents).  c_tile.soff is padded with offset 0 (a valid row, zero weights).
            constexpr int kSG = 4;
            const char* spb = reinterpret_cast<const char*>(sp);
            float xa[kSG], xb[kSG];
            auto ldx = [&](float (&x)[kSG], int i0) {
#pragma unroll
                for (int u = 0; u < kSG; ++u) x[u] = *reinterpret_cast<const float*>(spb + c_tile.soff[i0 + u]);
            };
            auto mac = [&](const float (&x)[kSG], int i0) {
#pragma unroll
                for (int u = 0; u < kSG; ++u) {
#pragma unroll
                    for (int q = 0; q < QT; q += 2) {
                        const unsigned long long v = *reinterpret_cast<const unsigned long long*>(&c_tile.qh[(i0 + u) * QT + q]);
                        acc[q / 2] = fma_f32x2(v, x[u], acc[q / 2]);
                    }
                }
            };
            ldx(xa, 0);
#pragma unroll
            for (int i0 = 0; i0 < GS_STRIP_MAX; i0 += 2 * kSG) {
                if (i0 >= nh) break;
                if (i0 + kSG < nh) ldx(xb, i0 + kSG);
                mac(xa, i0);
                if (i0 + kSG >= nh) break;
                if (i0 + 2 * kSG < GS_STRIP_MAX && i0 + 2 * kSG < nh) ldx(xa, i0 + 2 * kSG);
                mac(xb, i0 + kSG);
            }
        } else {
            // The strip values of the next kSG strips are loaded before the multiply-adds of the current ones: a strip value is
            // one DRAM round trip per block of 32 documents, and with 4 in flight that wait is 20 % of the kernel's stall
            // samples (profiles/r02_kernels.md).  c_tile.hl is padded with valid strip numbers up to a multiple of kSG.
            constexpr int kSG = 4;
            float xn[kSG];
#pragma unroll
            for (int u = 0; u < kSG; ++u) xn[u] = sp[(size_t)c_tile.hl[u] * N_pad];
#pragma unroll 1
            for (int i0 = 0; i0 < nh; i0 += kSG) {
                float x[kSG];
#pragma unroll
                for (int u = 0; u < kSG; ++u) x[u] = xn[u];
                if (i0 + kSG < nh) {
#pragma unroll
                    for (int u = 0; u < kSG; ++u) xn[u] = sp[(size_t)c_tile.hl[i0 + kSG + u] * N_pad];
                }
#pragma unroll
                for (int u = 0; u < kSG; ++u) {
#pragma unroll
                    for (int q = 0; q < QT; q += 4) {
                        const ulonglong2 v = *reinterpret_cast<const ulonglong2*>(&c_tile.qh[(i0 + u) * QT + q]);
                        acc[q / 2] = fma_f32x2(v.x, x[u], acc[q / 2]);
                        acc[q / 2 + 1] = fma_f32x2(v.y, x[u], acc[q / 2 + 1]);
                    }
                }
            }
        }
#pragma unroll
        for (int q = 0; q < QT / 2; ++q) {
            float lo, hi;
            asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(acc[q]));
            myacc[2 * q] = lo;
            myacc[2 * q + 1] = hi;
        }
    } else {
        A acc[QT];
#pragma unroll
        for (int q = 0; q < QT; ++q) acc[q] = myacc[q];
        // integer impacts: the document's bytes of four strips packed into one word, the tile's weights of the same four
        // strips packed per query (k_build_qtile): one IDP4A per (four strips, query); the bytes of the next 8 strips are
        // loaded before the IDP4As of the current ones
        if constexpr (QT <= 16) {
            // unrolled like the fp32 branch: constant offsets, strip addresses from c_tile.soff, two alternating groups
            const char* spb = reinterpret_cast<const char*>(sp);
            uint32_t xa[8], xb[8];
            auto ldx = [&](uint32_t (&x)[8], int i0) {
#pragma unroll
                for (int u = 0; u < 8; ++u) x[u] = (uint32_t) * reinterpret_cast<const uint8_t*>(spb + c_tile.soff[i0 + u]);
            };
            auto mac = [&](const uint32_t (&x)[8], int i0) {
                const uint32_t lo = x[0] | (x[1] << 8) | (x[2] << 16) | (x[3] << 24);
                const uint32_t hi = x[4] | (x[5] << 8) | (x[6] << 16) | (x[7] << 24);
#pragma unroll
                for (int q = 0; q < QT; ++q) {
                    acc[q] = (A)__dp4a(lo, c_tile.qh[(i0 >> 2) * QT + q], (uint32_t)acc[q]);
                    acc[q] = (A)__dp4a(hi, c_tile.qh[((i0 >> 2) + 1) * QT + q], (uint32_t)acc[q]);
                }
            };
            ldx(xa, 0);
#pragma unroll
            for (int i0 = 0; i0 < GS_STRIP_MAX; i0 += 16) {
                if (i0 >= nh) break;
                if (i0 + 8 < nh) ldx(xb, i0 + 8);
                mac(xa, i0);
                if (i0 + 8 >= nh) break;
                if (i0 + 16 < GS_STRIP_MAX && i0 + 16 < nh) ldx(xa, i0 + 16);
                mac(xb, i0 + 8);
            }
        } else {
            uint32_t xn[8];
#pragma unroll
            for (int u = 0; u < 8; ++u) xn[u] = (uint32_t)sp[(size_t)c_tile.hl[u] * N_pad];
#pragma unroll 1
            for (int i0 = 0; i0 < nh; i0 += 8) {
                const uint32_t xa = xn[0] | (xn[1] << 8) | (xn[2] << 16) | (xn[3] << 24);
                const uint32_t xb = xn[4] | (xn[5] << 8) | (xn[6] << 16) | (xn[7] << 24);
                if (i0 + 8 < nh) {
#pragma unroll
                    for (int u = 0; u < 8; ++u) xn[u] = (uint32_t)sp[(size_t)c_tile.hl[i0 + 8 + u] * N_pad];
                }
#pragma unroll
                for (int q = 0; q < QT; ++q) {
                    acc[q] = (A)__dp4a(xa, c_tile.qh[(i0 >> 2) * QT + q], (uint32_t)acc[q]);
                    acc[q] = (A)__dp4a(xb, c_tile.qh[((i0 >> 2) + 1) * QT + q], (uint32_t)acc[q]);
                }
            }
        }
#pragma unroll
        for (int q = 0; q < QT; ++q) myacc[q] = acc[q];
    }
}

// QT <= 16: in line (unrolled, no call: the loads of the next block's first chunk stay in flight across the contraction
// instead of being saved around a call).  Larger tiles: a separate function — compiled on its own, the strip loop's index
// stays in a uniform register and the body stays small in the instruction cache.
template <int WT, int QT>
__device__ __noinline__ void strips_call(typename NumD<WT>::A* __restrict__ myacc, const typename NumD<WT>::W* __restrict__ sp,
                                         int64_t N_pad) {
    strips_body<WT, QT>(myacc, sp, N_pad);
}
template <int WT, int QT>
__device__ __forceinline__ void strips_phase(typename NumD<WT>::A* __restrict__ myacc, const typename NumD<WT>::W* __restrict__ sp,
                                             int64_t N_pad) {
    if constexpr (QT <= 16) strips_body<WT, QT>(myacc, sp, N_pad);
    else strips_call<WT, QT>(myacc, sp, N_pad);
}

template <int WT, int QT>
__global__ void __launch_bounds__(Geo<QT>::NW * 32, 1) k_score_doc(const DocParams p) {
    using W = typename NumD<WT>::W;
    using A = typename NumD<WT>::A;
    using G = Geo<QT>;
    constexpr int AST = G::AST, NW = G::NW, QCAP = G::QCAP;
    extern __shared__ __align__(16) unsigned char smem[];
    if (*p.status != 0) return;
    const int Wd = p.Wd;
    const uint32_t R = c_tile.R, np = c_tile.np;
    const int nh = (int)c_tile.nh;
    const uint2* g_rows = p.rows + c_tile.row_off;
    const uint2* g_pairs = p.pairs + c_tile.pair_off;
    const bool sparse_in_smem = (size_t)(R + np) * 8 <= (size_t)p.sparse_cap_bytes;

    uint32_t* s_bm = reinterpret_cast<uint32_t*>(smem);                           // [Wd]
    uint32_t* s_pre = s_bm + Wd;                                                  // [Wd]
    unsigned long long* s_soff = reinterpret_cast<unsigned long long*>(s_pre + Wd);   // [GS_STRIP_MAX] copy of c_tile.soff (lane-indexed reads)
    unsigned char* pw = reinterpret_cast<unsigned char*>(s_soff + GS_STRIP_MAX);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    uint2* queue = reinterpret_cast<uint2*>(pw + (size_t)warp * G::per_warp);     // [QCAP]
    A* s_acc = reinterpret_cast<A*>(queue + QCAP);                                // [32][AST]
    uint2* s_pairs = reinterpret_cast<uint2*>(pw + (size_t)NW * G::per_warp);     // [np]  when it fits
    uint2* s_rows = s_pairs + np;                                                 // [R]

    const bool filter = p.sink.thr != nullptr;
    {   // stage the query tile
        for (int i = threadIdx.x; i < 2 * Wd; i += NW * 32) s_bm[i] = p.tile_bm[i];   // bitmap and prefix are adjacent
        if (threadIdx.x < GS_STRIP_MAX) s_soff[threadIdx.x] = c_tile.soff[threadIdx.x];
        if (sparse_in_smem) {
            for (uint32_t i = threadIdx.x; i < np; i += NW * 32) s_pairs[i] = g_pairs[i];
            for (uint32_t i = threadIdx.x; i < R; i += NW * 32) s_rows[i] = g_rows[i];
        }
    }
    __syncthreads();
    // the block loop exists twice, with the row table and the pairs in shared memory (the normal case) or, when a
    // tile's tables do not fit, in global memory: one address space per instantiation, no generic loads
    auto run = [&](auto sp_tag) {
    constexpr bool SP = decltype(sp_tag)::value;
    const uint2* rows = SP ? s_rows : g_rows;
    const uint2* pairs = SP ? s_pairs : g_pairs;

    const W* __restrict__ strips = reinterpret_cast<const W*>(p.strips);
    const unsigned lt = (1u << lane) - 1u;
    A* myacc = s_acc + lane * AST;
    const int subs_per_tile = p.Ts >> 5;
    // 32-bit block, chunk and document numbers in the loop state (the launcher checks the ranges): registers are what
    // limits the loads in flight here
    const int n_subs = (int)(p.ts.count * subs_per_tile);
    const int sb_stride = (int)gridDim.x * NW;

    // lane d applies the queued hits of document d (contiguous: the queue is in stream order); one loop over (hit, pair)
    auto walk = [&](int n) {
        __syncwarp();
        int lo = 0, hi = n;
        for (int it = 32 - __clz(n); it > 0; --it) {          // lower bound of the first entry with doc position >= lane
            const int mid = (lo + hi) >> 1;
            if (lo < hi) {
                if ((int)(queue[mid].x >> GS_FWD_DOC_SHIFT) < lane) lo = mid + 1; else hi = mid;
            }
        }
        int end = __shfl_down_sync(0xFFFFFFFFu, lo, 1);
        if (lane == 31) end = n;
        int j = lo;
        uint32_t i = 0, i_end = 0;
        A w = A(0);
        for (;;) {
            if (i == i_end) {                                  // next hit of this document
                if (j >= end) break;
                const uint2 e = queue[j++];
                const uint32_t t = e.x & kTermMask;
                w = NumD<WT>::from_bits(e.y);
                const uint32_t word = s_bm[t >> 5];
                const uint2 r = rows[s_pre[t >> 5] + __popc(word & ((1u << (t & 31)) - 1u))];
                i = r.x;
                i_end = r.y;                                   // every row holds at least one pair
            }
            const uint2 pr = pairs[i++];
            myacc[pr.x] = NumD<WT>::mac(myacc[pr.x], NumD<WT>::from_bits(pr.y), w);
        }
        __syncwarp();
    };

    // block -> (start, chunks) of its posting range, or nothing beyond the collection
    auto block_of = [&](int sb, int& doc0) -> int {
        const int64_t tile = p.ts.first + (sb / subs_per_tile) * (int64_t)p.ts.stride;
        const int64_t d = tile * p.Ts + (sb % subs_per_tile) * 32;
        doc0 = (int)d;
        return d < p.N ? (int)(d >> 5) : -1;
    };
    const uint32_t* __restrict__ wp1 = reinterpret_cast<const uint32_t*>(p.fwd_w);     // u8: 4 weights per word
    const uint4* __restrict__ wp4 = reinterpret_cast<const uint4*>(p.fwd_w);           // f32
    const uint4* __restrict__ tp4 = reinterpret_cast<const uint4*>(p.fwd_terms);
    // chunk c (128 postings) of the index: lane holds postings 4*lane .. 4*lane+3
    auto load_chunk = [&](int chunk, uint4& t4, uint4& w4, bool pf = false) {
        const uint4* tptr = tp4 + (size_t)(uint32_t)chunk * 32 + lane;
        t4 = ld_stream4(tptr);
        // rolling L2 prefetch: a lane whose 16 bytes start a 128-byte line (lanes 0, 8, 16, 24) asks for the same line of
        // the chunk kPfDist - 1 further on — the load's own address plus a constant, no address arithmetic of its own
        if (pf) asm volatile("prefetch.global.L2 [%0];" ::"l"(reinterpret_cast<const char*>(tptr) + (kPfDist - 1) * 512));
        if (WT == GS_W_F32) {
            const uint4* wptr = wp4 + (size_t)(uint32_t)chunk * 32 + lane;
            if (pf) asm volatile("prefetch.global.L2 [%0];" ::"l"(reinterpret_cast<const char*>(wptr) + (kPfDist - 1) * 512));
            w4 = ld_stream4(wptr);
        } else if (p.fwd_packed) {                 // compressed postings: term | impact << 19 | (doc & 31) << 27
            w4 = make_uint4((t4.x >> 19) & 0xFFu, (t4.y >> 19) & 0xFFu, (t4.z >> 19) & 0xFFu, (t4.w >> 19) & 0xFFu);
            t4 = make_uint4(t4.x & 0xF807FFFFu, t4.y & 0xF807FFFFu, t4.z & 0xF807FFFFu, t4.w & 0xF807FFFFu);
        } else {
            const uint32_t v = ld_stream1(wp1 + (size_t)(uint32_t)chunk * 32 + lane);
            w4 = make_uint4(v & 0xFFu, (v >> 8) & 0xFFu, (v >> 16) & 0xFFu, v >> 24);
        }
    };
    // block -> first chunk and number of chunks of its posting range (c0 < 0: block beyond the collection)
    auto range_of = [&](int sbx, int& d0, int& cc0, int& ncc) {
        cc0 = -1; ncc = 0; d0 = 0;
        if (sbx >= n_subs) return;
        const int blk = block_of(sbx, d0);
        if (blk < 0) return;
        cc0 = (int)(p.fwd_blk[blk] / GS_FWD_CHUNK);
        ncc = (int)(p.fwd_blk[blk + 1] / GS_FWD_CHUNK) - cc0;
    };
    int sb = (int)blockIdx.x * NW + warp;
    int doc0 = 0, c0 = -1;                           // first document and first chunk of the current block
    int nc = 0;                                      // its chunks
    // two chunk buffers: chunk i of a block lives in buffer i % 2 while it is in flight / being filtered (the chunk loop is
    // unrolled by two so that no buffer is ever copied to another: the rotation by register moves was a quarter of the
    // loop's instructions).  A third buffer (two chunks in flight) spills at 64 registers and measured slower (69.7 vs
    // 57.5 ms per 500-query batch); 24 or 28 warps with 80 / 72 registers and two chunks in flight: 64.4 / 62.0 ms
    uint4 tA = make_uint4(0, 0, 0, 0), wA = tA, tB = tA, wB = tA;
    range_of(sb, doc0, c0, nc);
    if (nc > 0) load_chunk(c0, tA, wA);
    for (; sb < n_subs; sb += sb_stride) {
        // the next block's range, asked for now, needed after the walk
        int doc0n, c0n, ncn;
        range_of(sb + sb_stride, doc0n, c0n, ncn);
        if (c0 < 0) {                              // block beyond the collection
            doc0 = doc0n; c0 = c0n; nc = ncn;
            if (nc > 0) load_chunk(c0, tA, wA);
            continue;
        }
        // the 128-byte strip segments of this block's documents, one line per lane and turn, into the L2 (no registers, no
        // shared memory): asked for before the walk, read after it.  Not a whole block earlier: in one block's time the
        // stream turns the whole L2 over, and the lines were gone again (1.9 GB of re-reads per pass, measured); at the
        // block's start: 57.5 ms per 500-query batch against 54.9 here
        auto prefetch_strips = [&]() {
            for (int i = lane; i < nh; i += 32)
                asm volatile("prefetch.global.L2 [%0];" ::"l"(reinterpret_cast<const char*>(strips + doc0) + s_soff[i]));
        };
        // rolling L2 prefetch of the posting stream (load_chunk): the lanes whose 16 bytes start a 128-byte line ask for
        // the same line of the chunk kPfDist ahead of the one being filtered
        const bool pf_lane = (lane & 7) == 0;
        for (int i = lane; i < 32 * AST; i += 32) s_acc[i] = A(0);

        // ---- tail: the block's postings as one flat range -> bitmap filter -> hit queue -> per-document walk
        int cnt = 0;
        auto filter_chunk = [&](const uint4& tc, const uint4& wc) {
            if (cnt + GS_FWD_CHUNK > QCAP) { walk(cnt); cnt = 0; }
            const uint32_t tw[4] = {tc.x, tc.y, tc.z, tc.w};
            const uint32_t ww[4] = {wc.x, wc.y, wc.z, wc.w};
            uint32_t h[4];
#pragma unroll
            for (int u = 0; u < 4; ++u) h[u] = (s_bm[(tw[u] >> 5) & (kTermMask >> 5)] >> (tw[u] & 31u)) & 1u;
            const uint32_t nhit = h[0] + h[1] + h[2] + h[3];
            const unsigned b0 = __ballot_sync(0xFFFFFFFFu, nhit & 1u), b1 = __ballot_sync(0xFFFFFFFFu, nhit & 2u),
                           b2 = __ballot_sync(0xFFFFFFFFu, nhit & 4u);
            if ((b0 | b1 | b2) != 0u) {
                int pos = cnt + __popc(b0 & lt) + 2 * __popc(b1 & lt) + 4 * __popc(b2 & lt);
#pragma unroll
                for (int u = 0; u < 4; ++u) {
                    if (h[u]) queue[pos] = make_uint2(tw[u], ww[u]);
                    pos += (int)h[u];
                }
                cnt += __popc(b0) + 2 * __popc(b1) + 4 * __popc(b2);
            }
        };
        for (int i = 0;;) {                          // one chunk in flight ahead of the one being filtered
            if (i >= nc) break;
            if (i + 1 < nc) load_chunk(c0 + i + 1, tB, wB, pf_lane && i + kPfDist < nc);
            filter_chunk(tA, wA);
            ++i;
            if (i >= nc) break;
            if (i + 1 < nc) load_chunk(c0 + i + 1, tA, wA, pf_lane && i + kPfDist < nc);
            filter_chunk(tB, wB);
            ++i;
        }
        prefetch_strips();
        walk(cnt);
        // first chunks of the next block: in flight during the contraction
        if (ncn > 0) load_chunk(c0n, tA, wA);

        // ---- head strips: thread = document, QT accumulators in registers, weights as uniform constant operands
        const int64_t doc = (int64_t)doc0 + lane;
        if (nh > 0) strips_phase<WT, QT>(myacc, strips + doc, p.N_pad);
        A acc[QT];
#pragma unroll
        for (int q = 0; q < QT; ++q) acc[q] = myacc[q];

        // ---- sink: this thread owns the cells (qa + q, doc)
        if (doc < p.N) {
            if (!filter) {
                uint32_t* out = p.sink.dense + p.q_rel * p.sink.ld + (int64_t)sb * 32 + lane;
#pragma unroll
                for (int q = 0; q < QT; ++q)
                    if (q < p.nqt) out[(int64_t)q * p.sink.ld] = NumD<WT>::bits(acc[q]);
            } else {
#pragma unroll
                for (int q = 0; q < QT; ++q) {
                    if (!(acc[q] < NumD<WT>::from_bits(c_tile.thr_s[q]))) {
                        const uint64_t key = gs_make_key(gs_ord_bits<WT>(NumD<WT>::bits(acc[q])), (uint32_t)doc);
                        if (q < p.nqt && key >= c_tile.thr_key[q]) {
                            const int64_t b = p.qa + q;
                            const uint32_t pos = atomicAdd(&p.sink.cand_cnt[b * GS_CNT_STRIDE], 1u);
                            if ((int64_t)pos < p.sink.cand_cap) p.sink.cand[b * p.sink.cand_cap + pos] = key;
                        }
                    }
                }
            }
        }
        __syncwarp();
        doc0 = doc0n; c0 = c0n; nc = ncn;
    }
    };
    if (sparse_in_smem) run(std::true_type{}); else run(std::false_type{});
}

int norm_qt(int qtile) {
    if (qtile <= 0) return 32;
    int q = 8;
    while (q < qtile && q < kMaxQT) q <<= 1;
    return q;
}

// The constant tile is one per device: searches that use it are serialised (host side by the mutex, device side by
// making a search's stream wait for the previous search's last pass).
std::mutex g_tile_mu;
cudaEvent_t g_tile_free[64] = {};

template <int WT, int QT>
gs_status_t launch_passes(DocParams p, const unsigned char* scratch, int Wd, int64_t n_subs, int n_passes, int64_t q0, int64_t nq,
                          int sms, int smem_max, cudaStream_t s) {
    using G = Geo<QT>;
    const size_t fixed = G::fixed(Wd) + (size_t)G::NW * G::per_warp;
    if (fixed > (size_t)smem_max) return GS_ERR_OUT_OF_RANGE;     // vocabulary too large for the shared-memory bitmap
    const size_t smem = (size_t)smem_max;
    p.sparse_cap_bytes = (int32_t)(smem - fixed);
    const unsigned grid = (unsigned)std::max<int64_t>(1, std::min<int64_t>(sms, (n_subs + G::NW - 1) / G::NW));
    GS_CUDA(gs_optin_smem(k_score_doc<WT, QT>));
    int dev = 0;
    cudaGetDevice(&dev);
    std::lock_guard<std::mutex> lock(g_tile_mu);
    cudaEvent_t& ev = g_tile_free[dev & 63];
    if (!ev) GS_CUDA(cudaEventCreateWithFlags(&ev, cudaEventDisableTiming));
    else GS_CUDA(cudaStreamWaitEvent(s, ev, 0));
    for (int pass = 0; pass < n_passes; ++pass) {
        const unsigned char* base = scratch + (size_t)pass * pass_bytes(Wd);
        {
            GsProfScope ps(GS_K_QTILE, s, 0);
            GS_CUDA(cudaMemcpyToSymbolAsync(c_tile, base, tile_copy_bytes(QT), 0, cudaMemcpyDeviceToDevice, s));
        }
        p.tile_bm = reinterpret_cast<const uint32_t*>(base + off_bm());
        p.qa = q0 + (int64_t)pass * QT;
        p.q_rel = (int64_t)pass * QT;
        p.nqt = (int32_t)std::min<int64_t>(QT, q0 + nq - p.qa);
        {
            GsProfScope ps(GS_K_SCORE_DOC, s);
            k_score_doc<WT, QT><<<grid, G::NW * 32, smem, s>>>(p);
        }
        ++gs_tls_launches;
    }
    GS_CUDA(cudaEventRecord(ev, s));
    GS_CUDA(cudaGetLastError());
    return GS_OK;
}
template <int WT>
gs_status_t launch_doc_qt(int QT, const DocParams& p, const unsigned char* scratch, int Wd, int64_t n_subs, int n_passes,
                          int64_t q0, int64_t nq, int sms, int smem_max, cudaStream_t s) {
    switch (QT) {
        case 8: return launch_passes<WT, 8>(p, scratch, Wd, n_subs, n_passes, q0, nq, sms, smem_max, s);
        case 16: return launch_passes<WT, 16>(p, scratch, Wd, n_subs, n_passes, q0, nq, sms, smem_max, s);
        case 32: return launch_passes<WT, 32>(p, scratch, Wd, n_subs, n_passes, q0, nq, sms, smem_max, s);
        default: return launch_passes<WT, 64>(p, scratch, Wd, n_subs, n_passes, q0, nq, sms, smem_max, s);
    }
}

}  // namespace

int gs_score_doc_qtile(int qtile) { return norm_qt(qtile); }

size_t gs_score_doc_scratch_bytes_ex(const gs_index* ix, int qtile, int64_t nq, int64_t q_nnz) {
    const int QT = norm_qt(qtile);
    const int64_t passes = std::max<int64_t>((nq + QT - 1) / QT, 1);
    const int Wd = bm_words(ix->V);
    const size_t n1 = (size_t)(q_nnz + passes + 1);
    return pass_bytes(Wd) * (size_t)passes + 2 * up256(n1 * 4) + up256(n1 * 8) + up256((size_t)q_nnz * 8);
}

gs_status_t gs_launch_score_doc(const gs_index* ix, const gs_csr_t* q, const gs_qbatch& qb, int64_t q0, int64_t nq,
                                int qtile, const gs_tileset& ts, const gs_sink& sink, void* scratch, cudaStream_t s) {
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
            GS_CUDA(gs_optin_smem(k_build_qtile<GS_W_F32>));
            k_build_qtile<GS_W_F32><<<n_passes, 1024, bsm, s>>>(q->indptr, q->term_ids, q->weights, ix->head_slot, ix->H, q0, nq,
                                                              QT, ix->V, Wd, sink.thr, (unsigned char*)scratch, passes_cap, q->nnz, qb.status,
                                                              (int64_t)ix->N_pad * 4);
        } else {
            GS_CUDA(gs_optin_smem(k_build_qtile<GS_W_U8>));
            k_build_qtile<GS_W_U8><<<n_passes, 1024, bsm, s>>>(q->indptr, q->term_ids, q->weights, ix->head_slot, ix->H, q0, nq,
                                                             QT, ix->V, Wd, sink.thr, (unsigned char*)scratch, passes_cap, q->nnz, qb.status,
                                                             (int64_t)ix->N_pad);
        }
        ++gs_tls_launches;
        GS_CUDA(cudaGetLastError());
    }
    const SharedScratch ss = shared_scratch((unsigned char*)scratch, Wd, passes_cap, q->nnz);
    DocParams p{};
    p.fwd_blk = ix->fwd_blk; p.fwd_terms = ix->fwd_terms; p.fwd_w = ix->fwd_w; p.fwd_packed = ix->fwd_packed ? 1 : 0;
    p.strips = ix->head_strip; p.N_pad = ix->N_pad;
    p.N = ix->N; p.V = ix->V; p.Ts = ix->Ts; p.Wd = Wd;
    p.rows = ss.rows; p.pairs = ss.pairs;
    p.ts = ts; p.sink = sink; p.status = qb.status;
    const int64_t n_subs = (int64_t)ts.count * (ix->Ts / 32);
    // the kernel keeps block, chunk and document numbers in 32 bits
    if (n_subs >= (1LL << 31) - (1LL << 20) || ix->N_pad + ix->Ts >= (1LL << 31) || ix->P_fwd / GS_FWD_CHUNK >= (1LL << 31) - 8) return GS_ERR_OUT_OF_RANGE;
    return ix->wtype == GS_W_F32
               ? launch_doc_qt<GS_W_F32>(QT, p, (const unsigned char*)scratch, Wd, n_subs, n_passes, q0, nq, sms, smem_max, s)
               : launch_doc_qt<GS_W_U8>(QT, p, (const unsigned char*)scratch, Wd, n_subs, n_passes, q0, nq, sms, smem_max, s);
}
