// topk.cu — S3: exact per-query top-k under the strict order (score desc, doc id asc) (kernel K3').
//
// The paper takes torch.topk over the whole [B,N] score buffer
// and attributes its recall < 1 to unspecified tie order (L129, L396).  Here every candidate is a
// 64-bit composite key ord(score)<<32 | ~doc, so all keys of a query are distinct and the order is
// total: an MSD radix select (11-bit digits, shared-memory histograms) finds the exact k-th key,
// one pass collects the k keys >= it, and a bitonic network (warp shuffles for the short strides,
// shared memory for the long ones) sorts them.  The select runs either over dense score rows
// (fallback / threshold sample) or over the candidate key lists the scoring kernels emit.
#include <cooperative_groups.h>

#include <algorithm>
#include <mutex>

#include "gs_internal.cuh"

#define GS_SEL_TARGET 128     // CTAs a select launch aims for before it stops splitting rows over clusters

namespace {

constexpr int kSelThreads = 512;
constexpr int kItemsPerCta = 16384;

struct SelState {
    unsigned long long prefix;   // key bits decided so far (undecided low bits are 0)
    unsigned int k_rem;          // how many of the items matching `prefix` are still wanted
    int shift;                   // bit position of the next digit (+width); <= 0 when all bits are decided
    int done;
    unsigned int n_items;
    unsigned int out_cnt;
    unsigned int pad[2];
};

__device__ __forceinline__ int64_t src_count(const gs_sel_src& s, int64_t b) {
    return s.keys ? (int64_t)min((uint64_t)s.counts[b * s.cnt_stride], (uint64_t)s.cap) : s.n_cols;
}
// key of item i of row b, or 0 when the item does not exist (column beyond the last document)
template <int WT>
__device__ __forceinline__ uint64_t src_key(const gs_sel_src& s, int64_t b, int64_t i) {
    if (s.keys) return s.keys[b * s.cap + i];
    int64_t doc = i;
    if (s.Ts > 0) {                                   // column -> doc id of a strided tile set (columns < 2^31)
        const uint32_t jt = (uint32_t)i / (uint32_t)s.Ts;
        doc = ((int64_t)s.ts.first + (int64_t)jt * s.ts.stride) * s.Ts + ((uint32_t)i - jt * (uint32_t)s.Ts);
    }
    if (doc >= s.n_docs) return 0ull;
    return gs_make_key(gs_ord_bits<WT>(s.dense[b * s.ld + i]), (uint32_t)doc);
}

__global__ void k_sel_init(gs_sel_src src, int64_t rows, int32_t k, SelState* st, uint32_t* hist) {
    const int64_t b = blockIdx.x;
    if (threadIdx.x == 0) {
        int64_t n = src_count(src, b);
        if (!src.keys) {   // dense: number of live documents among the columns
            int64_t live = 0;
            if (src.Ts > 0) {
                for (int64_t j = 0; j < src.ts.count; ++j) {
                    int64_t d0 = ((int64_t)src.ts.first + j * src.ts.stride) * src.Ts;
                    live += max((int64_t)0, min((int64_t)src.Ts, src.n_docs - d0));
                }
            } else live = min(n, src.n_docs);
            n = live;
        }
        SelState s;
        s.prefix = 0ull;
        s.k_rem = (unsigned)min((int64_t)k, n);
        s.shift = 64;
        s.done = (n <= k) ? 1 : 0;     // everything is selected: threshold key 0 (no live key is 0)
        s.n_items = (unsigned)n;
        s.out_cnt = 0;
        st[b] = s;
    }
    for (int i = threadIdx.x; i < GS_SEL_BINS; i += blockDim.x) hist[b * GS_SEL_BINS + i] = 0;
}

// histogram of the next digit over the items whose decided bits equal the prefix
template <int WT>
__global__ void __launch_bounds__(kSelThreads) k_sel_hist(gs_sel_src src, const SelState* __restrict__ st,
                                                          uint32_t* __restrict__ hist) {
    const int64_t b = blockIdx.y;
    const SelState s = st[b];
    if (s.done) return;
    const int64_t n = src_count(src, b);
    const int64_t i0 = (int64_t)blockIdx.x * kItemsPerCta;
    if (i0 >= n) return;
    __shared__ uint32_t sh[GS_SEL_BINS];
    for (int i = threadIdx.x; i < GS_SEL_BINS; i += kSelThreads) sh[i] = 0;
    __syncthreads();
    const int width = min(GS_SEL_BITS, s.shift);
    const int lo = s.shift - width;                          // digit = bits [lo, lo+width)
    const uint64_t himask = s.shift >= 64 ? 0ull : ~((1ull << s.shift) - 1ull);
    const int64_t i1 = min(n, i0 + kItemsPerCta);
    for (int64_t i = i0 + threadIdx.x; i < i1; i += kSelThreads) {
        const uint64_t key = src_key<WT>(src, b, i);
        if (key != 0ull && (key & himask) == s.prefix) atomicAdd(&sh[(key >> lo) & ((1u << width) - 1u)], 1u);
    }
    __syncthreads();
    for (int i = threadIdx.x; i < GS_SEL_BINS; i += kSelThreads)
        if (sh[i]) atomicAdd(&hist[b * GS_SEL_BINS + i], sh[i]);
}

// pick the digit value that contains the k_rem-th largest item, update the state, clear the histogram
__global__ void __launch_bounds__(GS_SEL_BINS / 4) k_sel_scan(SelState* __restrict__ st, uint32_t* __restrict__ hist) {
    const int64_t b = blockIdx.x;
    SelState s = st[b];
    if (s.done) return;
    uint32_t* h = hist + b * GS_SEL_BINS;
    __shared__ uint32_t part[GS_SEL_BINS / 4];
    __shared__ int sel_bin;
    __shared__ uint32_t sel_above, sel_cnt;
    const int tid = threadIdx.x;               // thread tid owns bins [4*tid, 4*tid+4), scanned from the TOP
    uint32_t c[4], tot = 0;
    for (int j = 0; j < 4; ++j) { c[j] = h[4 * tid + j]; tot += c[j]; }
    part[tid] = tot;
    __syncthreads();
    // suffix sums over threads (512 partials): simple log-step scan in shared memory
    for (int o = 1; o < GS_SEL_BINS / 4; o <<= 1) {
        uint32_t v = (tid + o < GS_SEL_BINS / 4) ? part[tid + o] : 0;
        __syncthreads();
        part[tid] += v;
        __syncthreads();
    }
    uint32_t above = part[tid] - tot;          // items in bins strictly above this thread's bins
    for (int j = 3; j >= 0; --j) {
        if (above < s.k_rem && above + c[j] >= s.k_rem) { sel_bin = 4 * tid + j; sel_above = above; sel_cnt = c[j]; }
        above += c[j];
    }
    __syncthreads();
    for (int j = 0; j < 4; ++j) h[4 * tid + j] = 0;
    if (tid == 0) {
        const int width = min(GS_SEL_BITS, s.shift);
        const int lo = s.shift - width;
        s.prefix |= (unsigned long long)sel_bin << lo;
        s.k_rem -= sel_above;
        s.shift = lo;
        // every item of the chosen bin is wanted, or no bits are left: the threshold is decided
        if (sel_cnt == s.k_rem || lo == 0) s.done = 1;
        st[b] = s;
    }
}

// collect the items with key >= threshold: exactly k_total of them (all keys are distinct)
template <int WT>
__global__ void __launch_bounds__(kSelThreads) k_sel_collect(gs_sel_src src, SelState* __restrict__ st, int32_t k,
                                                             uint64_t* __restrict__ sel) {
    const int64_t b = blockIdx.y;
    const int64_t n = src_count(src, b);
    const int64_t i0 = (int64_t)blockIdx.x * kItemsPerCta;
    if (i0 >= n) return;
    const uint64_t thr = st[b].prefix;
    const int64_t i1 = min(n, i0 + kItemsPerCta);
    for (int64_t i = i0 + threadIdx.x; i < i1; i += kSelThreads) {
        const uint64_t key = src_key<WT>(src, b, i);
        if (key != 0ull && key >= thr) {
            const unsigned pos = atomicAdd(&st[b].out_cnt, 1u);
            if (pos < (unsigned)k) sel[b * k + pos] = key;
        }
    }
}

// bitonic sort (descending) of the selected keys, then decode (id, score); also the k-th key
template <int WT>
__global__ void k_sel_sort(const SelState* __restrict__ st, const uint64_t* __restrict__ sel, int32_t k, int kp2,
                           int32_t* __restrict__ out_ids, uint32_t* __restrict__ out_scores,
                           uint64_t* __restrict__ out_thr, uint64_t* __restrict__ out_keys,
                           uint32_t* __restrict__ out_cnt, int64_t out_cap) {
    extern __shared__ uint64_t sk[];
    const int64_t b = blockIdx.x;
    const unsigned cnt = min(st[b].out_cnt, (unsigned)k);
    for (int i = threadIdx.x; i < kp2; i += blockDim.x) sk[i] = (unsigned)i < cnt ? sel[b * k + i] : 0ull;
    __syncthreads();
    for (int size = 2; size <= kp2; size <<= 1) {
        for (int stride = size >> 1; stride > 0; stride >>= 1) {
            if (stride >= 32) {
                for (int i = threadIdx.x; i < kp2 / 2; i += blockDim.x) {
                    const int lo = 2 * i - (i & (stride - 1));
                    const int hi = lo + stride;
                    const bool desc = (lo & size) == 0;
                    const uint64_t x = sk[lo], y = sk[hi];
                    if ((x < y) == desc) { sk[lo] = y; sk[hi] = x; }
                }
                __syncthreads();
            } else {
                // strides < 32: finish this merge step inside warps with shuffles
                for (int base = 0; base < kp2; base += blockDim.x) {
                    const int i = base + threadIdx.x;
                    uint64_t v = i < kp2 ? sk[i] : 0ull;
                    for (int st2 = stride; st2 > 0; st2 >>= 1) {
                        const uint64_t o = __shfl_xor_sync(0xFFFFFFFFu, v, st2);
                        const bool lower = (i & st2) == 0;
                        const bool desc = (i & size) == 0;
                        const bool take_max = lower == desc;
                        v = take_max ? (v > o ? v : o) : (v < o ? v : o);
                    }
                    if (i < kp2) sk[i] = v;
                }
                __syncthreads();
                break;
            }
        }
    }
    for (int i = threadIdx.x; i < k; i += blockDim.x) {
        const uint64_t key = sk[i];
        if (out_ids) {
            if (key == 0ull) {
                out_ids[b * k + i] = -1;
                out_scores[b * k + i] = WT == GS_W_F32 ? 0xFF800000u : 0x80000000u;   // -inf | INT32_MIN
            } else {
                out_ids[b * k + i] = (int32_t)(0xFFFFFFFFu - (uint32_t)key);
                const uint32_t o = (uint32_t)(key >> 32);
                out_scores[b * k + i] = WT == GS_W_F32 ? gs_unord_f32(o) : (o ^ 0x80000000u);
            }
        }
        if (out_keys && key != 0ull) out_keys[b * out_cap + i] = key;
    }
    if (threadIdx.x == 0) {
        // threshold for the filter phase: the k-th best key seen so far, or 0 when fewer than k exist
        if (out_thr) out_thr[b] = cnt >= (unsigned)k ? sk[k - 1] : 0ull;
        if (out_cnt) out_cnt[b] = cnt;
    }
}

// ---- one thread-block CLUSTER per row: the whole select (histogram passes, pick, collect, bitonic sort, decode) in
// ONE launch.  Used when a row has at most kRowFusedMax items (candidate lists, threshold samples).  The CTAs of a
// cluster split the row; each keeps a histogram in its own shared memory, every CTA sums the cluster's histograms
// through distributed shared memory and takes the same decision, the selected keys are gathered in CTA 0's shared
// memory (remote atomics, aggregated per warp), which sorts and decodes them.  The row is re-read from L2 once per
// digit.  15 launches become 1 — what a batch-1 search spends its time on once scoring takes 0.15 ms — and a
// large batch keeps all SMs busy with one cluster per query.
constexpr int kRowThreads = 1024;
constexpr int64_t kRowFusedMax = 1 << 20;
constexpr int kRowUnroll = 4;

template <int WT>
__global__ void __launch_bounds__(kRowThreads, 2) k_sel_row(gs_sel_src src, int32_t k, int kp2, int32_t* __restrict__ out_ids,
                                                         uint32_t* __restrict__ out_scores, uint64_t* __restrict__ out_thr) {
    namespace cg = cooperative_groups;
    cg::cluster_group cluster = cg::this_cluster();
    const int C = (int)cluster.num_blocks(), rank = (int)cluster.block_rank();
    extern __shared__ __align__(16) unsigned char sm_raw[];
    uint64_t* sk = reinterpret_cast<uint64_t*>(sm_raw);                        // [kp2]   (used in CTA 0)
    uint32_t* hist = reinterpret_cast<uint32_t*>(sk + kp2);                    // [GS_SEL_BINS]
    __shared__ uint32_t part[kRowThreads / 32];
    __shared__ unsigned long long s_prefix;
    __shared__ uint32_t s_krem, s_cnt;
    __shared__ int s_shift, s_done;
    __shared__ long long s_live;                                               // dense rows: columns [0, s_live) are documents
    const int64_t b = blockIdx.x / C;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int64_t n = src_count(src, b);
    const int64_t per = ((n + C - 1) / C + 3) / 4 * 4;                         // this CTA's slice of the row
    const int64_t i_lo = min(n, per * rank), i_hi = min(n, i_lo + per);
    if (tid == 0) {
        int64_t live = n;
        if (!src.keys) {
            live = 0;
            if (src.Ts > 0) {
                for (int64_t j = 0; j < src.ts.count; ++j) {
                    const int64_t d0 = ((int64_t)src.ts.first + j * src.ts.stride) * src.Ts;
                    live += max((int64_t)0, min((int64_t)src.Ts, src.n_docs - d0));
                }
            } else live = min(n, src.n_docs);
        }
        s_prefix = 0ull;
        s_krem = (uint32_t)min((int64_t)k, live);
        s_shift = 64;
        s_done = live <= k ? 1 : 0;            // everything is selected: threshold key 0 (no live key is 0)
        s_cnt = 0;
        s_live = live;                         // (columns are in doc order: only the end of the last tile can lie past the last document)
    }
    __syncthreads();
    // Dense rows: while the digit lies in the score half of the key (digits never straddle bit 32: 11 + 11 + 10 bits, twice)
    // an item is its 32 ordered score bits — no doc id, no 64-bit key; the doc half is only looked at to split score ties
    // (rare) and for the few items the collect pass takes.
    const bool dense = src.keys == nullptr;
    const uint32_t* drow = dense ? src.dense + b * src.ld : nullptr;
    const int64_t d_hi = dense ? min(i_hi, (int64_t)s_live) : 0;
    while (!s_done) {                          // every CTA of the cluster takes the same decisions
        const int shift = s_shift;
        const unsigned long long prefix = s_prefix;
        const int width = min(GS_SEL_BITS, shift > 32 ? shift - 32 : shift);
        const int lo = shift - width;
        const uint64_t himask = shift >= 64 ? 0ull : ~((1ull << shift) - 1ull);
        for (int i = tid; i < GS_SEL_BINS; i += kRowThreads) hist[i] = 0;
        __syncthreads();
        if (dense && lo >= 32) {
            const uint32_t pre32 = (uint32_t)(prefix >> 32), hm32 = (uint32_t)(himask >> 32);
            const int lo32 = lo - 32;
            for (int64_t base = i_lo; base < d_hi; base += kRowUnroll * kRowThreads) {
                uint32_t o[kRowUnroll];
#pragma unroll
                for (int u = 0; u < kRowUnroll; ++u) {
                    const int64_t i = base + tid + (int64_t)u * kRowThreads;
                    o[u] = i < d_hi ? gs_ord_bits<WT>(drow[i]) : 0u;
                }
#pragma unroll
                for (int u = 0; u < kRowUnroll; ++u) {
                    const bool live = base + tid + (int64_t)u * kRowThreads < d_hi && (o[u] & hm32) == pre32;
                    const uint32_t digit = live ? ((o[u] >> lo32) & ((1u << width) - 1u)) : 0xFFFFFFFFu;
                    // lanes of a warp mostly share the digit in the first pass (leading score bits) and mostly differ in
                    // the later ones: one atomic for the warp when all agree, one per lane otherwise
                    const uint32_t d0 = __shfl_sync(0xFFFFFFFFu, digit, 0);
                    if (__all_sync(0xFFFFFFFFu, digit == d0)) {
                        if (lane == 0 && live) atomicAdd(&hist[digit], 32u);
                    } else if (live) atomicAdd(&hist[digit], 1u);
                }
            }
        } else
        for (int64_t base = i_lo; base < i_hi; base += kRowUnroll * kRowThreads) {   // uniform trip count; loads in flight
            uint64_t key[kRowUnroll];
#pragma unroll
            for (int u = 0; u < kRowUnroll; ++u) {
                const int64_t i = base + tid + (int64_t)u * kRowThreads;
                key[u] = i < i_hi ? src_key<WT>(src, b, i) : 0ull;
            }
#pragma unroll
            for (int u = 0; u < kRowUnroll; ++u) {
                // scores share their leading bits, so a digit's counter is hot: one atomic per distinct digit per warp
                const bool live = key[u] != 0ull && (key[u] & himask) == prefix;
                const uint32_t digit = live ? (uint32_t)((key[u] >> lo) & ((1u << width) - 1u)) : 0xFFFFFFFFu;
                const uint32_t d0 = __shfl_sync(0xFFFFFFFFu, digit, 0);        // as in the dense passes above
                if (__all_sync(0xFFFFFFFFu, digit == d0)) {
                    if (lane == 0 && live) atomicAdd(&hist[digit], 32u);
                } else if (live) atomicAdd(&hist[digit], 1u);
            }
        }
        cluster.sync();
        // thread t owns bins 2t, 2t+1 (summed over the cluster); suffix sums from the top bin down
        uint32_t c0 = 0, c1 = 0;
        for (int r = 0; r < C; ++r) {
            const uint2 v = *reinterpret_cast<const uint2*>(cluster.map_shared_rank(hist, r) + 2 * tid);
            c0 += v.x;
            c1 += v.y;
        }
        uint32_t incl = c0 + c1;                                  // inclusive suffix sum over threads >= tid
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t v = __shfl_down_sync(0xFFFFFFFFu, incl, o);
            if (lane + o < 32) incl += v;
        }
        if (lane == 0) part[warp] = incl;
        __syncthreads();
        if (warp == 0) {
            uint32_t v = part[lane], inc2 = v;
            for (int o = 1; o < 32; o <<= 1) {
                const uint32_t u = __shfl_down_sync(0xFFFFFFFFu, inc2, o);
                if (lane + o < 32) inc2 += u;
            }
            part[lane] = inc2 - v;                                // items in warps above this one
        }
        __syncthreads();
        const uint32_t k_rem = s_krem;
        uint32_t above = part[warp] + incl - (c0 + c1);           // items in bins strictly above this thread's bins
        cluster.sync();                                           // all remote reads done before the next zeroing; s_krem read
        for (int j = 1; j >= 0; --j) {
            const uint32_t c = j ? c1 : c0;
            if (above < k_rem && above + c >= k_rem) {            // exactly one (thread, bin) matches
                s_prefix = prefix | ((unsigned long long)(2 * tid + j) << lo);
                s_krem = k_rem - above;
                s_shift = lo;
                if (c == k_rem - above || lo == 0) s_done = 1;    // the whole bin is wanted, or no bits are left
            }
            above += c;
        }
        __syncthreads();
    }
    // Threshold-only call (the sample select of a search: no ids, no scores): once the score half of the key is resolved,
    // the prefix itself — selected digits, zeros below — is the answer.  The keys >= prefix are exactly the k selected
    // ones, so it bounds the k-th key from below and differs from it in doc-id bits only; the filter that uses it
    // (key >= threshold) lets the same sample cells pass.  Skips the collect pass, two cluster barriers and the sort
    // (a third of this launch at one row).  The loop ran (more than k live keys) whenever s_shift has left 64.
    if (out_ids == nullptr && out_thr != nullptr && s_shift <= 32) {
        if (rank == 0 && tid == 0) out_thr[b] = s_prefix;
        return;                                // no CTA reads another's shared memory after the loop's last cluster barrier
    }
    // collect the keys >= threshold (exactly min(k, live) of them: all keys are distinct) in CTA 0, sort, decode
    const uint64_t thr = s_prefix;
    if (rank == 0)
        for (int i = tid; i < kp2; i += kRowThreads) sk[i] = 0ull;
    cluster.sync();
    uint64_t* sk0 = cluster.map_shared_rank(sk, 0);
    uint32_t* cnt0 = cluster.map_shared_rank(&s_cnt, 0);
    for (int64_t base = i_lo; base < i_hi; base += kRowUnroll * kRowThreads) {
        uint64_t key[kRowUnroll];
        if (dense) {                           // the full key only of items whose score reaches the threshold's
            uint32_t o[kRowUnroll];
#pragma unroll
            for (int u = 0; u < kRowUnroll; ++u) {
                const int64_t i = base + tid + (int64_t)u * kRowThreads;
                o[u] = i < d_hi ? gs_ord_bits<WT>(drow[i]) : 0u;
            }
#pragma unroll
            for (int u = 0; u < kRowUnroll; ++u) {
                const int64_t i = base + tid + (int64_t)u * kRowThreads;
                key[u] = (i < d_hi && o[u] >= (uint32_t)(thr >> 32)) ? src_key<WT>(src, b, i) : 0ull;
            }
        } else {
#pragma unroll
            for (int u = 0; u < kRowUnroll; ++u) {
                const int64_t i = base + tid + (int64_t)u * kRowThreads;
                key[u] = i < i_hi ? src_key<WT>(src, b, i) : 0ull;
            }
        }
#pragma unroll
        for (int u = 0; u < kRowUnroll; ++u) {
            const bool take = key[u] != 0ull && key[u] >= thr;
            const unsigned m = __ballot_sync(0xFFFFFFFFu, take);
            if (m) {
                uint32_t pos0 = 0;
                if (lane == __ffs(m) - 1) pos0 = atomicAdd(cnt0, (uint32_t)__popc(m));
                pos0 = __shfl_sync(0xFFFFFFFFu, pos0, __ffs(m) - 1);
                const uint32_t pos = pos0 + __popc(m & ((1u << lane) - 1u));
                if (take && pos < (uint32_t)k) sk0[pos] = key[u];
            }
        }
    }
    cluster.sync();
    if (rank != 0) return;
    const uint32_t cnt = min(s_cnt, (uint32_t)k);
    for (int size = 2; size <= kp2; size <<= 1) {
        for (int stride = size >> 1; stride > 0; stride >>= 1) {
            for (int i = tid; i < kp2 / 2; i += kRowThreads) {
                const int lo2 = 2 * i - (i & (stride - 1));
                const int hi2 = lo2 + stride;
                const bool desc = (lo2 & size) == 0;
                const uint64_t x = sk[lo2], y = sk[hi2];
                if ((x < y) == desc) { sk[lo2] = y; sk[hi2] = x; }
            }
            __syncthreads();
        }
    }
    for (int i = tid; i < k; i += kRowThreads) {
        const uint64_t key = sk[i];
        if (out_ids) {
            if (key == 0ull) {
                out_ids[b * k + i] = -1;
                out_scores[b * k + i] = WT == GS_W_F32 ? 0xFF800000u : 0x80000000u;   // -inf | INT32_MIN
            } else {
                out_ids[b * k + i] = (int32_t)(0xFFFFFFFFu - (uint32_t)key);
                const uint32_t o = (uint32_t)(key >> 32);
                out_scores[b * k + i] = WT == GS_W_F32 ? gs_unord_f32(o) : (o ^ 0x80000000u);
            }
        }
    }
    if (tid == 0 && out_thr) out_thr[b] = cnt >= (uint32_t)k ? sk[k - 1] : 0ull;
}

struct Scratch { SelState* st; uint32_t* hist; uint64_t* sel; };
Scratch carve(void* scratch, int64_t rows, int32_t k) {
    unsigned char* p = (unsigned char*)scratch;
    Scratch s;
    s.st = (SelState*)p;
    p += ((size_t)rows * sizeof(SelState) + 255) / 256 * 256;
    s.hist = (uint32_t*)p;
    p += ((size_t)rows * GS_SEL_BINS * 4 + 255) / 256 * 256;
    s.sel = (uint64_t*)p;
    (void)k;
    return s;
}

template <int WT>
gs_status_t run_select(const gs_sel_src& src, int64_t rows, int32_t k, int32_t* out_ids, void* out_scores,
                       uint64_t* out_thr, uint64_t* out_keys, uint32_t* out_cnt, int64_t out_cap, void* scratch,
                       cudaStream_t s) {
    Scratch sc = carve(scratch, rows, k);
    const int64_t max_items = src.keys ? src.cap : src.n_cols;
    const unsigned chunks = (unsigned)std::max<int64_t>(1, (max_items + kItemsPerCta - 1) / kItemsPerCta);
    if (rows > 65535) return GS_ERR_OUT_OF_RANGE;
    if (max_items <= kRowFusedMax && !out_keys && !out_cnt) {
        int kp2 = 32;
        while (kp2 < k) kp2 <<= 1;
        const size_t smem = (size_t)kp2 * 8 + GS_SEL_BINS * 4;
        GS_CUDA(gs_optin_smem(k_sel_row<WT>));
        // CTAs per row: enough to spread a few rows over the chip, one when there are rows to spare
        int C = 1;
        while (C < 8 && rows * C < GS_SEL_TARGET && max_items > (int64_t)C * 8192) C <<= 1;
        cudaLaunchConfig_t cfg{};
        cfg.gridDim = dim3((unsigned)(rows * C));
        cfg.blockDim = dim3(kRowThreads);
        cfg.dynamicSmemBytes = smem;
        cfg.stream = s;
        cudaLaunchAttribute attr[1];
        attr[0].id = cudaLaunchAttributeClusterDimension;
        attr[0].val.clusterDim.x = (unsigned)C;
        attr[0].val.clusterDim.y = 1;
        attr[0].val.clusterDim.z = 1;
        cfg.attrs = attr;
        cfg.numAttrs = 1;
        {
            GsProfScope ps(GS_K_SELECT, s);
            GS_CUDA(cudaLaunchKernelEx(&cfg, k_sel_row<WT>, src, k, kp2, out_ids, (uint32_t*)out_scores, out_thr));
        }
        ++gs_tls_launches;
        GS_CUDA(cudaGetLastError());
        return GS_OK;
    }
    {
        GsProfScope ps(GS_K_SELECT, s, 14);
        k_sel_init<<<(unsigned)rows, 256, 0, s>>>(src, rows, k, sc.st, sc.hist);
        ++gs_tls_launches;
        for (int shift = 64; shift > 0; shift -= GS_SEL_BITS) {
            k_sel_hist<WT><<<dim3(chunks, (unsigned)rows), kSelThreads, 0, s>>>(src, sc.st, sc.hist);
            k_sel_scan<<<(unsigned)rows, GS_SEL_BINS / 4, 0, s>>>(sc.st, sc.hist);
            gs_tls_launches += 2;
        }
        k_sel_collect<WT><<<dim3(chunks, (unsigned)rows), kSelThreads, 0, s>>>(src, sc.st, k, sc.sel);
        ++gs_tls_launches;
    }
    int kp2 = 32;
    while (kp2 < k) kp2 <<= 1;
    const int threads = std::min(1024, std::max(32, kp2));
    {
        GsProfScope ps(GS_K_SORT, s);
        k_sel_sort<WT><<<(unsigned)rows, threads, (size_t)kp2 * 8, s>>>(sc.st, sc.sel, k, kp2, out_ids, (uint32_t*)out_scores,
                                                                       out_thr, out_keys, out_cnt, out_cap);
    }
    ++gs_tls_launches;
    GS_CUDA(cudaGetLastError());
    return GS_OK;
}

}  // namespace

size_t gs_select_scratch_bytes(int64_t rows, int32_t k) {
    size_t b = ((size_t)rows * sizeof(SelState) + 255) / 256 * 256;
    b += ((size_t)rows * GS_SEL_BINS * 4 + 255) / 256 * 256;
    b += ((size_t)rows * (size_t)k * 8 + 255) / 256 * 256;
    return b;
}

gs_status_t gs_launch_select(const gs_sel_src& src, int64_t rows, int32_t k, int32_t* out_ids, void* out_scores,
                             uint64_t* out_thr, uint64_t* out_keys, uint32_t* out_cnt, int64_t out_cap, void* scratch,
                             cudaStream_t s) {
    if (rows <= 0) return GS_OK;
    return src.wtype == GS_W_F32
               ? run_select<GS_W_F32>(src, rows, k, out_ids, out_scores, out_thr, out_keys, out_cnt, out_cap, scratch, s)
               : run_select<GS_W_U8>(src, rows, k, out_ids, out_scores, out_thr, out_keys, out_cnt, out_cap, scratch, s);
}

// ------------------------------------------------------------------------------------------------
// gs_topk_dense_static: gs_topk_dense for callers that cannot allocate (CUDA graph capture, serving loops, harnesses that
// forbid cudaMalloc) — the select's scratch (per-row state, digit histograms, selected keys: what gs_topk_dense takes as
// `workspace`) lives in a file-scope device array instead.  Every GPU that loads the library holds the array until the
// process exits, so it is modest: GS_TOPK_STATIC_SCRATCH_BYTES.
//
// In host code the array's NAME is a host-side stand-in, not a device address (a kernel handed it would fault or, where the
// GPU can reach host memory, silently use the wrong memory): the device address comes from cudaGetSymbolAddress, asked once
// per device with that device current and kept.  All calls share the array and it keeps the last call's contents: the first
// launch of every call (k_sel_init) re-initialises the state and the histograms of the rows in use, and the selected-key
// region is only read where this call wrote it, so nothing has to be cleared by the caller — but two calls that overlap on
// the GPU (different streams, or the same stream from two threads without ordering) race on it.
// Calls no cudaMalloc / cudaFree / allocating library routine.
// ------------------------------------------------------------------------------------------------
static __device__ __align__(256) unsigned char g_topk_static_scratch[GS_TOPK_STATIC_SCRATCH_BYTES];

namespace {
constexpr int kMaxDevices = 64;
std::mutex g_static_mu;
void* g_static_ptr[kMaxDevices] = {};      // device address of g_topk_static_scratch, per device

gs_status_t static_scratch(void** out) {
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) { cudaGetLastError(); return GS_ERR_UNSUPPORTED_DEVICE; }
    if (dev < 0 || dev >= kMaxDevices) return GS_ERR_UNSUPPORTED_DEVICE;
    int major = 0;
    if (cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev) != cudaSuccess) { cudaGetLastError(); return GS_ERR_UNSUPPORTED_DEVICE; }
    if (major != 10) return GS_ERR_UNSUPPORTED_DEVICE;          // the library holds sm_100a code only
    std::lock_guard<std::mutex> lock(g_static_mu);
    if (g_static_ptr[dev] == nullptr) {
        void* ptr = nullptr;
        GS_CUDA(cudaGetSymbolAddress(&ptr, g_topk_static_scratch));   // device `dev` is current
        if (ptr == nullptr) return GS_ERR_CUDA;
        g_static_ptr[dev] = ptr;
    }
    *out = g_static_ptr[dev];
    return GS_OK;
}

bool on_device(const void* p) {
    if (!p) return false;
    cudaPointerAttributes a{};
    if (cudaPointerGetAttributes(&a, p) != cudaSuccess) { cudaGetLastError(); return false; }
    return a.type == cudaMemoryTypeDevice || a.type == cudaMemoryTypeManaged;
}
}  // namespace

extern "C" GS_API gs_status_t gs_topk_dense_static(const void* scores, int32_t wtype, int64_t rows, int64_t n, int64_t ld, int32_t k,
                                                   int32_t* out_ids, void* out_scores, gs_stream_t stream) {
    if (!out_ids || !out_scores || rows < 0 || n < 0 || ld < n) return GS_ERR_INVALID_ARG;
    if (wtype != GS_W_F32 && wtype != GS_W_U8) return GS_ERR_INVALID_ARG;
    if (k < 1 || k > GS_MAX_K) return GS_ERR_OUT_OF_RANGE;
    if (rows > 65535 || n >= 0x7FFFFFFFLL) return GS_ERR_OUT_OF_RANGE;
    // the maximum: the call's scratch need must fit the static array
    if (gs_select_scratch_bytes(rows, k) > (size_t)GS_TOPK_STATIC_SCRATCH_BYTES) return GS_ERR_OUT_OF_RANGE;
    void* scratch = nullptr;
    GS_TRY(static_scratch(&scratch));
    if (n > 0 && rows > 0 && !on_device(scores)) return GS_ERR_INVALID_ARG;
    if (!on_device(out_ids) || !on_device(out_scores)) return GS_ERR_INVALID_ARG;
    gs_tls_launches = 0;
    gs_sel_src src{};
    src.dense = (const uint32_t*)scores; src.ld = ld; src.n_cols = n; src.n_docs = n; src.Ts = 0; src.wtype = wtype;
    return gs_launch_select(src, rows, k, out_ids, out_scores, nullptr, nullptr, nullptr, 0, scratch, (cudaStream_t)stream);
}
