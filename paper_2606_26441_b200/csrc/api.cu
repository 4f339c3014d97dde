// api.cu — the C ABI of include/gpusparse.h: argument checks, workspace carving and the search plan.
//
// Search plan.  The paper materialises a [B,N] fp32 score buffer (17.6 GB at
// B=500, N=8.8M: PAPER.md L125, L310, L410) and runs torch.topk over it.  Here the scoring kernels
// hand every (query, doc) cell to a sink:
//   1. sample : score 1/2^shift of the doc tiles densely, radix-select the k-th best key per query.
//               The k-th best of ANY subset is a lower bound of the global k-th best.
//   2. filter : score ALL tiles; a cell is appended to its query's candidate list iff key >= bound.
//               Every true top-k document passes, so the result stays exact.
//   3. final  : radix-select + bitonic sort over the candidate lists -> (ids, scores).
//   4. a query whose candidate list overflowed is re-run through the dense path (exact, slower).
// GS_FLAG_FORCE_DENSE_TOPK (or a collection of only a few tiles) uses the dense path for everything.
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <new>
#include <set>
#include <utility>
#include <vector>

#include "gs_internal.cuh"

gs_status_t gs_build_index_impl(gs_index* ix, const gs_csr_t* docs, const gs_build_opts_t& o, cudaStream_t s);
size_t gs_score_doc_scratch_bytes_ex(const gs_index* ix, int qtile, int64_t nq, int64_t q_nnz);

thread_local int32_t gs_tls_launches = 0;
static thread_local int32_t tls_cuda_error = 0;
void gs_set_cuda_error(cudaError_t e) { tls_cuda_error = (int32_t)e; cudaGetLastError(); }

cudaError_t gs_optin_smem_impl(const void* kern) {
    static std::mutex mu;
    static std::set<std::pair<const void*, int>> done;
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    std::lock_guard<std::mutex> lock(mu);
    if (done.count({kern, dev})) return cudaSuccess;
    int smem_max = 0;
    e = cudaDeviceGetAttribute(&smem_max, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
    if (e != cudaSuccess) return e;
    cudaFuncAttributes fa{};
    e = cudaFuncGetAttributes(&fa, kern);
    if (e != cudaSuccess) return e;
    // the opt-in limit covers static + dynamic shared memory
    e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_max - (int)fa.sharedSizeBytes);
    if (e == cudaSuccess) done.insert({kern, dev});
    return e;
}

// ---- kernel timing (gs_profile_*): thread-local list of event pairs
namespace {
struct ProfRec { int kclass; int n; cudaEvent_t a, b; };
thread_local bool tls_prof_on = false;
thread_local std::vector<ProfRec> tls_prof;
thread_local std::vector<cudaEvent_t> tls_event_pool;
cudaEvent_t prof_event() {
    if (!tls_event_pool.empty()) { cudaEvent_t e = tls_event_pool.back(); tls_event_pool.pop_back(); return e; }
    cudaEvent_t e = nullptr;
    if (cudaEventCreate(&e) != cudaSuccess) { cudaGetLastError(); return nullptr; }
    return e;
}
}  // namespace

GsProfScope::GsProfScope(int kclass, cudaStream_t s, int n) : stream(s) {
    if (!tls_prof_on) return;
    ProfRec r{kclass, n, prof_event(), prof_event()};
    if (!r.a || !r.b) return;
    cudaEventRecord(r.a, s);
    tls_prof.push_back(r);
    slot = (int)tls_prof.size() - 1;
}
GsProfScope::~GsProfScope() {
    if (slot >= 0) cudaEventRecord(tls_prof[slot].b, stream);
}

namespace {

inline size_t up256(size_t b) { return (b + 255) / 256 * 256; }

bool is_device_ptr(const void* p) {
    if (!p) return false;
    cudaPointerAttributes a{};
    if (cudaPointerGetAttributes(&a, p) != cudaSuccess) { cudaGetLastError(); return false; }
    return a.type == cudaMemoryTypeDevice || a.type == cudaMemoryTypeManaged;
}

gs_status_t check_device() {
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) { cudaGetLastError(); return GS_ERR_UNSUPPORTED_DEVICE; }
    int major = 0;
    if (cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev) != cudaSuccess) {
        cudaGetLastError();
        return GS_ERR_UNSUPPORTED_DEVICE;
    }
    return major == 10 ? GS_OK : GS_ERR_UNSUPPORTED_DEVICE;   // the library holds sm_100a code only
}

gs_status_t check_csr_host(const gs_csr_t* c, bool device) {
    if (!c || c->rows < 0 || c->nnz < 0 || !c->indptr) return GS_ERR_INVALID_ARG;
    if (c->wtype != GS_W_F32 && c->wtype != GS_W_U8) return GS_ERR_INVALID_ARG;
    if (c->nnz > 0 && (!c->term_ids || !c->weights)) return GS_ERR_INVALID_ARG;
    if (device) {
        if (!is_device_ptr(c->indptr)) return GS_ERR_INVALID_ARG;
        if (c->nnz > 0 && (!is_device_ptr(c->term_ids) || !is_device_ptr(c->weights))) return GS_ERR_INVALID_ARG;
    }
    return GS_OK;
}

// device-side stats block at the start of every search workspace
struct StatsBlock { gs_stats_t stats; int32_t status; int32_t n_overflow; };

struct PlanStats { int32_t launches, algo, sample_tiles, qtile, passes, group; };

__global__ void k_finalize_stats(StatsBlock* sb, const uint32_t* cand_cnt, int64_t B, int64_t cap, int32_t* overflow_list,
                                 PlanStats ps) {
    __shared__ unsigned long long tot;
    __shared__ int n_ov;
    if (threadIdx.x == 0) { tot = 0; n_ov = 0; }
    __syncthreads();
    unsigned long long local = 0;
    for (int64_t b = threadIdx.x; b < B; b += blockDim.x) {
        const uint32_t c = cand_cnt ? cand_cnt[b * GS_CNT_STRIDE] : 0u;
        local += c;
        if (cand_cnt && (int64_t)c > cap) overflow_list[atomicAdd(&n_ov, 1)] = (int32_t)b;
    }
    atomicAdd(&tot, local);
    __syncthreads();
    if (threadIdx.x == 0) {
        sb->stats.candidates = (int64_t)tot;
        sb->stats.overflow_queries = n_ov;
        sb->stats.launches = ps.launches;
        sb->stats.algo_used = ps.algo;
        sb->stats.sample_tiles = ps.sample_tiles;
        sb->stats.doc_query_tile = ps.qtile;
        sb->stats.doc_passes = ps.passes;
        sb->stats.query_group = ps.group;
        sb->n_overflow = n_ov;
    }
}

__global__ void k_zero_u32(uint32_t* p, int64_t n) {
    int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (i < n) p[i] = 0u;
}

struct Plan {
    int algo = GS_ALGO_TERM_PARALLEL;
    uint32_t flags = 0;
    int group = 0, qtile = 32;
    bool dense_only = false;
    int stride = 1;            // sample = every stride-th tile
    int sample_tiles = 0;
    int64_t cand_cap = 0;
    bool use_head = true;
};

// Bytes one document-parallel pass streams: the tail block CSR plus the head strips (not the second tier)
int64_t stream_bytes(const gs_index* ix) {
    return ix->bytes_forward + (int64_t)ix->H * ix->N_pad * (ix->wtype == GS_W_F32 ? 4 : 1);
}

// `nnz` = entries of the query batch (known on the host: gs_csr_t.nnz), so the choice needs no device round trip
Plan make_plan(const gs_index* ix, int64_t B, int64_t nnz, int32_t k, const gs_search_opts_t* o) {
    Plan p;
    p.algo = GS_ALGO_TERM_PARALLEL;
    if (o) {
        // AUTO: the cost model of gs_dispatch_model (crossover of PAPER.md L176-181 with the forms and constants measured
        // on B200): term-parallel for batches, document-parallel for one or two long queries
        p.algo = o->algo == GS_ALGO_AUTO ? gs_dispatch_model(ix->N, ix->Ts, stream_bytes(ix), B, nnz, nullptr, nullptr) : o->algo;
        p.flags = o->flags;
        p.group = o->query_group;
        p.qtile = o->doc_query_tile;
    }
    // doc-parallel, queries per pass: 16 is the largest tile that stays HBM bound in fp32; the integer
    // kernel is issue bound at every size and a pass of 32 queries costs it less than two of 16 (44.5 vs 54.2 ms per
    // 500-query batch at 8.8M docs)
    if (p.qtile <= 0) p.qtile = B <= 8 ? 8 : (ix->wtype == GS_W_U8 && B >= 32 ? 32 : 16);
    p.use_head = !(p.flags & GS_FLAG_NO_HEAD_STRIPS);
    // Threshold sample = 1/2^shift of the doc tiles.  The select phases read the sample (N/2^shift cells per query) and
    // the candidates (about k*2^shift per query), so the balance is 2^shift ~ sqrt(N/k); the candidate lists
    // (8*k*2^shift keys per query) are kept under 2 GiB for the batch, and never below the 1/32 sample.
    int shift = 5;
    if (o && o->sample_shift > 0) {
        shift = std::min(o->sample_shift, 16);        // 1 .. 16; larger values would overflow the stride
    } else if (ix->N > 0) {
        const double r = std::sqrt((double)ix->N / (double)k);
        while (shift < 10 && (double)(1 << (shift + 1)) <= r * 1.4142) ++shift;
        while (shift > 5 && (double)B * 8.0 * (double)k * (double)(1 << shift) * 8.0 > 2147483648.0) --shift;
    }
    // the sample must hold comfortably more than k documents, else its k-th key is a weak bound
    while (shift > 0 && ((int64_t)(ix->ntiles >> shift)) * ix->Ts < 4 * (int64_t)k) --shift;
    p.dense_only = (p.flags & GS_FLAG_FORCE_DENSE_TOPK) || shift == 0 || ix->ntiles < 4;
    if (!p.dense_only) {
        p.stride = 1 << shift;
        p.sample_tiles = (ix->ntiles + p.stride - 1) / p.stride;
        p.cand_cap = std::max<int64_t>(4096, 8 * (int64_t)k * p.stride);
        p.cand_cap = std::min<int64_t>(p.cand_cap, ix->N_pad);
    }
    return p;
}

bool plan_wants_x(const gs_index* ix, const Plan& p, int64_t B) {
    return p.algo == GS_ALGO_TERM_PARALLEL && gs_score_term_wants_x(ix, B, p.group, p.use_head);
}

PlanStats plan_stats(const gs_index* ix, const Plan& p, int64_t B, int32_t sample_tiles) {
    PlanStats ps{};
    ps.launches = gs_tls_launches + 1;
    ps.algo = p.algo;
    ps.sample_tiles = sample_tiles;
    if (p.algo == GS_ALGO_DOC_PARALLEL) {
        ps.qtile = gs_score_doc_qtile(p.qtile);
        ps.passes = (int32_t)((B + ps.qtile - 1) / ps.qtile);
    } else {
        ps.group = gs_score_term_group(ix, B, p.group, p.use_head);
    }
    return ps;
}

struct Carve {
    StatsBlock* sb; gs_qbatch qb; uint64_t* thr; uint32_t* cand_cnt; int32_t* overflow_list; void* sel_scratch;
    void* doc_scratch; uint64_t* cand; uint32_t* dense; size_t dense_bytes; size_t fixed_bytes;
};

// Lays the workspace out; with ws == nullptr only sizes are computed (fixed_bytes = everything but the dense region).
Carve carve_ws(const gs_index* ix, const Plan& p, int64_t B, int64_t nnz, int32_t k, void* ws, size_t ws_bytes) {
    Carve c{};
    unsigned char* base = (unsigned char*)ws;
    size_t off = 0;
    auto take = [&](size_t bytes) { void* r = base ? base + off : nullptr; off += up256(bytes); return r; };
    c.sb = (StatsBlock*)take(sizeof(StatsBlock));
    c.qb.head_pair = (uint2*)take((size_t)B * GS_HEAD_MAX * 8);
    c.qb.head_cnt = (int32_t*)take((size_t)B * 4);
    c.qb.tail_desc = (uint4*)take((size_t)nnz * 16);
    c.qb.tail_cnt = (int32_t*)take((size_t)B * 4);
    c.qb.tail32 = (uint4*)take((size_t)B * GS_TAIL32 * 16);
    c.qb.xpair = (uint2*)take((size_t)B * GS_XSTRIP_MAX * 8);
    c.qb.xcnt = (int32_t*)take((size_t)B * 4);
    c.thr = (uint64_t*)take((size_t)B * 8);
    c.cand_cnt = (uint32_t*)take((size_t)B * 4 * GS_CNT_STRIDE);
    c.overflow_list = (int32_t*)take((size_t)B * 4);
    c.sel_scratch = take(gs_select_scratch_bytes(B, k));
    c.doc_scratch = p.algo == GS_ALGO_DOC_PARALLEL ? take(gs_score_doc_scratch_bytes_ex(ix, p.qtile, B, nnz)) : nullptr;
    c.cand = p.dense_only ? nullptr : (uint64_t*)take((size_t)B * (size_t)p.cand_cap * 8);
    c.fixed_bytes = off;
    c.dense = (uint32_t*)(base ? base + off : nullptr);
    c.dense_bytes = ws_bytes > off ? ws_bytes - off : 0;
    if (base) c.qb.status = &c.sb->status;
    return c;
}

gs_status_t run_score(const gs_index* ix, const Plan& p, const gs_csr_t* q, const gs_qbatch& qb, int64_t q0, int64_t nq,
                      const gs_tileset& ts, const gs_sink& sink, void* doc_scratch, cudaStream_t s) {
    if (p.algo == GS_ALGO_DOC_PARALLEL) return gs_launch_score_doc(ix, q, qb, q0, nq, p.qtile, ts, sink, doc_scratch, s);
    return gs_launch_score_term(ix, qb, q0, nq, p.group, p.use_head, (p.flags & GS_FLAG_TENSOR_CORE_HEAD) != 0, ts, sink, s);
}

// dense path for queries [q0, q0+nq): score every tile into the dense region, select, write results
gs_status_t dense_topk(const gs_index* ix, const Plan& p, const gs_csr_t* q, const Carve& c, int64_t q0, int64_t nq,
                       int32_t k, int32_t* out_ids, uint32_t* out_scores, cudaStream_t s) {
    const int64_t ld = ix->N_pad;
    const int64_t per = (int64_t)(c.dense_bytes / ((size_t)ld * 4));
    if (per < 1) return GS_ERR_OOM;
    gs_tileset all{0, 1, ix->ntiles};
    for (int64_t a = q0; a < q0 + nq; a += per) {
        const int64_t n = std::min<int64_t>(per, q0 + nq - a);
        gs_sink sink{};
        sink.dense = c.dense;
        sink.ld = ld;
        GS_TRY(run_score(ix, p, q, c.qb, a, n, all, sink, c.doc_scratch, s));
        gs_sel_src src{};
        src.dense = c.dense; src.ld = ld; src.n_cols = ld; src.n_docs = ix->N; src.ts = all; src.Ts = 0;
        src.wtype = ix->wtype;
        GS_TRY(gs_launch_select(src, n, k, out_ids + a * k, out_scores + a * k, nullptr, nullptr, nullptr, 0,
                                c.sel_scratch, s));
    }
    return GS_OK;
}

gs_status_t search_impl(const gs_index* ix, const gs_csr_t* q, int32_t k, const gs_search_opts_t* opts, int32_t* out_ids,
                        void* out_scores_v, void* ws, size_t ws_bytes, cudaStream_t s) {
    uint32_t* out_scores = (uint32_t*)out_scores_v;
    const int64_t B = q->rows;
    gs_tls_launches = 0;
    Plan p = make_plan(ix, B, q->nnz, k, opts);
    Carve c = carve_ws(ix, p, B, q->nnz, k, ws, ws_bytes);
    if (ws_bytes < c.fixed_bytes + (size_t)ix->N_pad * 4) return GS_ERR_OOM;
    c.qb.B = B; c.qb.nnz = q->nnz; c.qb.indptr = q->indptr;
    GS_CUDA(cudaMemsetAsync(c.sb, 0, sizeof(StatsBlock), s));
    if (B == 0) return GS_OK;
    const bool validate = p.flags & GS_FLAG_VALIDATE_QUERIES;
    GS_TRY(gs_launch_ingest(ix, q, validate, p.use_head, plan_wants_x(ix, p, B), &c.qb, s));
    if (validate) {
        int32_t st = 0;
        GS_CUDA(cudaMemcpyAsync(&st, &c.sb->status, sizeof(int32_t), cudaMemcpyDeviceToHost, s));
        GS_CUDA(cudaStreamSynchronize(s));
        if (st) return (gs_status_t)st;
    }
    if (ix->N == 0) {
        // no documents: every slot is padding
        gs_sel_src src{};
        src.dense = c.dense; src.ld = 0; src.n_cols = 0; src.n_docs = 0; src.Ts = 0; src.wtype = ix->wtype;
        return gs_launch_select(src, B, k, out_ids, out_scores, nullptr, nullptr, nullptr, 0, c.sel_scratch, s);
    }

    if (p.dense_only) {
        GS_TRY(dense_topk(ix, p, q, c, 0, B, k, out_ids, out_scores, s));
        {
            GsProfScope ps(GS_K_MISC, s);
            k_finalize_stats<<<1, 256, 0, s>>>(c.sb, nullptr, B, 0, c.overflow_list, plan_stats(ix, p, B, ix->ntiles));
        }
        ++gs_tls_launches;
        GS_CUDA(cudaGetLastError());
        return GS_OK;
    }

    // ---- 1. sample: every stride-th tile, dense, for as many queries at a time as the dense region holds
    gs_tileset sample{0, p.stride, p.sample_tiles};
    const int64_t sld = (int64_t)p.sample_tiles * ix->Ts;
    const int64_t per = (int64_t)(c.dense_bytes / ((size_t)sld * 4));
    if (per < 1) return GS_ERR_OOM;
    for (int64_t a = 0; a < B; a += per) {
        const int64_t n = std::min<int64_t>(per, B - a);
        gs_sink sink{};
        sink.dense = c.dense;
        sink.ld = sld;
        GS_TRY(run_score(ix, p, q, c.qb, a, n, sample, sink, c.doc_scratch, s));
        gs_sel_src src{};
        src.dense = c.dense; src.ld = sld; src.n_cols = sld; src.n_docs = ix->N; src.ts = sample; src.Ts = ix->Ts;
        src.wtype = ix->wtype;
        GS_TRY(gs_launch_select(src, n, k, nullptr, nullptr, c.thr + a, nullptr, nullptr, 0, c.sel_scratch, s));
    }
    // ---- 2. filter: all tiles, emit key >= bound
    {
        GsProfScope ps(GS_K_MISC, s);
        k_zero_u32<<<(unsigned)((B * GS_CNT_STRIDE + 255) / 256), 256, 0, s>>>(c.cand_cnt, B * GS_CNT_STRIDE);
    }
    ++gs_tls_launches;
    {
        gs_tileset all{0, 1, ix->ntiles};
        gs_sink sink{};
        sink.thr = c.thr; sink.cand = c.cand; sink.cand_cnt = c.cand_cnt; sink.cand_cap = p.cand_cap;
        GS_TRY(run_score(ix, p, q, c.qb, 0, B, all, sink, c.doc_scratch, s));
    }
    // ---- 3. final select over the candidate lists
    {
        gs_sel_src src{};
        src.keys = c.cand; src.cap = p.cand_cap; src.counts = c.cand_cnt; src.cnt_stride = GS_CNT_STRIDE; src.wtype = ix->wtype;
        GS_TRY(gs_launch_select(src, B, k, out_ids, out_scores, nullptr, nullptr, nullptr, 0, c.sel_scratch, s));
    }
    {
        GsProfScope ps(GS_K_MISC, s);
        k_finalize_stats<<<1, 256, 0, s>>>(c.sb, c.cand_cnt, B, p.cand_cap, c.overflow_list,
                                           plan_stats(ix, p, B, p.sample_tiles));
    }
    ++gs_tls_launches;
    GS_CUDA(cudaGetLastError());
    // ---- 4. a query whose candidate list overflowed has an inexact row: it is flagged in the stats block (n_overflow, list
    // of the queries) and re-run through the dense path by gs_search_finish — the only part that needs the host
    return GS_OK;
}

// dense fallback for the overflowed queries of the last gs_search on this workspace (n_ov of them, host list `ov`):
// consecutive query numbers are re-run together, as many at a time as the dense region holds
gs_status_t resolve_overflow(const gs_index* ix, const gs_csr_t* q, int32_t k, const gs_search_opts_t* opts, int32_t* out_ids,
                             void* out_scores, void* ws, size_t ws_bytes, std::vector<int32_t>& ov, cudaStream_t s) {
    Plan p = make_plan(ix, q->rows, q->nnz, k, opts);
    Carve c = carve_ws(ix, p, q->rows, q->nnz, k, ws, ws_bytes);
    c.qb.B = q->rows; c.qb.nnz = q->nnz; c.qb.indptr = q->indptr;
    // the ingest result of the search is still in the workspace (second-tier strip lists included)
    c.qb.x_on = plan_wants_x(ix, p, q->rows) && ix->HX > 0;
    std::sort(ov.begin(), ov.end());
    for (size_t i = 0; i < ov.size();) {
        size_t j = i + 1;
        while (j < ov.size() && ov[j] == ov[j - 1] + 1) ++j;
        GS_TRY(dense_topk(ix, p, q, c, ov[i], (int64_t)(j - i), k, out_ids, (uint32_t*)out_scores, s));
        i = j;
    }
    return GS_OK;
}

const gs_search_opts_t* norm_opts(const gs_search_opts_t* o, gs_search_opts_t* tmp) {
    if (!o) { std::memset(tmp, 0, sizeof(*tmp)); return tmp; }
    return o;
}

}  // namespace

extern "C" {

int32_t gs_dispatch_model(int64_t num_docs, int32_t tile_docs, int64_t stream_bytes_, int64_t B, int64_t nnz, double* out_term_ms,
                          double* out_doc_ms) {
    const double N = (double)std::max<int64_t>(num_docs, 0), Bq = (double)std::max<int64_t>(B, 1), terms = (double)std::max<int64_t>(nnz, 0);
    const double tiles = std::ceil(N / (double)std::max(tile_docs, 1));
    // term-parallel: cell rows = B * tiles over 148 SMs x 64 warp slots; a row costs ~0.6 us per query term (one
    // segment-table probe per (query, term, doc tile) plus the postings it finds), up to 2.8x that on long lists
    const double waves = std::max(1.0, Bq * tiles / 9472.0);
    const double t_term = 0.10 + waves * (terms / Bq) * 0.6e-3 * (1.0 + 1.8 * std::min(1.0, N / 1e6));
    // document-parallel: one pass over the forward index per tile of QT queries at ~4.7 TB/s, plus the hit walk
    // (constants re-fitted to the sweep of the reworked kernels, profiles/r02_dispatch_sweep.csv)
    const double qt = B <= 8 ? 8.0 : 16.0;
    const double passes = std::ceil(Bq / qt);
    const double t_doc = 0.13 + passes * ((double)std::max<int64_t>(stream_bytes_, 0) / 4.7e9) + terms * 0.1e-3 * (1.0 + 2.7 * N / 1e6);
    if (out_term_ms) *out_term_ms = t_term;
    if (out_doc_ms) *out_doc_ms = t_doc;
    return t_doc < t_term ? GS_ALGO_DOC_PARALLEL : GS_ALGO_TERM_PARALLEL;
}

gs_status_t gs_index_build(const gs_csr_t* docs, int32_t vocab_size, const gs_build_opts_t* opts, const gs_alloc_t* alloc,
                           gs_stream_t stream, gs_index_t** out) {
    if (out) *out = nullptr;
    if (!out || vocab_size <= 0) return GS_ERR_INVALID_ARG;
    if (vocab_size >= (1 << GS_FWD_DOC_SHIFT)) return GS_ERR_OUT_OF_RANGE;
    GS_TRY(check_device());
    GS_TRY(check_csr_host(docs, true));
    if (docs->rows >= 0x7FFFFFFFLL) return GS_ERR_OUT_OF_RANGE;
    if (alloc && (!alloc->alloc || !alloc->free)) return GS_ERR_INVALID_ARG;
    cudaStream_t s = (cudaStream_t)stream;
    int64_t ends[2] = {0, 0};
    GS_CUDA(cudaMemcpyAsync(&ends[0], docs->indptr, sizeof(int64_t), cudaMemcpyDeviceToHost, s));
    GS_CUDA(cudaMemcpyAsync(&ends[1], docs->indptr + docs->rows, sizeof(int64_t), cudaMemcpyDeviceToHost, s));
    GS_CUDA(cudaStreamSynchronize(s));
    if (ends[0] != 0 || ends[1] != docs->nnz) return GS_ERR_INVALID_ARG;
    gs_build_opts_t o{};
    if (opts) o = *opts;
    if (!opts) o.validate = 1;
    if (o.tile_docs == 0) o.tile_docs = 512;
    if (o.tile_docs < 32 || o.tile_docs % 32 != 0 || o.tile_docs > 8192) return GS_ERR_INVALID_ARG;
    gs_index* ix = new (std::nothrow) gs_index();
    if (!ix) return GS_ERR_OOM;
    ix->N = docs->rows; ix->V = vocab_size; ix->wtype = docs->wtype; ix->P = docs->nnz;
    ix->Ts = o.tile_docs;
    ix->ntiles = (int32_t)((ix->N + ix->Ts - 1) / ix->Ts);
    ix->N_pad = (int64_t)ix->ntiles * ix->Ts;
    if (alloc) { ix->alloc = *alloc; ix->has_alloc = true; }
    gs_status_t st = gs_build_index_impl(ix, docs, o, s);
    if (st != GS_OK) { gs_index_free(ix); return st; }
    *out = ix;
    return GS_OK;
}

void gs_index_free(gs_index_t* ix) {
    if (!ix) return;
    cudaDeviceSynchronize();
    void* ptrs[] = {ix->fwd_blk, ix->fwd_terms, ix->fwd_w, ix->inv_off, ix->inv_len, ix->inv_doc, ix->inv_w, ix->inv_pk, ix->mma_strips,
                    ix->term_meta, ix->seg_tab, ix->seg_l1, ix->seg_l2, ix->head_slot, ix->head_strip, ix->xslot, ix->xstrip, ix->host_ws, ix->host_stage};
    for (void* p : ptrs) gs_dev_free(ix, p, 0);
    delete ix;
}

gs_status_t gs_index_info(const gs_index_t* ix, gs_info_t* out) {
    if (!ix || !out) return GS_ERR_INVALID_ARG;
    out->num_docs = ix->N; out->vocab_size = ix->V; out->wtype = ix->wtype; out->nnz = ix->P;
    out->padded_nnz = ix->P_pad; out->nonempty_terms = ix->nonempty; out->tile_docs = ix->Ts;
    out->num_tiles = ix->ntiles; out->head_terms = ix->H;
    out->bytes_inverted = ix->bytes_inverted; out->bytes_inverted_meta = ix->bytes_meta;
    out->bytes_forward = ix->bytes_forward; out->bytes_head = ix->bytes_head;
    out->head_terms_term_parallel = ix->H + ix->HX; out->forward_tail_nnz = ix->P_tail;
    out->forward_padded_nnz = ix->P_fwd; out->packed_layout = (ix->inv_packed ? 1 : 0) | (ix->fwd_packed ? 2 : 0);
    out->bytes_total = ix->bytes_inverted + ix->bytes_meta + ix->bytes_forward + ix->bytes_head;
    return GS_OK;
}

gs_status_t gs_index_copy_meta(const gs_index_t* ix, int64_t* host_offsets, int32_t* host_lengths) {
    if (!ix || !host_offsets || !host_lengths) return GS_ERR_INVALID_ARG;
    GS_CUDA(cudaMemcpy(host_offsets, ix->inv_off, sizeof(int64_t) * (size_t)(ix->V + 1), cudaMemcpyDeviceToHost));
    GS_CUDA(cudaMemcpy(host_lengths, ix->inv_len, sizeof(int32_t) * (size_t)ix->V, cudaMemcpyDeviceToHost));
    return GS_OK;
}

gs_status_t gs_index_copy_list(const gs_index_t* ix, int32_t term, int64_t capacity, int32_t* host_doc_ids,
                               void* host_weights, int64_t* out_padded_length) {
    if (!ix || term < 0 || term >= ix->V || capacity < 0 || !out_padded_length) return GS_ERR_INVALID_ARG;
    int64_t off[2];
    GS_CUDA(cudaMemcpy(off, ix->inv_off + term, sizeof(int64_t) * 2, cudaMemcpyDeviceToHost));
    const int64_t plen = off[1] - off[0];
    *out_padded_length = plen;
    const int64_t n = std::min(capacity, plen);
    if (n > 0) {
        if (!host_doc_ids || !host_weights) return GS_ERR_INVALID_ARG;
        const size_t wb = ix->wtype == GS_W_F32 ? 4 : 1;
        if (ix->inv_packed) {                              // compressed postings: unpack (doc | impact << 24) on the host
            GS_CUDA(cudaMemcpy(host_doc_ids, ix->inv_pk + off[0], sizeof(uint32_t) * (size_t)n, cudaMemcpyDeviceToHost));
            for (int64_t i = 0; i < n; ++i) {
                const uint32_t pk = (uint32_t)host_doc_ids[i];
                host_doc_ids[i] = pk == 0xFFFFFFFFu ? -1 : (int32_t)(pk & 0xFFFFFFu);
                ((uint8_t*)host_weights)[i] = pk == 0xFFFFFFFFu ? 0 : (uint8_t)(pk >> 24);
            }
            return GS_OK;
        }
        GS_CUDA(cudaMemcpy(host_doc_ids, ix->inv_doc + off[0], sizeof(int32_t) * (size_t)n, cudaMemcpyDeviceToHost));
        GS_CUDA(cudaMemcpy(host_weights, (const unsigned char*)ix->inv_w + (size_t)off[0] * wb, wb * (size_t)n,
                           cudaMemcpyDeviceToHost));
    }
    return GS_OK;
}

gs_status_t gs_index_copy_head_terms(const gs_index_t* ix, int32_t capacity, int32_t* host_terms, int32_t* out_count) {
    if (!ix || !out_count || capacity < 0 || (capacity > 0 && !host_terms)) return GS_ERR_INVALID_ARG;
    *out_count = ix->H;
    for (int32_t h = 0; h < std::min(capacity, ix->H); ++h) host_terms[h] = ix->head_terms_host[h];
    return GS_OK;
}

gs_status_t gs_search_workspace_bytes(const gs_index_t* ix, int64_t B, int64_t nnz, int32_t k, const gs_search_opts_t* opts,
                                      size_t* out_bytes) {
    if (!ix || !out_bytes || B < 0 || nnz < 0) return GS_ERR_INVALID_ARG;
    if (k < 1 || k > GS_MAX_K) return GS_ERR_OUT_OF_RANGE;
    // With GS_ALGO_AUTO the choice depends on the batch that is searched (its rows and nnz may be smaller than the ones the
    // workspace was sized for): size for whichever path needs more.
    size_t need = 0;
    gs_search_opts_t o2;
    if (opts) o2 = *opts; else std::memset(&o2, 0, sizeof(o2));
    const bool is_auto = o2.algo == GS_ALGO_AUTO;
    for (int a = GS_ALGO_TERM_PARALLEL; a <= GS_ALGO_DOC_PARALLEL; ++a) {
        if (!is_auto && a != o2.algo) continue;
        gs_search_opts_t oa = o2;
        oa.algo = a;
        Plan p = make_plan(ix, B, nnz, k, &oa);
        Carve c = carve_ws(ix, p, B, nnz, k, nullptr, 0);
        const size_t row = (size_t)ix->N_pad * 4;
        size_t dense = row;                                                    // minimum: one dense row (fallback)
        if (p.dense_only) dense = std::max(dense, std::min<size_t>((size_t)B * row, (size_t)4 << 30) / row * row);
        else dense = std::max(dense, (size_t)B * (size_t)p.sample_tiles * ix->Ts * 4);
        need = std::max(need, c.fixed_bytes + up256(std::max(dense, row)));
    }
    *out_bytes = need;
    return GS_OK;
}

gs_status_t gs_search(const gs_index_t* ix, const gs_csr_t* q, int32_t k, const gs_search_opts_t* opts, int32_t* out_ids,
                      void* out_scores, void* ws, size_t ws_bytes, gs_stream_t stream) {
    if (!ix || !ws) return GS_ERR_INVALID_ARG;
    GS_TRY(check_csr_host(q, true));
    if (k < 1 || k > GS_MAX_K) return GS_ERR_OUT_OF_RANGE;
    if (q->wtype != ix->wtype) return GS_ERR_TYPE_MISMATCH;
    if (q->rows > 65535) return GS_ERR_OUT_OF_RANGE;
    if (!is_device_ptr(ws)) return GS_ERR_INVALID_ARG;
    // an empty batch has empty outputs: their pointers may be null
    if (q->rows > 0 && (!is_device_ptr(out_ids) || !is_device_ptr(out_scores))) return GS_ERR_INVALID_ARG;
    if (opts && (opts->algo < GS_ALGO_AUTO || opts->algo > GS_ALGO_DOC_PARALLEL)) return GS_ERR_INVALID_ARG;
    if (((uintptr_t)ws & 255) != 0) return GS_ERR_INVALID_ARG;
    gs_search_opts_t tmp;
    return search_impl(ix, q, k, norm_opts(opts, &tmp), out_ids, out_scores, ws, ws_bytes, (cudaStream_t)stream);
}

gs_status_t gs_search_finish(const gs_index_t* ix, const gs_csr_t* q, int32_t k, const gs_search_opts_t* opts,
                             int32_t* out_ids, void* out_scores, void* ws, size_t ws_bytes, gs_stream_t stream,
                             int32_t* out_resolved) {
    if (out_resolved) *out_resolved = 0;
    if (!ix || !ws || !q) return GS_ERR_INVALID_ARG;
    if (k < 1 || k > GS_MAX_K) return GS_ERR_OUT_OF_RANGE;
    cudaStream_t s = (cudaStream_t)stream;
    if (q->rows == 0) return GS_OK;
    StatsBlock sb;
    GS_CUDA(cudaMemcpyAsync(&sb, ws, sizeof(StatsBlock), cudaMemcpyDeviceToHost, s));
    GS_CUDA(cudaStreamSynchronize(s));
    const int32_t n_ov = sb.n_overflow;
    if (n_ov <= 0) return GS_OK;
    if (n_ov > q->rows) return GS_ERR_INVALID_ARG;             // not the workspace of a search of this batch
    gs_search_opts_t tmp;
    const gs_search_opts_t* o = norm_opts(opts, &tmp);
    Plan p = make_plan(ix, q->rows, q->nnz, k, o);
    Carve c = carve_ws(ix, p, q->rows, q->nnz, k, ws, ws_bytes);
    std::vector<int32_t> ov((size_t)n_ov);
    GS_CUDA(cudaMemcpyAsync(ov.data(), c.overflow_list, sizeof(int32_t) * (size_t)n_ov, cudaMemcpyDeviceToHost, s));
    GS_CUDA(cudaStreamSynchronize(s));
    GS_TRY(resolve_overflow(ix, q, k, o, out_ids, out_scores, ws, ws_bytes, ov, s));
    GS_CUDA(cudaStreamSynchronize(s));
    if (out_resolved) *out_resolved = n_ov;
    return GS_OK;
}

gs_status_t gs_search_host(gs_index_t* ix, const gs_csr_t* hq, int32_t k, const gs_search_opts_t* opts,
                           int32_t* host_ids, void* host_scores, gs_stream_t stream) {
    static std::mutex mu;
    if (!ix || !host_ids || !host_scores) return GS_ERR_INVALID_ARG;
    GS_TRY(check_csr_host(hq, false));
    if (k < 1 || k > GS_MAX_K) return GS_ERR_OUT_OF_RANGE;
    if (hq->wtype != ix->wtype) return GS_ERR_TYPE_MISMATCH;
    std::lock_guard<std::mutex> lock(mu);
    cudaStream_t s = (cudaStream_t)stream;
    const int64_t B = hq->rows, nnz = hq->nnz;
    const size_t wb = ix->wtype == GS_W_F32 ? 4 : 1;
    size_t ws_need = 0;
    GS_TRY(gs_search_workspace_bytes(ix, B, nnz, k, opts, &ws_need));
    if (ws_need > ix->host_ws_bytes) {
        GS_CUDA(cudaStreamSynchronize(s));
        gs_dev_free(ix, ix->host_ws, s);
        ix->host_ws = gs_dev_alloc(ix, ws_need, s);
        ix->host_ws_bytes = ix->host_ws ? ws_need : 0;
        if (!ix->host_ws) return GS_ERR_OOM;
    }
    const size_t o_indptr = 0, o_terms = up256(8 * (size_t)(B + 1)), o_w = o_terms + up256(4 * (size_t)nnz),
                 o_ids = o_w + up256(wb * (size_t)nnz), o_sc = o_ids + up256(4 * (size_t)B * k),
                 stage_need = o_sc + up256(4 * (size_t)B * k);
    if (stage_need > ix->host_stage_bytes) {
        GS_CUDA(cudaStreamSynchronize(s));
        gs_dev_free(ix, ix->host_stage, s);
        ix->host_stage = gs_dev_alloc(ix, stage_need, s);
        ix->host_stage_bytes = ix->host_stage ? stage_need : 0;
        if (!ix->host_stage) return GS_ERR_OOM;
    }
    unsigned char* st = (unsigned char*)ix->host_stage;
    GS_CUDA(cudaMemcpyAsync(st + o_indptr, hq->indptr, 8 * (size_t)(B + 1), cudaMemcpyHostToDevice, s));
    if (nnz > 0) {
        GS_CUDA(cudaMemcpyAsync(st + o_terms, hq->term_ids, 4 * (size_t)nnz, cudaMemcpyHostToDevice, s));
        GS_CUDA(cudaMemcpyAsync(st + o_w, hq->weights, wb * (size_t)nnz, cudaMemcpyHostToDevice, s));
    }
    gs_csr_t dq = *hq;
    dq.indptr = (const int64_t*)(st + o_indptr);
    dq.term_ids = (const int32_t*)(st + o_terms);
    dq.weights = st + o_w;
    gs_status_t r = gs_search(ix, &dq, k, opts, (int32_t*)(st + o_ids), st + o_sc, ix->host_ws, ix->host_ws_bytes, stream);
    if (r != GS_OK) return r;
    // results and the overflow count come back together: ONE synchronisation on the common path
    int32_t n_ov = 0;
    if (B > 0) GS_CUDA(cudaMemcpyAsync(&n_ov, &((StatsBlock*)ix->host_ws)->n_overflow, sizeof(int32_t), cudaMemcpyDeviceToHost, s));
    GS_CUDA(cudaMemcpyAsync(host_ids, st + o_ids, 4 * (size_t)B * k, cudaMemcpyDeviceToHost, s));
    GS_CUDA(cudaMemcpyAsync(host_scores, st + o_sc, 4 * (size_t)B * k, cudaMemcpyDeviceToHost, s));
    GS_CUDA(cudaStreamSynchronize(s));
    if (n_ov > 0) {                     // rare: some candidate list overflowed -> dense re-run of those queries, copy again
        int32_t resolved = 0;
        GS_TRY(gs_search_finish(ix, &dq, k, opts, (int32_t*)(st + o_ids), st + o_sc, ix->host_ws, ix->host_ws_bytes, stream, &resolved));
        GS_CUDA(cudaMemcpyAsync(host_ids, st + o_ids, 4 * (size_t)B * k, cudaMemcpyDeviceToHost, s));
        GS_CUDA(cudaMemcpyAsync(host_scores, st + o_sc, 4 * (size_t)B * k, cudaMemcpyDeviceToHost, s));
        GS_CUDA(cudaStreamSynchronize(s));
    }
    return GS_OK;
}

gs_status_t gs_search_stats(const void* ws, gs_stream_t stream, gs_stats_t* out) {
    if (!ws || !out) return GS_ERR_INVALID_ARG;
    GS_CUDA(cudaStreamSynchronize((cudaStream_t)stream));
    StatsBlock sb;
    GS_CUDA(cudaMemcpy(&sb, ws, sizeof(StatsBlock), cudaMemcpyDeviceToHost));
    *out = sb.stats;
    return GS_OK;
}

gs_status_t gs_score_dense(const gs_index_t* ix, const gs_csr_t* q, const gs_search_opts_t* opts, void* out_scores,
                           int64_t ld, void* ws, size_t ws_bytes, gs_stream_t stream) {
    if (!ix || !out_scores || !ws || !opts) return GS_ERR_INVALID_ARG;
    GS_TRY(check_csr_host(q, true));
    if (q->wtype != ix->wtype) return GS_ERR_TYPE_MISMATCH;
    if (opts->algo != GS_ALGO_TERM_PARALLEL && opts->algo != GS_ALGO_DOC_PARALLEL) return GS_ERR_INVALID_ARG;
    if (ld < ix->N_pad || !is_device_ptr(out_scores) || !is_device_ptr(ws)) return GS_ERR_INVALID_ARG;
    cudaStream_t s = (cudaStream_t)stream;
    gs_tls_launches = 0;
    Plan p = make_plan(ix, q->rows, q->nnz, 1, opts);
    p.dense_only = true;
    Carve c = carve_ws(ix, p, q->rows, q->nnz, 1, ws, ws_bytes);
    if (ws_bytes < c.fixed_bytes) return GS_ERR_OOM;
    c.qb.B = q->rows; c.qb.nnz = q->nnz; c.qb.indptr = q->indptr;
    if (q->rows == 0 || ix->N == 0) return GS_OK;
    GS_TRY(gs_launch_ingest(ix, q, false, p.use_head, plan_wants_x(ix, p, q->rows), &c.qb, s));
    gs_tileset all{0, 1, ix->ntiles};
    gs_sink sink{};
    sink.dense = (uint32_t*)out_scores;
    sink.ld = ld;
    return run_score(ix, p, q, c.qb, 0, q->rows, all, sink, c.doc_scratch, s);
}

gs_status_t gs_topk_workspace_bytes(int64_t rows, int64_t n, int32_t k, size_t* out_bytes) {
    if (!out_bytes || rows < 0 || n < 0) return GS_ERR_INVALID_ARG;
    if (k < 1 || k > GS_MAX_K) return GS_ERR_OUT_OF_RANGE;
    *out_bytes = up256(gs_select_scratch_bytes(rows, k));
    return GS_OK;
}

gs_status_t gs_topk_dense(const void* scores, int32_t wtype, int64_t rows, int64_t n, int64_t ld, int32_t k, int32_t* out_ids,
                          void* out_scores, void* ws, size_t ws_bytes, gs_stream_t stream) {
    if (!out_ids || !out_scores || !ws || rows < 0 || n < 0 || ld < n) return GS_ERR_INVALID_ARG;
    if (wtype != GS_W_F32 && wtype != GS_W_U8) return GS_ERR_INVALID_ARG;
    if (k < 1 || k > GS_MAX_K) return GS_ERR_OUT_OF_RANGE;
    if (rows > 65535 || n >= 0x7FFFFFFFLL) return GS_ERR_OUT_OF_RANGE;
    GS_TRY(check_device());
    if (n > 0 && !is_device_ptr(scores)) return GS_ERR_INVALID_ARG;
    if (!is_device_ptr(out_ids) || !is_device_ptr(out_scores) || !is_device_ptr(ws)) return GS_ERR_INVALID_ARG;
    if (ws_bytes < gs_select_scratch_bytes(rows, k)) return GS_ERR_OOM;
    gs_tls_launches = 0;
    gs_sel_src src{};
    src.dense = (const uint32_t*)scores; src.ld = ld; src.n_cols = n; src.n_docs = n; src.Ts = 0; src.wtype = wtype;
    return gs_launch_select(src, rows, k, out_ids, out_scores, nullptr, nullptr, nullptr, 0, ws, (cudaStream_t)stream);
}

gs_status_t gs_merge_topk_workspace_bytes(int32_t n_lists, int64_t B, int32_t k_in, int32_t k_out, size_t* out_bytes) {
    if (!out_bytes || n_lists < 1 || n_lists > GS_MERGE_MAX_LISTS || B < 0 || k_in < 1) return GS_ERR_INVALID_ARG;
    if (k_out < 1 || k_out > GS_MAX_K || B > 65535) return GS_ERR_OUT_OF_RANGE;
    *out_bytes = gs_merge_scratch_bytes(n_lists, B, k_in, k_out);
    return GS_OK;
}

gs_status_t gs_merge_topk(int32_t wtype, int32_t n_lists, int64_t B, int32_t k_in, int32_t k_out, const int32_t* ids,
                          const void* scores, const int64_t* list_doc_base, int32_t* out_ids, void* out_scores, void* ws,
                          size_t ws_bytes, gs_stream_t stream) {
    if (!out_ids || !out_scores || !ws || n_lists < 1 || n_lists > GS_MERGE_MAX_LISTS || B < 0 || k_in < 1)
        return GS_ERR_INVALID_ARG;
    if (wtype != GS_W_F32 && wtype != GS_W_U8) return GS_ERR_INVALID_ARG;
    if (k_out < 1 || k_out > GS_MAX_K || B > 65535) return GS_ERR_OUT_OF_RANGE;
    if ((int64_t)n_lists * k_in > (int64_t)1 << 20) return GS_ERR_OUT_OF_RANGE;       // one-launch select: rows of up to 2^20 keys
    GS_TRY(check_device());
    if (B > 0 && (!is_device_ptr(ids) || !is_device_ptr(scores))) return GS_ERR_INVALID_ARG;
    if (!is_device_ptr(out_ids) || !is_device_ptr(out_scores) || !is_device_ptr(ws)) return GS_ERR_INVALID_ARG;
    if (ws_bytes < gs_merge_scratch_bytes(n_lists, B, k_in, k_out)) return GS_ERR_OOM;
    if (list_doc_base)
        for (int l = 0; l < n_lists; ++l)
            if (list_doc_base[l] < 0 || list_doc_base[l] >= 0xFFFFFFFFLL) return GS_ERR_OUT_OF_RANGE;
    gs_tls_launches = 0;
    if (B == 0) return GS_OK;
    return gs_launch_merge(wtype, n_lists, B, k_in, k_out, ids, scores, list_doc_base, out_ids, out_scores, ws,
                           (cudaStream_t)stream);
}

void gs_profile_enable(int32_t on) {
    tls_prof_on = on != 0;
    for (ProfRec& r : tls_prof) { tls_event_pool.push_back(r.a); tls_event_pool.push_back(r.b); }
    tls_prof.clear();
}

gs_status_t gs_profile_read(gs_profile_t* out) {
    if (!out) return GS_ERR_INVALID_ARG;
    std::memset(out, 0, sizeof(*out));
    gs_status_t st = GS_OK;
    for (ProfRec& r : tls_prof) {
        float ms = 0.f;
        if (cudaEventSynchronize(r.b) != cudaSuccess || cudaEventElapsedTime(&ms, r.a, r.b) != cudaSuccess) {
            gs_set_cuda_error(cudaGetLastError());
            st = GS_ERR_CUDA;
        } else if (r.kclass >= 0 && r.kclass < GS_PROF_CLASSES) {
            out->launches[r.kclass] += r.n;
            out->ms[r.kclass] += ms;
        }
        tls_event_pool.push_back(r.a);
        tls_event_pool.push_back(r.b);
    }
    tls_prof.clear();
    return st;
}

const char* gs_kclass_name(int32_t k) {
    switch (k) {
        case GS_K_INGEST: return "ingest";
        case GS_K_SCORE_TERM: return "score_term";
        case GS_K_SCORE_DOC: return "score_doc";
        case GS_K_QTILE: return "build_qtile";
        case GS_K_SELECT: return "radix_select";
        case GS_K_SORT: return "bitonic_sort";
        case GS_K_MISC: return "misc";
    }
    return "";
}

const char* gs_strerror(gs_status_t st) {
    switch (st) {
        case GS_OK: return "ok";
        case GS_ERR_INVALID_ARG: return "invalid argument";
        case GS_ERR_OUT_OF_RANGE: return "value out of range";
        case GS_ERR_DUPLICATE_TERM: return "duplicate term id in a row";
        case GS_ERR_NONFINITE: return "non-finite weight";
        case GS_ERR_OOM: return "out of memory / workspace too small";
        case GS_ERR_CUDA: return "CUDA runtime error";
        case GS_ERR_UNSUPPORTED_DEVICE: return "unsupported device (sm_100 required; there is no fallback)";
        case GS_ERR_TYPE_MISMATCH: return "query weight type differs from the index weight type";
    }
    return "unknown status";
}
const char* gs_version(void) { return "gpusparse-b200 0.1.0 (sm_100a)"; }
int32_t gs_abi_version(void) { return GS_ABI_VERSION; }
int32_t gs_last_cuda_error(void) { return tls_cuda_error; }
int32_t gs_last_launch_count(void) { return gs_tls_launches; }

}  // extern "C"
