"""Parity of the CUDA path (through the C ABI) against the CPU oracle — `-m gpu`, run on the B200 box.

Integer-impact mode must be bit-exact; fp32 mode within tol(x) = max(1e-5*|x|, 1e-6) with the set/order
rules of tests/parity.py (BASELINE.json north_star).  Inputs come from the seeded generator
(paper_2606_26441_b200.workload) or are built by hand here; expected values come from `oracle/` only.
"""
import json
import os

import numpy as np
import pytest

import oracle
from paper_2606_26441_b200 import workload as wl
import parity  # tests/parity.py (pytest puts tests/ on sys.path)

pytestmark = pytest.mark.gpu
GOLD = os.path.join(os.path.dirname(__file__), "golden")
ALGOS = ["term", "term_w2", "doc"]


def aopt(algo):
    """Search options of a parametrised kernel: "term" = term-parallel (default: 2 cell rows per CTA), "term_w2" = the same
    kernel with 5 cell rows per CTA (other tile/query interleaving), "doc" = document-parallel."""
    return {"term": dict(algo="term"), "term_w2": dict(algo="term", query_group=5), "doc": dict(algo="doc")}[algo]


@pytest.fixture(scope="module")
def gs():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("gpu tests need a CUDA device (run through gpurun)")
    from paper_2606_26441_b200 import binding
    binding.lib()
    return binding


def dev(csr):
    import torch
    d = torch.device("cuda:0")
    return (torch.from_numpy(np.ascontiguousarray(csr.indptr)).to(d), torch.from_numpy(np.ascontiguousarray(csr.terms)).to(d),
            torch.from_numpy(np.ascontiguousarray(csr.weights)).to(d))


def csr_from_dicts(rows, dtype):
    indptr, terms, weights = [0], [], []
    for r in rows:
        for t, w in r.items():
            terms.append(int(t))
            weights.append(w)
        indptr.append(len(terms))
    return wl.Csr(np.array(indptr, np.int64), np.array(terms, np.int32), np.array(weights, dtype))


def gpu_search(gs, ix, queries, k, **opt):
    ids, sc = ix.search(*dev(queries), k, **opt)
    return ids.cpu().numpy(), sc.cpu().numpy()


def compare(gs, docs, queries, vocab, k, g_ids, g_sc):
    """Full comparison of a GPU result against the oracle's exhaustive search."""
    R_d, R_q = oracle.as_rows(docs, vocab), oracle.as_rows(queries, vocab)
    o_ids, o_sc = oracle.search(R_q, R_d, k)
    if docs.weights.dtype == np.uint8:
        parity.check_int_exact(g_ids, g_sc, o_ids, o_sc)
        return 0.0, 0
    def true_scores(b, ids):
        return oracle.score_pairs(R_q, R_d, np.full(len(ids), b, np.int64), ids.astype(np.int64))
    return parity.check_f32(g_ids, g_sc, o_ids, o_sc, true_scores, docs.rows)


# ----------------------------------------------------------------------------------------------------
# hand-worked example (tests/golden/handworked_3doc.json) and the index layout of Eq. 2
# ----------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("algo", ALGOS)
@pytest.mark.parametrize("mode", ["f32", "u8"])
def test_handworked_three_docs(gs, mode, algo):
    g = json.load(open(os.path.join(GOLD, "handworked_3doc.json")))
    c = g[mode]
    dt = np.float32 if mode == "f32" else np.uint8
    docs, queries = csr_from_dicts(c["docs"], dt), csr_from_dicts(c["queries"], dt)
    ix = gs.Index.from_numpy(docs, g["vocab"])
    ids, sc = gpu_search(gs, ix, queries, c["k"], **aopt(algo))
    assert ids.tolist() == c["expect_ids"]
    assert sc.tolist() == c["expect_scores"]
    ix.close()


def test_index_layout_eq2(gs):
    g = json.load(open(os.path.join(GOLD, "handworked_3doc.json")))
    docs = csr_from_dicts(g["f32"]["docs"], np.float32)
    ix = gs.Index.from_numpy(docs, g["vocab"])
    inf, lay = ix.info(), g["index_layout"]
    assert inf["nnz"] == lay["postings"] and inf["nonempty_terms"] == lay["nonempty_terms"]
    assert inf["padded_nnz"] == lay["padded_slots"]
    ids, w = ix.posting_list(3)
    assert len(ids) == 32
    assert [[int(i), float(x)] for i, x in zip(ids[:2], w[:2])] == lay["term3_list"]
    assert np.all(ids[2:] == -1) and np.all(w[2:] == 0)          # sentinel (doc_id=-1, score=0), L90
    off, ln = ix.meta()
    assert np.all(off % 32 == 0) and off[-1] == lay["padded_slots"]
    assert np.array_equal(np.diff(off), (ln.astype(np.int64) + 31) // 32 * 32)
    ix.close()


# ----------------------------------------------------------------------------------------------------
# BASELINE.json configs[0] (tiny): element-by-element score parity + top-k parity, both kernels
# ----------------------------------------------------------------------------------------------------
@pytest.fixture(scope="module")
def tiny():
    w = wl.make_workload("tiny")
    return w


def _dense_parity(gs, docs, queries, vocab, algo, **build_kw):
    ix = gs.Index.from_numpy(docs, vocab, **build_kw)
    S = ix.score_dense(*dev(queries), **aopt(algo)).cpu().numpy()[:, :docs.rows]
    R_d, R_q = oracle.as_rows(docs, vocab), oracle.as_rows(queries, vocab)
    _, _, A = oracle.search(R_q, R_d, 1, all_scores=True)
    if docs.weights.dtype == np.uint8:
        assert np.array_equal(S.astype(np.int64), A.astype(np.int64))
    else:
        err = np.abs(S.astype(np.float64) - A)
        assert np.all(err <= parity.tol(A)), f"max err {err.max()}"
        assert np.all(S[A == 0.0] == 0.0)             # a doc with no shared term scores exactly 0
    ix.close()


@pytest.mark.parametrize("algo", ALGOS)
@pytest.mark.parametrize("mode", ["f32", "u8"])
@pytest.mark.parametrize("build_kw", [dict(), dict(tile_docs=96, head_max=-1), dict(tile_docs=2048, head_max=5)])
def test_tiny_all_scores(gs, tiny, mode, algo, build_kw):
    docs = tiny.docs if mode == "f32" else tiny.docs.to_u8()
    queries = tiny.queries if mode == "f32" else tiny.queries.to_u8()
    _dense_parity(gs, docs, queries, tiny.vocab, algo, **build_kw)


@pytest.mark.parametrize("mode", ["f32", "u8"])
@pytest.mark.parametrize("qtile", [8, 16, 32, 64])
@pytest.mark.parametrize("build_kw", [dict(), dict(head_max=-1), dict(head_max=64, head_density=0.02)])
def test_doc_parallel_query_tiles(gs, mode, qtile, build_kw):
    """Every query-tile width of the doc-parallel kernel: several passes with a ragged last one (B = 75),
    with all / none / 64 of the lists as dense strips; scores element by element, then top-k."""
    w = wl.make_workload("tiny", n_docs=3000, n_queries=75)
    docs = w.docs if mode == "f32" else w.docs.to_u8()
    queries = w.queries if mode == "f32" else w.queries.to_u8()
    ix = gs.Index.from_numpy(docs, w.vocab, **build_kw)
    S = ix.score_dense(*dev(queries), algo="doc", doc_query_tile=qtile).cpu().numpy()[:, :docs.rows]
    R_d, R_q = oracle.as_rows(docs, w.vocab), oracle.as_rows(queries, w.vocab)
    _, _, A = oracle.search(R_q, R_d, 1, all_scores=True)
    if mode == "u8":
        assert np.array_equal(S.astype(np.int64), A.astype(np.int64))
    else:
        assert np.all(np.abs(S.astype(np.float64) - A) <= parity.tol(A))
    ids, sc = gpu_search(gs, ix, queries, 100, algo="doc", doc_query_tile=qtile)
    compare(gs, docs, queries, w.vocab, 100, ids, sc)
    ix.close()


@pytest.mark.parametrize("qtile", [8, 32, 64])
def test_doc_parallel_long_rows(gs, qtile):
    """Documents far longer than the hit queue (128 entries) whose postings nearly all hit the query tile, and
    queries with thousands of terms (query tile rows spill from shared memory to global memory)."""
    rng = np.random.default_rng(7)
    V, N, B = 30522, 257, 40
    docs = csr_from_dicts([{int(t): float(np.float32(rng.uniform(0.1, 2.0))) for t in rng.choice(V, size=int(n), replace=False)}
                           for n in rng.integers(1, 3000, size=N)], np.float32)
    queries = csr_from_dicts([{int(t): float(np.float32(rng.uniform(0.1, 2.0))) for t in rng.choice(V, size=int(n), replace=False)}
                              for n in rng.integers(1, 6000, size=B)], np.float32)
    ix = gs.Index.from_numpy(docs, V)
    S = ix.score_dense(*dev(queries), algo="doc", doc_query_tile=qtile).cpu().numpy()[:, :N]
    R_d, R_q = oracle.as_rows(docs, V), oracle.as_rows(queries, V)
    _, _, A = oracle.search(R_q, R_d, 1, all_scores=True)
    # up to ~600 shared terms per pair: the fp32 bound is n * 2^-24 relative, beyond BASELINE's 1e-5
    assert np.all(np.abs(S.astype(np.float64) - A) <= np.maximum(4e-5 * np.abs(A), 1e-6))
    ids, sc = gpu_search(gs, ix, queries, 10, algo="doc", doc_query_tile=qtile)
    assert ids.shape == (B, 10) and np.all(ids >= 0)
    # the top-10 against the oracle's, with the same widened relative bound: structure, values, set, order
    o_ids, o_sc = oracle.search(R_q, R_d, 10)
    for b in range(B):
        t = A[b, ids[b]]
        bound = lambda x: np.maximum(4e-5 * np.abs(x), 1e-6)
        assert len(set(ids[b].tolist())) == 10 and np.all(np.diff(sc[b]) <= 0)
        eq = np.nonzero(np.diff(sc[b]) == 0)[0]
        assert np.all(ids[b][eq] < ids[b][eq + 1])
        assert np.all(np.abs(sc[b].astype(np.float64) - t) <= bound(t))
        tau = o_sc[b][9]
        assert np.all(np.isin(o_ids[b][o_sc[b] > tau + 2 * bound(tau)], ids[b])), "a clearly-top-k document is missing"
        assert np.all(t >= tau - 2 * bound(tau)), "a returned document is clearly below the k-th score"
        assert np.all(t[:-1] >= t[1:] - 2 * bound(t[1:])), "returned order contradicts true scores"
    ix.close()


@pytest.mark.parametrize("algo", ALGOS)
@pytest.mark.parametrize("mode", ["f32", "u8"])
@pytest.mark.parametrize("k", [1, 10, 33, 1000])
def test_tiny_topk(gs, tiny, mode, algo, k):
    docs = tiny.docs if mode == "f32" else tiny.docs.to_u8()
    queries = tiny.queries if mode == "f32" else tiny.queries.to_u8()
    ix = gs.Index.from_numpy(docs, tiny.vocab)
    for flags in (0, gs.GS_FLAG_FORCE_DENSE_TOPK, gs.GS_FLAG_NO_HEAD_STRIPS | gs.GS_FLAG_VALIDATE_QUERIES):
        ids, sc = gpu_search(gs, ix, queries, k, **aopt(algo), flags=flags)
        compare(gs, docs, queries, tiny.vocab, k, ids, sc)
    ix.close()


@pytest.mark.parametrize("algo", ALGOS)
@pytest.mark.parametrize("n_docs", [1, 31, 33, 1000, 4097, 10_007])
def test_ragged_collection_sizes(gs, algo, n_docs):
    """N not a multiple of the warp block / tile; includes collections smaller than one tile."""
    docs = wl.make_docs("tiny", n_docs=n_docs, seed=3)
    queries = wl.make_queries("tiny", n_queries=7, seed=3)
    for d, q in ((docs, queries), (docs.to_u8(), queries.to_u8())):
        ix = gs.Index.from_numpy(d, wl.VOCAB, tile_docs=256)
        for k in (1, 10, 50):
            ids, sc = gpu_search(gs, ix, q, k, **aopt(algo))
            compare(gs, d, q, wl.VOCAB, k, ids, sc)
        ix.close()


# ----------------------------------------------------------------------------------------------------
# degenerate cases and closed forms (SURVEY §8c pins, here applied to the CUDA path)
# ----------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("algo", ALGOS)
def test_empty_query_empty_batch_and_k_gt_n(gs, algo):
    import torch
    docs = wl.make_docs("tiny", n_docs=40, seed=5)
    ix = gs.Index.from_numpy(docs, wl.VOCAB)
    # query 1 is empty: all scores 0 -> ids ascending; k > N -> (-1, -inf) padding
    q = wl.make_queries("tiny", n_queries=3, seed=5)
    a, b = int(q.indptr[1]), int(q.indptr[2])
    q = wl.Csr(np.array([0, a, a, a + int(q.indptr[3]) - b], np.int64), np.delete(q.terms, slice(a, b)),
               np.delete(q.weights, slice(a, b)))
    ids, sc = gpu_search(gs, ix, q, 64, **aopt(algo))
    compare(gs, docs, q, wl.VOCAB, 64, ids, sc)
    assert ids[1, :40].tolist() == list(range(40)) and np.all(sc[1, :40] == 0)
    assert np.all(ids[:, 40:] == -1) and np.all(np.isneginf(sc[:, 40:]))
    # B = 0
    e = wl.Csr(np.zeros(1, np.int64), np.zeros(0, np.int32), np.zeros(0, np.float32))
    d = torch.device("cuda:0")
    ids0, sc0 = ix.search(torch.zeros(1, dtype=torch.int64, device=d), torch.zeros(0, dtype=torch.int32, device=d),
                          torch.zeros(0, dtype=torch.float32, device=d), 5, **aopt(algo))
    assert tuple(ids0.shape) == (0, 5) and tuple(sc0.shape) == (0, 5)
    ix.close()
    # integer twin of the padding rule
    du, qu = docs.to_u8(), q.to_u8()
    ixu = gs.Index.from_numpy(du, wl.VOCAB)
    ids, sc = gpu_search(gs, ixu, qu, 64, **aopt(algo))
    compare(gs, du, qu, wl.VOCAB, 64, ids, sc)
    assert np.all(sc[:, 40:] == np.iinfo(np.int32).min)
    ixu.close()


@pytest.mark.parametrize("algo", ALGOS)
@pytest.mark.parametrize("N,k,tile", [(5000, 100, 64), (70_001, 1000, 512), (70_001, 4096, 512)])
def test_closed_form_ties_across_tiles(gs, algo, N, k, tile):
    """Every doc holds only term 0 with weight floor(d/2): ranking known in closed form, pairs tie -> lower id first."""
    indptr = np.arange(N + 1, dtype=np.int64)
    docs = wl.Csr(indptr, np.zeros(N, np.int32), (np.arange(N) // 2).astype(np.float32))
    q = csr_from_dicts([{0: 1.0}, {0: 0.5}], np.float32)
    ix = gs.Index.from_numpy(docs, 4, tile_docs=tile)
    ids, sc = gpu_search(gs, ix, q, k, **aopt(algo))
    # descending score = descending floor(d/2); inside a pair (2j, 2j+1) the lower id comes first
    order = sorted(range(N), key=lambda d: (-(d // 2), d))[:k]
    assert ids[0].tolist() == order and ids[1].tolist() == order
    assert sc[0].tolist() == [float(d // 2) for d in order]
    assert sc[1].tolist() == [0.5 * (d // 2) for d in order]
    ix.close()
    # u8 twin: weight (d mod 7)+1, query impact 3
    du = wl.Csr(indptr, np.zeros(N, np.int32), ((np.arange(N) % 7) + 1).astype(np.uint8))
    qu = csr_from_dicts([{0: 3}], np.uint8)
    ixu = gs.Index.from_numpy(du, 4, tile_docs=tile)
    ids, sc = gpu_search(gs, ixu, qu, k, **aopt(algo))
    order = sorted(range(N), key=lambda d: (-((d % 7) + 1), d))[:k]
    assert ids[0].tolist() == order and sc[0].tolist() == [3 * ((d % 7) + 1) for d in order]
    ixu.close()


@pytest.mark.parametrize("algo", ALGOS)
def test_padding_sentinel_never_surfaces(gs, algo):
    """A list of length 33 (== 1 mod 32); k > 33: the remaining slots are real zero-score docs in id order, never -1."""
    N, V = 300, 16
    rows = [{1: 1.0} for _ in range(N)]
    hit = list(range(5, 5 + 33 * 7, 7))
    for j, d in enumerate(hit):
        rows[d][7] = 1.0 + j
    docs = csr_from_dicts(rows, np.float32)
    ix = gs.Index.from_numpy(docs, V, tile_docs=32, head_max=-1)
    lids, _ = ix.posting_list(7)
    assert len(lids) == 64 and lids[:33].tolist() == hit and np.all(lids[33:] == -1)
    q = csr_from_dicts([{7: 2.0}], np.float32)
    ids, sc = gpu_search(gs, ix, q, 50, **aopt(algo))
    assert ids[0, :33].tolist() == hit[::-1]
    rest = [d for d in range(N) if d not in set(hit)][:17]
    assert ids[0, 33:].tolist() == rest and np.all(sc[0, 33:] == 0) and np.all(ids >= 0)
    ix.close()


@pytest.mark.parametrize("algo", ALGOS)
def test_signed_weights_and_negative_zero(gs, algo):
    """Any finite weight is legal: negative scores rank below zero-score docs; -0.0 ties with +0.0."""
    rng = np.random.default_rng(11)
    N, V = 3000, 200
    rows = []
    for _ in range(N):
        t = rng.choice(V, size=int(rng.integers(1, 30)), replace=False)
        rows.append({int(x): float(np.float32(rng.normal())) for x in t})
    rows[10] = {3: -0.0}
    docs = csr_from_dicts(rows, np.float32)
    qs = []
    for _ in range(9):
        t = rng.choice(V, size=int(rng.integers(1, 12)), replace=False)
        qs.append({int(x): float(np.float32(rng.normal())) for x in t})
    qs.append({3: 1.0})
    q = csr_from_dicts(qs, np.float32)
    ix = gs.Index.from_numpy(docs, V, tile_docs=128)
    for k in (10, 2999, 3000):
        ids, sc = gpu_search(gs, ix, q, k, **aopt(algo))
        R_d, R_q = oracle.as_rows(docs, V), oracle.as_rows(q, V)
        o_ids, o_sc = oracle.search(R_q, R_d, k)
        # cancellation makes |score| small relative to the summands: compare with an absolute bound from the summand sizes
        for b in range(q.rows):
            t = oracle.score_pairs(R_q, R_d, np.full(k, b, np.int64), ids[b].astype(np.int64))
            atol = 1e-5 * 30 * 16
            assert np.all(np.abs(sc[b] - t) <= atol), "score error"
            assert np.all(np.diff(sc[b]) <= 0) and len(set(ids[b].tolist())) == k
            eq = np.nonzero(np.diff(sc[b]) == 0)[0]
            assert np.all(ids[b][eq] < ids[b][eq + 1])
            # the top-k SET against the oracle's (same rule as parity.check_f32_row, with the absolute bound): every
            # document clearly above the oracle's k-th score is returned, nothing returned is clearly below it, and the
            # returned order does not contradict the true scores
            tau = o_sc[b][k - 1]
            must = o_ids[b][o_sc[b] > tau + 2 * atol]
            assert np.all(np.isin(must, ids[b])), "a clearly-top-k document is missing"
            assert np.all(t >= tau - 2 * atol), "a returned document is clearly below the k-th score"
            assert np.all(t[:-1] >= t[1:] - 2 * atol), "returned order contradicts true scores"
    ix.close()


# ----------------------------------------------------------------------------------------------------
# top-k selection alone (S3) on synthetic score arrays vs a host full sort
# ----------------------------------------------------------------------------------------------------
def host_topk(row, k):
    """(score desc, id asc) by a stable full sort; -0.0 ranks equal to +0.0."""
    n = len(row)
    key = row.astype(np.float64) + 0.0
    order = np.lexsort((np.arange(n), -key))[:k]
    return order


# rows of up to 2^20 items take the one-launch cluster select, longer rows the multi-launch one: both sides of the switch
@pytest.mark.parametrize("n,k", [(1, 1), (100, 100), (5000, 10), (100_000, 1000), (300_001, 4096), (1_048_576, 10),
                                 (1_048_577, 1000), (1_300_003, 4096)])
def test_topk_dense_synthetic_f32(gs, n, k):
    import torch
    rng = np.random.default_rng(n + k)
    rows = [
        np.zeros(n, np.float32),                                             # all equal
        np.arange(n, 0, -1).astype(np.float32),                              # strictly descending
        np.arange(n).astype(np.float32),                                     # strictly ascending
        rng.lognormal(0, 0.5, n).astype(np.float32),
        np.where(rng.random(n) < 0.5, 1.5, rng.random(n)).astype(np.float32),   # k-th value massively repeated
        (rng.integers(0, 3, n) * np.float32(1e-45)).astype(np.float32),      # denormals
        np.where(rng.random(n) < 0.5, -0.0, 0.0).astype(np.float32),         # +-0
        rng.normal(size=n).astype(np.float32),                               # signed
    ]
    S = np.stack(rows)
    k = min(k, gs.GS_MAX_K)
    ids, sc = gs.topk_dense(torch.from_numpy(S).cuda(), k)
    ids, sc = ids.cpu().numpy(), sc.cpu().numpy()
    for r in range(S.shape[0]):
        want = host_topk(S[r], k)
        assert np.array_equal(ids[r, :len(want)], want), f"row {r}"
        assert np.array_equal(sc[r, :len(want)] + 0.0, S[r][want] + 0.0)


def test_topk_dense_synthetic_i32(gs):
    import torch
    rng = np.random.default_rng(2)
    n, k = 77_777, 500
    S = np.stack([rng.integers(0, 50, n), rng.integers(-2**31, 2**31 - 1, n), np.full(n, 7)]).astype(np.int32)
    ids, sc = gs.topk_dense(torch.from_numpy(S).cuda(), k)
    for r in range(3):
        want = np.lexsort((np.arange(n), -S[r].astype(np.int64)))[:k]
        assert np.array_equal(ids[r].cpu().numpy(), want) and np.array_equal(sc[r].cpu().numpy(), S[r][want])


# ----------------------------------------------------------------------------------------------------
# host-buffer entry point, error codes, mid-scale sampled parity
# ----------------------------------------------------------------------------------------------------
def test_search_host_matches_device_search(gs, tiny):
    ix = gs.Index.from_numpy(tiny.docs, tiny.vocab)
    q = tiny.queries
    ids_h, sc_h = ix.search_host(q.indptr, q.terms, q.weights, 10, algo="term")
    ids_d, sc_d = gpu_search(gs, ix, q, 10, algo="term")
    assert np.array_equal(ids_h, ids_d) and np.array_equal(sc_h, sc_d)
    compare(gs, tiny.docs, q, tiny.vocab, 10, ids_h, sc_h)
    ix.close()


def test_error_codes(gs, tiny):
    import torch
    d = tiny.docs
    bad = wl.Csr(d.indptr[:11].copy(), d.terms[:int(d.indptr[10])].copy(), d.weights[:int(d.indptr[10])].copy())
    t = bad.terms.copy(); t[3] = wl.VOCAB
    with pytest.raises(gs.GsError) as e:
        gs.Index.from_numpy(wl.Csr(bad.indptr, t, bad.weights), wl.VOCAB)
    assert e.value.code == 2
    t = bad.terms.copy(); t[1] = t[0]
    with pytest.raises(gs.GsError) as e:
        gs.Index.from_numpy(wl.Csr(bad.indptr, t, bad.weights), wl.VOCAB)
    assert e.value.code == 3
    w = bad.weights.copy(); w[5] = np.nan
    with pytest.raises(gs.GsError) as e:
        gs.Index.from_numpy(wl.Csr(bad.indptr, bad.terms, w), wl.VOCAB)
    assert e.value.code == 4
    ix = gs.Index.from_numpy(bad, wl.VOCAB)
    q = tiny.queries
    with pytest.raises(gs.GsError) as e:
        gpu_search(gs, ix, q, 0)
    assert e.value.code == 2
    with pytest.raises(gs.GsError) as e:
        gpu_search(gs, ix, q.to_u8(), 5)
    assert e.value.code == 8
    qt = q.terms.copy(); qt[1] = qt[0]
    with pytest.raises(gs.GsError) as e:
        gpu_search(gs, ix, wl.Csr(q.indptr, qt, q.weights), 5, flags=gs.GS_FLAG_VALIDATE_QUERIES)
    assert e.value.code == 3
    ix.close()


@pytest.mark.parametrize("algo", ALGOS)
@pytest.mark.parametrize("mode", ["f32", "u8"])
def test_mid_prefix_full_compare(gs, mode, algo):
    """First 200K docs of the 8.8M collection (several hundred tiles, ragged tail), 8 queries, k=1000: full oracle compare."""
    docs = wl.make_docs("mid", n_docs=200_003)
    queries = wl.make_queries("mid", n_queries=8)
    if mode == "u8":
        docs, queries = docs.to_u8(), queries.to_u8()
    ix = gs.Index.from_numpy(docs, wl.VOCAB)
    ids, sc = gpu_search(gs, ix, queries, 1000, **aopt(algo))
    worst, subs = compare(gs, docs, queries, wl.VOCAB, 1000, ids, sc)
    st = ix.stats()
    assert st["overflow_queries"] == 0
    ix.close()


BATCH_KERNEL_WARPS = 32   # kBWarps of score_term.cu


@pytest.mark.parametrize("mode", ["f32", "u8"])
@pytest.mark.parametrize("qcfg", ["mid", "skew_b32"])
@pytest.mark.parametrize("build_kw", [dict(), dict(tile_docs=96, head_max=5), dict(head_max=-1), dict(tile_docs=1024, head_density=0.05)])
def test_batch_of_256_takes_the_cta_per_tile_term_kernels(gs, mode, build_kw, qcfg):
    """From 128 queries on (64 on collections of at least 8192 doc tiles) the term-parallel kernel runs as a persistent CTA per doc tile with the strips staged in shared
    memory (unless the index has no strips) — the batch kernel on 512-doc tiles, the generic staged kernel on other tile sizes:
    every score of 256 queries x 20 011 docs, and the top-50, against the oracle.  The "skew_b32" queries (5..256 terms,
    Zipf 1.3) have more than 32 tail terms, which the batch kernel probes in line after the prefetched first 32."""
    docs = wl.make_docs("mid", n_docs=20_011)
    queries = wl.make_queries(qcfg, n_queries=256)
    if mode == "u8":
        docs, queries = docs.to_u8(), queries.to_u8()
    ix = gs.Index.from_numpy(docs, wl.VOCAB, **build_kw)
    S = ix.score_dense(*dev(queries), algo="term").cpu().numpy()[:, :docs.rows]
    R_d, R_q = oracle.as_rows(docs, wl.VOCAB), oracle.as_rows(queries, wl.VOCAB)
    _, _, A = oracle.search(R_q, R_d, 1, all_scores=True)
    if mode == "u8":
        assert np.array_equal(S.astype(np.int64), A.astype(np.int64))
    else:
        assert np.all(np.abs(S.astype(np.float64) - A) <= parity.tol(A))
    # cell rows per CTA: batch kernel (512-doc tiles), generic staged shape (other tilings) or small shape (no strips)
    st_expect = 2 if build_kw.get("head_max", 0) == -1 else (32 if "tile_docs" in build_kw else BATCH_KERNEL_WARPS)
    for opt in (dict(algo="term"), dict(algo="auto"), dict(algo="term", flags=gs.GS_FLAG_FORCE_DENSE_TOPK)):
        ids, sc = gpu_search(gs, ix, queries, 50, **opt)
        assert ix.stats()["query_group"] == st_expect and ix.stats()["algo_used"] == 1
        compare(gs, docs, queries, wl.VOCAB, 50, ids, sc)
    ix.close()


@pytest.mark.parametrize("mode", ["f32", "u8"])
def test_candidate_overflow_of_a_batch_falls_back_to_the_dense_path_with_second_tier_strips(gs, mode):
    """130 queries over 200 000 docs built so that the threshold sample (every 64th doc tile at this N and k) sees none of the
    high-scoring documents: every candidate list overflows and the queries are re-run through the dense path in sub-batches
    (the warp-per-row kernel) while the batch still carries its second-tier strip lists (term 1: density 0.2).  Exact
    against the oracle."""
    n = 200_000
    dt = np.float32 if mode == "f32" else np.uint8
    d = np.arange(n)
    has1, has2 = (d % 5 == 3) & ((d // 512) % 64 != 0), d % 50 == 7
    nnz = 1 + has1.astype(np.int64) + has2.astype(np.int64)
    indptr = np.concatenate([[0], np.cumsum(nnz)]).astype(np.int64)
    terms = np.zeros(indptr[-1], np.int32)
    terms[indptr[:-1][has1] + 1] = 1
    terms[indptr[1:][has2] - 1] = 2
    docs = wl.Csr(indptr, terms, np.ones(indptr[-1], dt))
    queries = csr_from_dicts([{0: 1, 1: 1, 2: 1 + (b % 3)} for b in range(130)], dt)
    ix = gs.Index.from_numpy(docs, 8)
    assert ix.info()["head_terms_term_parallel"] > ix.info()["head_terms"]          # term 1 is a second-tier strip
    ids, sc = gpu_search(gs, ix, queries, 50, algo="term")
    assert ix.stats()["overflow_queries"] > 0
    compare(gs, docs, queries, 8, 50, ids, sc)
    ix.close()


def test_batch_kernel_is_deterministic_run_to_run(gs):
    """DESIGN.md R2: every (query, doc) cell is owned by one warp and its additions keep the query's term order, so the fp32
    scores of the batch kernel are bitwise identical from run to run (the candidate lists are not ordered, the results are)."""
    docs = wl.make_docs("mid", n_docs=20_011)
    queries = wl.make_queries("skew_b32", n_queries=256)
    ix = gs.Index.from_numpy(docs, wl.VOCAB)
    S0 = ix.score_dense(*dev(queries), algo="term").cpu().numpy()
    ids0, sc0 = gpu_search(gs, ix, queries, 100, algo="term")
    assert ix.stats()["query_group"] == BATCH_KERNEL_WARPS
    for _ in range(3):
        assert np.array_equal(ix.score_dense(*dev(queries), algo="term").cpu().numpy().view(np.uint32), S0.view(np.uint32))
        ids, sc = gpu_search(gs, ix, queries, 100, algo="term")
        assert np.array_equal(ids, ids0) and np.array_equal(sc.view(np.uint32), sc0.view(np.uint32))
    ix.close()


# ----------------------------------------------------------------------------------------------------
# paper scale (BASELINE.json configs[2] and [3]) in the launch configuration bench.py times
# ----------------------------------------------------------------------------------------------------
@pytest.fixture(scope="module")
def paper_docs():
    return wl.make_docs("paper")            # 8.8M docs, 1.06e9 postings (~3 s on the box's cores)


@pytest.mark.parametrize("mode,k", [("f32", 1000), ("u8", 10)])
def test_paper_scale_sampled(gs, paper_docs, mode, k):
    """All B=500 queries: structure + every returned score against the oracle's pairwise score (one merge each);
    a sample of queries (one per host core, at most 16): the complete top-k against the oracle's exhaustive search."""
    docs = paper_docs if mode == "f32" else paper_docs.to_u8()
    queries = wl.make_queries("paper" if mode == "f32" else "paper_u8")
    assert docs.rows == 8_800_000 and queries.rows == 500
    R_d, R_q = oracle.as_rows(docs, wl.VOCAB), oracle.as_rows(queries, wl.VOCAB)
    n_s = max(1, min(16, oracle.max_threads()))
    sample = np.linspace(0, queries.rows - 1, n_s).astype(np.int64)
    R_s = oracle.as_rows(wl.Csr(*_take_rows(queries, sample)), wl.VOCAB)
    o_ids, o_sc = oracle.search(R_s, R_d, k)
    ix = gs.Index.from_numpy(docs, wl.VOCAB)
    batch_ids = None
    for algo in ("term", "doc"):
        ids, sc = gpu_search(gs, ix, queries, k, **aopt(algo))
        batch_ids = ids
        assert ix.stats()["overflow_queries"] == 0
        b_idx = np.repeat(np.arange(queries.rows, dtype=np.int64), k)
        true = oracle.score_pairs(R_q, R_d, b_idx, ids.reshape(-1).astype(np.int64)).reshape(queries.rows, k)
        if mode == "u8":
            assert np.array_equal(sc.astype(np.int64), true)
            parity.check_int_exact(ids[sample], sc[sample], o_ids, o_sc)
        else:
            assert np.all(np.abs(sc - true) <= parity.tol(true))
            for j, b in enumerate(sample):
                parity.check_f32_row(ids[b], sc[b], o_ids[j], o_sc[j], true[b], docs.rows)
        for b in range(queries.rows):                      # structure of every row
            assert len(np.unique(ids[b])) == k and ids[b].min() >= 0 and ids[b].max() < docs.rows
            d = np.diff(sc[b].astype(np.float64))
            assert np.all(d <= 0) and np.all(ids[b][:-1][d == 0] < ids[b][1:][d == 0])
    # small batches take other plans (bigger threshold sample stride, document-parallel with a tile of 8)
    few = queries.slice_rows(0, 3)
    for opt in (dict(algo="term"), dict(algo="term", query_group=8), dict(algo="doc"), dict(algo="auto")):
        ids, sc = gpu_search(gs, ix, few, k, **opt)
        b_idx = np.repeat(np.arange(few.rows, dtype=np.int64), k)
        true = oracle.score_pairs(R_q, R_d, b_idx, ids.reshape(-1).astype(np.int64)).reshape(few.rows, k)
        if mode == "u8":
            assert np.array_equal(sc.astype(np.int64), true) and np.array_equal(ids, batch_ids[:few.rows])
        else:
            assert np.all(np.abs(sc - true) <= parity.tol(true))
            if sample[0] == 0:
                parity.check_f32_row(ids[0], sc[0], o_ids[0], o_sc[0], true[0], docs.rows)
    ix.close()


def _take_rows(csr, rows):
    indptr, terms, weights = [0], [], []
    for r in rows:
        t, w = csr.row(int(r))
        terms.append(t); weights.append(w)
        indptr.append(indptr[-1] + len(t))
    return np.array(indptr, np.int64), np.concatenate(terms), np.concatenate(weights)


# ----------------------------------------------------------------------------------------------------
# the boundary: asynchronous gs_search (CUDA-graph capture), gs_search_finish, allocator callbacks, indptr checks
# ----------------------------------------------------------------------------------------------------
def test_search_is_asynchronous_and_replays_from_a_cuda_graph(gs, tiny):
    """gs_search only enqueues work: captured once into a CUDA graph, the search is replayed for new query data written
    into the same buffers, and every replay matches the oracle (asynchronous on the stream, never allocates)."""
    import torch
    docs = wl.make_docs("mid", n_docs=60_011)
    ix = gs.Index.from_numpy(docs, wl.VOCAB)
    k, B = 10, 4
    all_q = wl.make_queries("mid", n_queries=3 * B)
    cap_nnz = int(max(all_q.slice_rows(i * B, (i + 1) * B).nnz for i in range(3)))
    d = torch.device("cuda:0")
    q_ip = torch.zeros(B + 1, dtype=torch.int64, device=d)
    q_t = torch.zeros(cap_nnz, dtype=torch.int32, device=d)
    q_w = torch.zeros(cap_nnz, dtype=torch.float32, device=d)
    ws = torch.empty(ix.workspace_bytes(B, cap_nnz, k, algo="term"), dtype=torch.uint8, device=d)
    out_ids = torch.empty((B, k), dtype=torch.int32, device=d)
    out_sc = torch.empty((B, k), dtype=torch.float32, device=d)

    def put(q):
        q_ip.copy_(torch.from_numpy(q.indptr))
        q_t[:q.nnz].copy_(torch.from_numpy(q.terms))
        q_w[:q.nnz].copy_(torch.from_numpy(q.weights))

    put(all_q.slice_rows(0, B))
    ix.search(q_ip, q_t, q_w, k, out_ids=out_ids, out_scores=out_sc, workspace=ws, algo="term")     # warm-up (module load, attributes)
    torch.cuda.synchronize()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g):
        ix.search(q_ip, q_t, q_w, k, out_ids=out_ids, out_scores=out_sc, workspace=ws, algo="term", finish=False)
    n_launch = gs.last_launch_count()
    assert n_launch > 0
    for i in range(3):
        q = all_q.slice_rows(i * B, (i + 1) * B)
        put(q)
        out_ids.fill_(-7)
        g.replay()
        torch.cuda.synchronize()
        assert ix.stats(ws)["overflow_queries"] == 0
        # the CSR arrays keep their captured length: entries past indptr[B] are never read
        compare(gs, docs, q, wl.VOCAB, k, out_ids.cpu().numpy(), out_sc.cpu().numpy())
    ix.close()


def test_finish_resolves_overflow_after_an_asynchronous_search(gs):
    """finish=False leaves the overflowed rows inexact and flagged; gs_search_finish re-runs exactly those queries."""
    n = 200_000
    d = np.arange(n)
    has1, has2 = (d % 5 == 3) & ((d // 512) % 64 != 0), d % 50 == 7
    nnz = 1 + has1.astype(np.int64) + has2.astype(np.int64)
    indptr = np.concatenate([[0], np.cumsum(nnz)]).astype(np.int64)
    terms = np.zeros(indptr[-1], np.int32)
    terms[indptr[:-1][has1] + 1] = 1
    terms[indptr[1:][has2] - 1] = 2
    docs = wl.Csr(indptr, terms, np.ones(indptr[-1], np.float32))
    # the queries that use term 1 (which the sampled tiles never hold) overflow; query 1 does not
    queries = csr_from_dicts([{0: 1, 1: 1, 2: 2}, {0: 1}, {0: 1, 1: 1, 2: 1}, {0: 2, 1: 1}], np.float32)
    ix = gs.Index.from_numpy(docs, 8)
    qd = dev(queries)
    ids, sc = ix.search(*qd, 50, algo="term", finish=False)
    st = ix.stats()
    n_ov = st["overflow_queries"]
    assert 2 <= n_ov <= 3
    resolved = ix.finish(*qd, 50, ids, sc, ix._last_ws, algo="term")
    assert resolved == n_ov
    compare(gs, docs, queries, 8, 50, ids.cpu().numpy(), sc.cpu().numpy())
    ix.close()


def test_index_build_through_allocator_callbacks(gs, tiny):
    """gs_alloc_t: everything the handle owns comes from the caller's allocator (here torch's caching allocator through
    ctypes callbacks) and goes back to it on gs_index_free."""
    import ctypes
    import torch
    live = {}

    @ctypes.CFUNCTYPE(ctypes.c_void_p, ctypes.c_size_t, ctypes.c_void_p, ctypes.c_void_p)
    def c_alloc(nbytes, stream, user):
        p = torch.cuda.caching_allocator_alloc(int(nbytes), device=0)
        live[p] = int(nbytes)
        return p

    @ctypes.CFUNCTYPE(None, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p)
    def c_free(ptr, stream, user):
        live.pop(ptr)
        torch.cuda.caching_allocator_delete(ptr)

    ix = gs.Index.from_numpy(tiny.docs, tiny.vocab, allocator=(c_alloc, c_free))
    assert len(live) >= 8 and sum(live.values()) >= ix.info()["bytes_total"]
    ids, sc = gpu_search(gs, ix, tiny.queries, 10, algo="term")
    compare(gs, tiny.docs, tiny.queries, tiny.vocab, 10, ids, sc)
    ids, sc = ix.search_host(tiny.queries.indptr, tiny.queries.terms, tiny.queries.weights, 10, algo="doc")
    compare(gs, tiny.docs, tiny.queries, tiny.vocab, 10, ids, sc)
    ix.close()
    assert not live, "gs_index_free must return every block to the allocator"


def test_malformed_query_indptr_is_rejected_not_dereferenced(gs, tiny):
    """A non-monotone / out-of-range query indptr must never index past the nnz-sized arrays: the rows are treated as
    empty, and with validation on the call returns GS_ERR_OUT_OF_RANGE."""
    ix = gs.Index.from_numpy(tiny.docs, tiny.vocab)
    q = tiny.queries
    for bad in ("decreasing", "past_end", "first_not_zero"):
        ip = q.indptr.copy()
        if bad == "decreasing":
            ip[3] = ip[2] - 1
        elif bad == "past_end":
            ip[-1] = q.nnz + 1000
        else:
            ip[0] = 2
        bq = wl.Csr(ip, q.terms, q.weights)
        for algo in ("term", "doc"):
            with pytest.raises(gs.GsError) as e:
                gpu_search(gs, ix, bq, 5, algo=algo, flags=gs.GS_FLAG_VALIDATE_QUERIES)
            assert e.value.code == 2
            ids, sc = gpu_search(gs, ix, bq, 5, algo=algo)       # validation off: memory-safe, result unspecified
            assert ids.shape == (q.rows, 5)
    ids, sc = gpu_search(gs, ix, q, 5)                           # the handle is still healthy
    compare(gs, tiny.docs, q, tiny.vocab, 5, ids, sc)
    ix.close()


# ----------------------------------------------------------------------------------------------------
# Compressed postings (PAPER.md L430 future work 2; gs_build_opts_t.pack_postings): integer-impact mode packs a posting into
# one 32-bit word in the inverted lists and in the forward index.  Both layouts must give the oracle's results bit for bit,
# the packed one must be the smaller one, and its lists must still read back as Eq. 2 states them.
# ----------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("pack", [True, False])
def test_compressed_postings_layout_and_eq2_readback(gs, pack):
    g = json.load(open(os.path.join(GOLD, "handworked_3doc.json")))
    docs = csr_from_dicts(g["u8"]["docs"], np.uint8)
    ix = gs.Index.from_numpy(docs, g["vocab"], pack_postings=pack)
    inf = ix.info()
    assert inf["packed_layout"] == (3 if pack else 0)
    assert inf["bytes_inverted"] == inf["padded_nnz"] * (4 if pack else 5)
    want = {}
    for d, row in enumerate(g["u8"]["docs"]):
        for t, w in row.items():
            want.setdefault(int(t), []).append((d, int(w)))
    for t, lst in want.items():
        ids, w = ix.posting_list(t)
        assert len(ids) == 32 and [(int(i), int(x)) for i, x in zip(ids[:len(lst)], w[:len(lst)])] == lst
        assert np.all(ids[len(lst):] == -1) and np.all(w[len(lst):] == 0)        # sentinel (doc_id=-1, score=0), L90
    ix.close()


@pytest.mark.parametrize("algo", ALGOS)
@pytest.mark.parametrize("build_kw", [dict(), dict(tile_docs=96, head_max=-1)])
def test_compressed_postings_match_the_two_array_layout_and_the_oracle(gs, tiny, algo, build_kw):
    docs, queries = tiny.docs.to_u8(), tiny.queries.to_u8()
    sizes = {}
    for pack in (True, False):
        _dense_parity(gs, docs, queries, tiny.vocab, algo, pack_postings=pack, **build_kw)
        ix = gs.Index.from_numpy(docs, tiny.vocab, pack_postings=pack, **build_kw)
        ids, sc = gpu_search(gs, ix, queries, 33, **aopt(algo))
        compare(gs, docs, queries, tiny.vocab, 33, ids, sc)
        inf = ix.info()
        sizes[pack] = (inf["bytes_inverted"], inf["bytes_forward"])
        ix.close()
    assert sizes[True][0] * 5 == sizes[False][0] * 4                  # 4 instead of 5 bytes per inverted posting
    assert sizes[True][1] < 0.85 * sizes[False][1]                    # forward index: -20 % minus the block pointers


def test_compressed_postings_in_the_batch_kernel(gs):
    """256 queries take the CTA-per-doc-tile batch kernel: its flat posting stream reads packed words."""
    docs = wl.make_docs("mid", n_docs=20_011).to_u8()
    queries = wl.make_queries("mid", n_queries=256).to_u8()
    for pack in (True, False):
        ix = gs.Index.from_numpy(docs, wl.VOCAB, pack_postings=pack)
        ids, sc = gpu_search(gs, ix, queries, 10, algo="term")
        assert ix.stats()["query_group"] >= 32
        compare(gs, docs, queries, wl.VOCAB, 10, ids, sc)
        ix.close()


# ----------------------------------------------------------------------------------------------------
# Integer-impact mode, batches: the head contraction on the tensor cores (tcgen05.mma kind::i8, k_score_term_mma,
# GS_FLAG_TENSOR_CORE_HEAD) must be bit-identical to the CUDA-core path and to the oracle — every score, then the top-k.
# ----------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("n_docs,n_q", [(20_011, 256), (3_000, 130), (70_001, 500)])
def test_tensor_core_head_contraction_is_bit_exact(gs, n_docs, n_q):
    docs = wl.make_docs("mid", n_docs=n_docs).to_u8()
    queries = wl.make_queries("mid", n_queries=n_q).to_u8()
    R_d, R_q = oracle.as_rows(docs, wl.VOCAB), oracle.as_rows(queries, wl.VOCAB)
    o_ids, o_sc, A = oracle.search(R_q, R_d, 100, all_scores=True)
    ix = gs.Index.from_numpy(docs, wl.VOCAB)
    for flags in (gs.GS_FLAG_TENSOR_CORE_HEAD, 0):
        S = ix.score_dense(*dev(queries), algo="term", flags=flags).cpu().numpy()[:, :docs.rows]
        assert np.array_equal(S.astype(np.int64), A.astype(np.int64)), f"flags={flags}"
        ids, sc = gpu_search(gs, ix, queries, 100, algo="term", flags=flags)
        assert ix.stats()["query_group"] >= 32
        parity.check_int_exact(ids, sc, o_ids, o_sc)
    ix.close()
