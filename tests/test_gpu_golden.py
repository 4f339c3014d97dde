"""Paper-scale parity of EVERY query against golden top-k lists — `-m gpu`, run on the B200 box.

The golden files under tests/golden/ were written by tests/golden/make_paper_golden.py, which calls only `oracle/`
(exhaustive merge scoring + full sort, Eq. 4, L61/L125) on the seeded generator's inputs.  They are
keyed by the generator's 64-bit array checksums: the inputs are regenerated here, their checksums compared with the
stored ones, and only then the results (last pin row).

  * BASELINE.json configs[2] (8.8M docs Zipf 1.1, B=500, k=1000, fp32) and configs[3] (uint8 twin, k=10): set, order and
    value of all 500 rows, both kernels, in the launch configuration bench.py times;
  * configs[4] (8.8M docs with Zipf 1.3 term ids, queries of 5..256 terms, k=10): B=1, B=32 and a batch of 64, every
    kernel shape, fp32 and the uint8 twin — on the collection's OWN distribution.
The smaller Zipf-1.3 collection (200 003 docs) is compared with the oracle directly.
"""
import os

import numpy as np
import pytest

import oracle
from paper_2606_26441_b200 import workload as wl
import parity

pytestmark = pytest.mark.gpu
GOLD = os.path.join(os.path.dirname(__file__), "golden")


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


def gpu_search(ix, queries, k, **opt):
    ids, sc = ix.search(*dev(queries), k, **opt)
    return ids.cpu().numpy(), sc.cpu().numpy()


def load_golden(name, docs, queries):
    path = os.path.join(GOLD, name)
    assert os.path.exists(path), f"{name} missing: run tests/golden/make_paper_golden.py"
    g = np.load(path)
    have = np.array([wl.checksum(docs.indptr), wl.checksum(docs.terms), wl.checksum(docs.weights),
                     wl.checksum(queries.indptr), wl.checksum(queries.terms), wl.checksum(queries.weights)], dtype=np.uint64)
    if not np.array_equal(have, g["checksums"]):
        pytest.skip(f"{name}: the generator's arrays differ from the ones the golden file was computed from (other libm?)")
    assert int(g["n_docs"]) == docs.rows
    return g["ids"], g["scores"]


def check_rows(mode, ids, sc, rows, o_ids, o_sc, R_q, R_d, n_docs):
    """GPU rows `ids/sc` (for the queries `rows` of R_q) against golden rows o_ids/o_sc of the same queries."""
    k = ids.shape[1]
    if mode == "u8":
        parity.check_int_exact(ids, sc, o_ids, o_sc)
        return 0.0, 0
    b_idx = np.repeat(np.asarray(rows, dtype=np.int64), k)
    true = oracle.score_pairs(R_q, R_d, b_idx, ids.reshape(-1).astype(np.int64)).reshape(len(rows), k)
    worst, subs = 0.0, 0
    for j in range(len(rows)):
        w, s = parity.check_f32_row(ids[j], sc[j], o_ids[j], o_sc[j], true[j], n_docs)
        worst, subs = max(worst, w), subs + s
    return worst, subs


# ----------------------------------------------------------------------------------------------------
# configs[2] / configs[3]: all 500 queries at 8.8M docs
# ----------------------------------------------------------------------------------------------------
@pytest.fixture(scope="module")
def paper_docs():
    return wl.make_docs("paper")


@pytest.mark.parametrize("mode,k,gold", [("f32", 1000, "paper_topk_f32.npz"), ("u8", 10, "paper_topk_u8.npz")])
def test_paper_scale_all_queries_against_golden(gs, paper_docs, mode, k, gold):
    docs = paper_docs if mode == "f32" else paper_docs.to_u8()
    queries = wl.make_queries("paper" if mode == "f32" else "paper_u8")
    o_ids, o_sc = load_golden(gold, docs, queries)
    assert o_ids.shape == (500, k)
    R_d = oracle.as_rows(docs, wl.VOCAB) if mode == "f32" else None      # only the fp32 comparator needs pairwise scores
    R_q = oracle.as_rows(queries, wl.VOCAB) if mode == "f32" else None
    ix = gs.Index.from_numpy(docs, wl.VOCAB)
    rows = np.arange(queries.rows)
    for opt in (dict(algo="auto"), dict(algo="term"), dict(algo="doc")):
        ids, sc = gpu_search(ix, queries, k, **opt)
        assert ix.stats()["overflow_queries"] == 0
        check_rows(mode, ids, sc, rows, o_ids, o_sc, R_q, R_d, docs.rows)
    ix.close()


# ----------------------------------------------------------------------------------------------------
# configs[4]: Zipf-1.3 documents.  Kernel shapes: warp-per-row (default for B < 64), pinned row groups, the batch
# kernel (B = 64 at 8.8M docs), doc-parallel with tiles of 8 / 16, AUTO.
# ----------------------------------------------------------------------------------------------------
SKEW_OPTS = [dict(algo="term"), dict(algo="term", query_group=1), dict(algo="term", query_group=8), dict(algo="doc"), dict(algo="auto")]


@pytest.fixture(scope="module")
def skew_docs():
    return wl.make_docs("skew_b32")


@pytest.mark.parametrize("mode,gold", [("f32", "skew_topk_f32.npz"), ("u8", "skew_topk_u8.npz")])
def test_skew_paper_scale_against_golden(gs, skew_docs, mode, gold):
    k = 10
    docs = skew_docs if mode == "f32" else skew_docs.to_u8()
    queries = wl.make_queries("skew_b32", n_queries=64)
    if mode == "u8":
        queries = queries.to_u8()
    o_ids, o_sc = load_golden(gold, docs, queries)
    R_d = oracle.as_rows(docs, wl.VOCAB) if mode == "f32" else None
    R_q = oracle.as_rows(queries, wl.VOCAB) if mode == "f32" else None
    ix = gs.Index.from_numpy(docs, wl.VOCAB)
    for opt in SKEW_OPTS:
        for b in (0, 1, 17):                                     # B = 1 (skew_b1): single queries
            ids, sc = gpu_search(ix, queries.slice_rows(b, b + 1), k, **opt)
            check_rows(mode, ids, sc, [b], o_ids[b:b + 1], o_sc[b:b + 1], R_q, R_d, docs.rows)
        ids, sc = gpu_search(ix, queries.slice_rows(0, 32), k, **opt)      # B = 32 (skew_b32)
        assert ix.stats()["overflow_queries"] == 0
        check_rows(mode, ids, sc, np.arange(32), o_ids[:32], o_sc[:32], R_q, R_d, docs.rows)
    for opt in (dict(algo="term"), dict(algo="doc", doc_query_tile=16)):   # 64 queries: the CTA-per-tile batch kernel
        ids, sc = gpu_search(ix, queries, k, **opt)
        check_rows(mode, ids, sc, np.arange(64), o_ids, o_sc, R_q, R_d, docs.rows)
    ix.close()


@pytest.mark.parametrize("mode", ["f32", "u8"])
def test_skew_docs_prefix_full_compare(gs, mode):
    """The first 200 003 documents of the Zipf-1.3 collection (391 doc tiles, ragged tail; more lists above the strip
    thresholds and far longer head lists than the Zipf-1.1 collections): B = 1 and B = 32 queries of 5..256 terms, k = 10,
    every kernel shape, against the oracle's exhaustive search; then every score of 128 queries element by element (128 queries take the CTA-per-tile batch kernel on this collection)."""
    docs = wl.make_docs("skew_b32", n_docs=200_003)
    queries = wl.make_queries("skew_b32", n_queries=128)
    if mode == "u8":
        docs, queries = docs.to_u8(), queries.to_u8()
    R_d, R_q = oracle.as_rows(docs, wl.VOCAB), oracle.as_rows(queries, wl.VOCAB)
    o_ids, o_sc, A = oracle.search(R_q, R_d, 10, all_scores=True)
    ix = gs.Index.from_numpy(docs, wl.VOCAB)
    assert ix.info()["head_terms"] >= 64
    for opt in SKEW_OPTS:
        ids, sc = gpu_search(ix, queries.slice_rows(5, 6), 10, **opt)
        check_rows(mode, ids, sc, [5], o_ids[5:6], o_sc[5:6], R_q, R_d, docs.rows)
        ids, sc = gpu_search(ix, queries.slice_rows(0, 32), 10, **opt)
        check_rows(mode, ids, sc, np.arange(32), o_ids[:32], o_sc[:32], R_q, R_d, docs.rows)
    ids, sc = gpu_search(ix, queries, 10, algo="term", query_group=-1)     # generic staged kernel
    check_rows(mode, ids, sc, np.arange(128), o_ids, o_sc, R_q, R_d, docs.rows)
    for algo in ("term", "doc"):
        S = ix.score_dense(*dev(queries), algo=algo).cpu().numpy()[:, :docs.rows]
        if mode == "u8":
            assert np.array_equal(S.astype(np.int64), A.astype(np.int64))
        else:
            # up to ~100 shared terms per pair on this collection: n * 2^-24 relative stays below 1e-5
            assert np.all(np.abs(S.astype(np.float64) - A) <= parity.tol(A))
    ix.close()
