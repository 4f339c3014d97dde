"""GS_ALGO_AUTO: the cost model of gs_dispatch_model (§5.3 crossover with B200-measured constants).

CPU part: the model is host arithmetic behind the C ABI, callable without a GPU.  It is checked against the paper's own
statement of the trade-off (the scatter side wins whenever a batch amortises the stream, L176-181) and against the B200
sweep recorded in profiles/r02_dispatch_sweep.md (which path was faster at each grid point).
GPU part: AUTO really takes both outcomes, and each outcome matches the oracle.
"""
import csv
import os

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def stream_bytes(n_docs, doc_nnz):
    return int(n_docs * doc_nnz * 8)          # forward postings + strips, about 8 bytes per posting in fp32


def test_model_picks_term_parallel_for_batches_and_doc_parallel_for_single_long_queries():
    from paper_2606_26441_b200 import binding as gs
    # BASELINE.json configs 1-5 (mean query nnz 25; config 5: ~131): all on the term-parallel side, as the paper finds (L181)
    for n, b, q in ((10_000, 16, 25), (1_000_000, 64, 25), (8_800_000, 500, 25), (8_800_000, 1, 131), (8_800_000, 32, 131)):
        algo, t, d = gs.dispatch_model(n, 512, stream_bytes(n, 120), b, b * q)
        assert algo == "term" and t < d
    # one query with hundreds of terms: the scatter probes every (term, doc tile) pair, the stream is read once
    for n in (20_000, 100_000, 1_000_000):
        for q in (1000, 4000):
            algo, t, d = gs.dispatch_model(n, 512, stream_bytes(n, 120), 1, q)
            assert algo == "doc" and d < t
    # monotone: more query terms never make a path cheaper; more queries never make the doc-parallel path cheaper
    _, t1, d1 = gs.dispatch_model(100_000, 512, stream_bytes(100_000, 120), 16, 16 * 25)
    _, t2, d2 = gs.dispatch_model(100_000, 512, stream_bytes(100_000, 120), 16, 16 * 250)
    _, t3, d3 = gs.dispatch_model(100_000, 512, stream_bytes(100_000, 120), 64, 64 * 250)
    assert t2 >= t1 and d2 >= d1 and d3 >= d2


def test_model_agrees_with_the_recorded_b200_sweep():
    """profiles/r02_dispatch_sweep.csv: measured ms of both paths on a 4 x 4 x 4 grid (collection, batch, query length).
    The model must name the faster path wherever the two differ by more than 10 %."""
    from paper_2606_26441_b200 import binding as gs
    with open(os.path.join(ROOT, "profiles", "r02_dispatch_sweep.csv"), newline="") as f:
        grid = [{k: (v if k == "winner" else float(v)) for k, v in r.items()} for r in csv.DictReader(f)]
    assert len(grid) >= 64
    wrong = 0
    for r in grid:
        algo, _, _ = gs.dispatch_model(int(r["n_docs"]), 512, stream_bytes(int(r["n_docs"]), int(r["doc_nnz"])), int(r["B"]),
                                       int(r["B"] * r["q_nnz"]))
        fast, slow = sorted((r["term_ms"], r["doc_ms"]))
        if slow > 1.10 * fast:
            assert algo == r["winner"], r
        elif algo != r["winner"]:
            wrong += 1
    assert wrong <= 4


@pytest.mark.gpu
@pytest.mark.parametrize("mode", ["f32", "u8"])
def test_auto_takes_both_paths_and_matches_the_oracle(mode):
    import torch
    import oracle
    import parity
    from paper_2606_26441_b200 import binding as gs, workload as wl
    docs = wl.make_rows(30_011, seed=3, stream=wl.STREAM_DOCS)
    long_q = wl.make_rows(1, seed=3, stream=wl.STREAM_QUERIES, mu=900, sigma=0.0, lo=900, hi=900)
    batch_q = wl.make_rows(48, seed=4, stream=wl.STREAM_QUERIES, mu=25, sigma=8, lo=5, hi=64)
    if mode == "u8":
        docs, long_q, batch_q = docs.to_u8(), long_q.to_u8(), batch_q.to_u8()
    R_d = oracle.as_rows(docs, wl.VOCAB)
    ix = gs.Index.from_numpy(docs, wl.VOCAB)
    d = torch.device("cuda:0")
    for q, want in ((long_q, "doc"), (batch_q, "term")):
        R_q = oracle.as_rows(q, wl.VOCAB)
        o_ids, o_sc = oracle.search(R_q, R_d, 10)
        ids, sc = ix.search(*[torch.from_numpy(np.ascontiguousarray(a)).to(d) for a in (q.indptr, q.terms, q.weights)], 10, algo="auto")
        assert ix.stats()["algo_used"] == gs.ALGOS[want]
        ids, sc = ids.cpu().numpy(), sc.cpu().numpy()
        if mode == "u8":
            parity.check_int_exact(ids, sc, o_ids, o_sc)
        else:
            # a (query, doc) pair shares at most the doc's terms (<= 400, ~100 in practice): n * 2^-24 relative
            # stays inside the 1e-5 of BASELINE.json
            parity.check_f32(ids, sc, o_ids, o_sc,
                             lambda b, i: oracle.score_pairs(R_q, R_d, np.full(len(i), b, np.int64), i.astype(np.int64)), docs.rows)
    ix.close()
