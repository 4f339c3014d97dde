"""Pins for the CPU oracle (oracle/oracle.c) against things OTHER than itself.

The paper prints no worked scoring example, so the pins are: brute-force dense evaluation of
Eq. 4 on tiny inputs, scipy.sparse's Q @ D.T, a hand-worked example
(tests/golden/handworked_3doc.json), one-hot queries (scores == a column of D), closed-form tie
rankings, and invariants the definition implies.  A dropped term, a wrong sign/index, a
transposed operand or a wrong tie rule fails at least one of them.
"""
import json
import os

import numpy as np
import pytest
import scipy.sparse as sp

import oracle
from paper_2606_26441_b200 import workload as wl

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def csr_from_dicts(rows, dtype):
    indptr, terms, weights = [0], [], []
    for r in rows:
        for t, w in r.items():
            terms.append(int(t))
            weights.append(w)
        indptr.append(len(terms))
    return wl.Csr(np.array(indptr, np.int64), np.array(terms, np.int32), np.array(weights, dtype))


def random_csr(rng, rows, vocab, max_nnz, dtype, allow_empty=True, signed=False):
    indptr, terms, weights = [0], [], []
    for _ in range(rows):
        n = int(rng.integers(0 if allow_empty else 1, max_nnz + 1))
        t = rng.choice(vocab, size=min(n, vocab), replace=False)
        terms.extend(t.tolist())
        if dtype == np.uint8:
            weights.extend(rng.integers(1, 256, size=len(t)).tolist())
        else:
            w = rng.lognormal(0.0, 0.5, size=len(t))
            if signed:
                w *= rng.choice([-1.0, 1.0], size=len(t))
            weights.extend(w.tolist())
        indptr.append(len(terms))
    return wl.Csr(np.array(indptr, np.int64), np.array(terms, np.int32), np.array(weights, dtype))


def dense(csr, vocab, dtype):
    m = np.zeros((csr.rows, vocab), dtype=dtype)
    for r in range(csr.rows):
        t, w = csr.row(r)
        m[r, t] = w
    return m


def brute_topk(S, k):
    """Plain python: sort (score desc, id asc), pad per reading R4."""
    ids, sc = [], []
    neg = -np.inf if S.dtype.kind == "f" else np.iinfo(np.int32).min
    for b in range(S.shape[0]):
        order = sorted(range(S.shape[1]), key=lambda d: (-S[b, d], d))[:k]
        ids.append(order + [-1] * (k - len(order)))
        sc.append([S[b, d] for d in order] + [neg] * (k - len(order)))
    return np.array(ids, np.int32).reshape(S.shape[0], k), np.array(sc).reshape(S.shape[0], k)


def run(docs, queries, vocab, k, **kw):
    return oracle.search(oracle.as_rows(queries, vocab), oracle.as_rows(docs, vocab), k, **kw)


# ---------------------------------------------------------------- hand-worked example
@pytest.mark.parametrize("mode", ["f32", "u8"])
def test_handworked_three_docs(mode):
    g = json.load(open(os.path.join(GOLD, "handworked_3doc.json")))
    c = g[mode]
    dt = np.float32 if mode == "f32" else np.uint8
    ids, sc = run(csr_from_dicts(c["docs"], dt), csr_from_dicts(c["queries"], dt), g["vocab"], c["k"])
    assert ids.tolist() == c["expect_ids"]
    assert sc.tolist() == c["expect_scores"]


# ---------------------------------------------------------------- brute force dense (tiny)
@pytest.mark.parametrize("seed", range(6))
def test_dense_bruteforce_f32(seed):
    rng = np.random.default_rng(seed)
    V, N, B, k = 48, int(rng.integers(1, 50)), 5, 7
    docs = random_csr(rng, N, V, 12, np.float32, signed=(seed % 2 == 1))
    qs = random_csr(rng, B, V, 9, np.float32, signed=(seed % 2 == 1))
    D, Q = dense(docs, V, np.float64), dense(qs, V, np.float64)
    S = np.zeros((B, N))
    for b in range(B):          # triple loop of Eq. 4 written out
        for d in range(N):
            for t in range(V):
                S[b, d] += Q[b, t] * D[d, t]
    ids, sc, al = run(docs, qs, V, k, all_scores=True)
    np.testing.assert_allclose(al, S, rtol=0, atol=1e-12)
    eids, esc = brute_topk(al, k)     # ordering checked on the oracle's own scores: no fp ambiguity
    assert np.array_equal(ids, eids)
    assert np.array_equal(sc, esc)
    bids, _ = brute_topk(S, k)
    # where brute-force scores are separated by more than rounding noise the ranking must agree too
    for b in range(B):
        srt = np.sort(S[b])[::-1]
        if len(srt) < 2 or np.min(np.abs(np.diff(srt))[: k + 1]) > 1e-9:
            assert ids[b].tolist() == bids[b].tolist()


@pytest.mark.parametrize("seed", range(6))
def test_dense_bruteforce_u8_exact(seed):
    rng = np.random.default_rng(100 + seed)
    V, N, B, k = 40, int(rng.integers(1, 50)), 4, 60
    docs = random_csr(rng, N, V, 10, np.uint8)
    qs = random_csr(rng, B, V, 8, np.uint8)
    S = dense(qs, V, np.int64) @ dense(docs, V, np.int64).T
    ids, sc, al = run(docs, qs, V, k, all_scores=True)
    assert np.array_equal(al, S)
    eids, esc = brute_topk(S.astype(np.int32), k)   # includes k > N padding (-1, INT32_MIN)
    assert np.array_equal(ids, eids)
    assert np.array_equal(sc, esc)


# ---------------------------------------------------------------- library routine: scipy.sparse
@pytest.mark.parametrize("mode", ["f32", "u8"])
def test_scipy_spmm_config1(mode):
    w = wl.make_workload("tiny")          # BASELINE.json configs[0]: N=10,000, B=16, k=10
    docs, qs = (w.docs, w.queries) if mode == "f32" else (w.docs.to_u8(), w.queries.to_u8())
    dt = np.float64 if mode == "f32" else np.int64
    D = sp.csr_matrix((docs.weights.astype(dt), docs.terms, docs.indptr), shape=(docs.rows, w.vocab))
    Q = sp.csr_matrix((qs.weights.astype(dt), qs.terms, qs.indptr), shape=(qs.rows, w.vocab))
    S = np.asarray((Q @ D.T).todense())
    ids, sc, al = run(docs, qs, w.vocab, 10, all_scores=True)
    if mode == "u8":
        assert np.array_equal(al, S)
        order = np.lexsort((np.arange(docs.rows)[None, :].repeat(qs.rows, 0), -S), axis=1)[:, :10]
        assert np.array_equal(ids, order.astype(np.int32))
    else:
        np.testing.assert_allclose(al, S, rtol=1e-13, atol=1e-13)
        for b in range(qs.rows):     # top-10 set equals scipy's up to near-ties
            top = np.argsort(-S[b], kind="stable")[:10]
            gap = S[b, top[-1]] - np.sort(S[b])[::-1][10]
            if gap > 1e-9:
                assert set(ids[b].tolist()) == set(top.tolist())
    assert np.all(np.diff(sc.astype(np.float64), axis=1) <= 0)


# ---------------------------------------------------------------- one-hot query == column of D
def test_one_hot_query_returns_posting_list():
    rng = np.random.default_rng(7)
    V, N = 64, 300
    docs = random_csr(rng, N, V, 10, np.float32)
    D = dense(docs, V, np.float64)
    for t in (0, 5, 63):
        q = wl.Csr(np.array([0, 1], np.int64), np.array([t], np.int32), np.array([1.0], np.float32))
        _, _, al = run(docs, q, V, 3, all_scores=True)
        assert np.array_equal(al[0], D[:, t])       # exactly the posting list of t, zero elsewhere


# ---------------------------------------------------------------- closed-form ties
@pytest.mark.parametrize("N,k", [(10, 10), (1000, 37), (4099, 1000)])
def test_closed_form_ties_f32(N, k):
    # every doc has the single term 0 with weight floor(d/2); query {0:1} -> score floor(d/2):
    # ranking is N-1, N-2 ... with each tied pair ordered lower id first.
    docs = wl.Csr(np.arange(N + 1, dtype=np.int64), np.zeros(N, np.int32), (np.arange(N) // 2).astype(np.float32))
    q = wl.Csr(np.array([0, 1], np.int64), np.array([0], np.int32), np.array([1.0], np.float32))
    ids, sc = run(docs, q, 4, k)
    exp = sorted(range(N), key=lambda d: (-(d // 2), d))[:k]
    assert ids[0].tolist() == exp
    assert sc[0].tolist() == [float(d // 2) for d in exp]


def test_closed_form_ties_u8():
    N, k = 5000, 1000
    docs = wl.Csr(np.arange(N + 1, dtype=np.int64), np.zeros(N, np.int32), ((np.arange(N) % 7) + 1).astype(np.uint8))
    q = wl.Csr(np.array([0, 1], np.int64), np.array([0], np.int32), np.array([3], np.uint8))
    ids, sc = run(docs, q, 2, k)
    exp = sorted(range(N), key=lambda d: (-((d % 7) + 1), d))[:k]
    assert ids[0].tolist() == exp
    assert sc[0].tolist() == [3 * ((d % 7) + 1) for d in exp]


def test_empty_query_and_k_gt_n():
    docs = csr_from_dicts([{"1": 1.0}, {"2": 2.0}], np.float32)
    q = csr_from_dicts([{}], np.float32)
    ids, sc = run(docs, q, 4, 4)
    assert ids.tolist() == [[0, 1, -1, -1]]
    assert sc[0, :2].tolist() == [0.0, 0.0] and np.all(np.isneginf(sc[0, 2:]))


# ---------------------------------------------------------------- invariants of the definition
@pytest.fixture(scope="module")
def small():
    w = wl.make_workload("tiny", n_docs=1500, n_queries=6)
    return w


def test_term_order_symmetry(small):
    rng = np.random.default_rng(3)
    V = small.vocab

    def shuffle(c):
        t, w = c.terms.copy(), c.weights.copy()
        for r in range(c.rows):
            a, b = int(c.indptr[r]), int(c.indptr[r + 1])
            p = rng.permutation(b - a)
            t[a:b], w[a:b] = t[a:b][p], w[a:b][p]
        return wl.Csr(c.indptr, t, w)

    a = run(small.docs, small.queries, V, 20, all_scores=True)
    b = run(shuffle(small.docs), shuffle(small.queries), V, 20, all_scores=True)
    assert all(np.array_equal(x, y) for x, y in zip(a, b))     # the oracle sorts rows first: bit-identical
    au = run(small.docs.to_u8(), small.queries.to_u8(), V, 20)
    bu = run(shuffle(small.docs).to_u8(), shuffle(small.queries).to_u8(), V, 20)
    assert all(np.array_equal(x, y) for x, y in zip(au, bu))


def test_batch_independence_and_prefix(small):
    V = small.vocab
    ids, sc = run(small.docs, small.queries, V, 50)
    for b in (0, 3, 5):
        i1, s1 = run(small.docs, small.queries.slice_rows(b, b + 1), V, 50)
        assert np.array_equal(i1[0], ids[b]) and np.array_equal(s1[0], sc[b])
    i10, s10 = run(small.docs, small.queries, V, 10)
    assert np.array_equal(i10, ids[:, :10]) and np.array_equal(s10, sc[:, :10])   # top-k1 is a prefix of top-k2
    for b in range(ids.shape[0]):
        assert len(set(ids[b].tolist())) == 50
        assert all((sc[b, i] > sc[b, i + 1]) or (sc[b, i] == sc[b, i + 1] and ids[b, i] < ids[b, i + 1])
                   for i in range(49))


def test_power_of_two_scaling(small):
    V = small.vocab
    ids, sc = run(small.docs, small.queries, V, 30)
    q2 = wl.Csr(small.queries.indptr, small.queries.terms, small.queries.weights * np.float32(4.0))
    ids2, sc2 = run(small.docs, q2, V, 30)
    assert np.array_equal(ids, ids2) and np.array_equal(sc * 4.0, sc2)


def test_role_swap_symmetry(small):
    V = small.vocab
    d = small.docs.slice_rows(0, 40)
    _, _, a = run(d, small.queries, V, 1, all_scores=True)
    _, _, b = run(small.queries, d, V, 1, all_scores=True)
    assert np.array_equal(a, b.T)
    qr, dr = oracle.as_rows(small.queries, V), oracle.as_rows(d, V)
    pb, pd = np.array([0, 2, 5, 5]), np.array([0, 7, 39, 1])
    assert np.array_equal(oracle.score_pairs(qr, dr, pb, pd), a[pb, pd])


def test_disjoint_rows_score_exactly_zero():
    docs = csr_from_dicts([{"0": 1.5, "2": 2.5}, {"4": 1.0}], np.float32)
    q = csr_from_dicts([{"1": 3.0, "3": 1.0, "5": 7.0}], np.float32)
    _, _, al = run(docs, q, 6, 1, all_scores=True)
    assert al.tolist() == [[0.0, 0.0]]


def test_rejects_bad_rows():
    ok = csr_from_dicts([{"0": 1.0}], np.float32)
    dup = wl.Csr(np.array([0, 2], np.int64), np.array([3, 3], np.int32), np.array([1, 1], np.float32))
    oor = wl.Csr(np.array([0, 1], np.int64), np.array([9], np.int32), np.array([1], np.float32))
    with pytest.raises(oracle.OracleError) as e:
        run(dup, ok, 8, 1)
    assert e.value.code == 3
    with pytest.raises(oracle.OracleError) as e:
        run(ok, oor, 8, 1)
    assert e.value.code == 2
    with pytest.raises(oracle.OracleError):
        run(ok, ok, 8, 0)


def test_u8_fits_int32_bound():
    # worst case of any BASELINE config: min(nnz_q, nnz_d) * 255^2 <= 256 * 65025 < 2^31
    n = 256
    docs = wl.Csr(np.array([0, n], np.int64), np.arange(n, dtype=np.int32), np.full(n, 255, np.uint8))
    ids, sc = run(docs, docs, 300, 1)
    assert sc.tolist() == [[n * 255 * 255]]
