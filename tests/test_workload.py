"""The seeded input generator: determinism, structure and the distributions BASELINE.json fixes."""
import numpy as np

from paper_2606_26441_b200 import workload as wl


def test_deterministic_and_prefix_property():
    a = wl.make_docs("paper", n_docs=3000)
    b = wl.make_docs("paper", n_docs=3000, nthreads=1)
    assert np.array_equal(a.indptr, b.indptr) and np.array_equal(a.terms, b.terms) and np.array_equal(a.weights, b.weights)
    c = wl.make_docs("mid", n_docs=500)          # same Zipf exponent: a prefix of the same collection
    assert np.array_equal(c.terms, a.terms[: c.nnz]) and np.array_equal(c.weights, a.weights[: c.nnz])
    d = wl.make_docs("paper", n_docs=100, row0=2900)
    assert np.array_equal(d.terms, a.terms[a.indptr[2900]:])
    assert wl.checksum(a.terms) == wl.checksum(b.terms) != wl.checksum(a.weights)
    assert not np.array_equal(wl.make_docs("paper", n_docs=50, seed=1).terms[:50], a.terms[:50])


def test_rows_are_valid_sparse_vectors():
    w = wl.make_workload("tiny", n_docs=4000)
    for c, lo, hi in ((w.docs, 20, 400), (w.queries, 5, 64)):
        n = np.diff(c.indptr)
        assert n.min() >= lo and n.max() <= hi
        assert c.terms.min() >= 0 and c.terms.max() < wl.VOCAB
        for r in range(0, c.rows, max(1, c.rows // 64)):
            t, _ = c.row(r)
            assert len(set(t.tolist())) == len(t)          # sampled WITHOUT replacement
        assert np.all(np.isfinite(c.weights)) and c.weights.min() > 0


def test_distributions_match_baseline_configs():
    d = wl.make_docs("paper", n_docs=60000)
    n = np.diff(d.indptr)
    assert abs(n.mean() - 120) < 1.0 and abs(n.std() - 40) < 1.5
    lw = np.log(d.weights.astype(np.float64))
    assert abs(lw.mean()) < 0.005 and abs(lw.std() - 0.5) < 0.005      # LogNormal(0, 0.5)
    cnt = np.bincount(d.terms, minlength=wl.VOCAB) / d.rows
    assert cnt[0] > 0.999 and np.all(np.diff(cnt[:6]) <= 0.01)         # term id 0 is rank 1 (hottest)
    assert 5 <= (cnt > 0.9).sum() <= 11 and 22 <= (cnt > 0.5).sum() <= 34   # Zipf(1.1) head
    q = wl.make_queries("paper")
    nq = np.diff(q.indptr)
    assert q.rows == 500 and abs(nq.mean() - 25) < 1.5 and nq.min() >= 5 and nq.max() <= 64
    q5 = wl.make_queries("skew_b32")
    n5 = np.diff(q5.indptr)
    assert q5.rows == 32 and n5.min() >= 5 and n5.max() <= 256 and n5.max() > 64
    d5 = wl.make_docs("skew_b1", n_docs=20000)
    c5 = np.bincount(d5.terms, minlength=wl.VOCAB) / d5.rows
    assert (c5 > 0.9).sum() > (cnt > 0.9).sum()                          # Zipf(1.3): longer head lists


def test_u8_quantisation_rule():
    w = np.array([0.0, 0.004, 0.005, 0.015, 0.025, 1.0, 1.005, 2.549, 2.551, 3.0, 100.0], np.float32)
    q = wl.quantize_u8(w)
    # clamp(round-half-even(100*w), 1, 255); 100*float32(0.005) is just below/above .5 as float -> use exact halves too
    assert q.tolist()[0] == 1 and q.tolist()[5] == 100 and q.tolist()[-1] == 255 and q.tolist()[-2] == 255
    assert wl.quantize_u8(np.array([0.125, 0.375], np.float32)).tolist() == [12, 38]   # 12.5 -> 12, 37.5 -> 38
    d = wl.make_docs("paper_u8", n_docs=2000)
    assert d.weights.dtype == np.uint8 and d.weights.min() >= 1
    f = wl.make_docs("paper", n_docs=2000)
    assert np.array_equal(d.terms, f.terms)
    assert np.array_equal(d.weights, np.clip(np.rint(100.0 * f.weights.astype(np.float64)), 1, 255).astype(np.uint8))
