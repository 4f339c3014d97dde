"""Comparators between the CUDA path and the oracle (SURVEY §8c / BASELINE.json north_star).

Integer-impact mode: ids and scores must be bit-identical.
fp32 mode, tol(x) = max(1e-5*|x|, 1e-6):
  (1) structure: ids unique and in range, GPU scores non-increasing, equal adjacent scores -> ids ascend;
  (2) values   : |gpu_score - S*(b,id)| <= tol(S*) for every returned entry (S* = oracle fp64 score);
  (3) set      : every oracle top-k doc with S* > tau* + 2 tol(tau*) is returned, and every returned
                 doc has S* >= tau* - 2 tol(tau*)   (tau* = oracle k-th score);
  (4) order    : adjacent returned docs i<j have S*(id_i) >= S*(id_j) - 2 tol.
"""
import numpy as np

REL, ABS = 1e-5, 1e-6


def tol(x):
    return np.maximum(REL * np.abs(x), ABS)


def check_int_exact(g_ids, g_sc, o_ids, o_sc):
    g_ids, g_sc = np.asarray(g_ids), np.asarray(g_sc)
    assert g_ids.shape == o_ids.shape and g_sc.shape == o_sc.shape
    if not np.array_equal(g_ids, o_ids) or not np.array_equal(g_sc.astype(np.int64), o_sc.astype(np.int64)):
        bad = np.argwhere((g_ids != o_ids) | (g_sc.astype(np.int64) != o_sc.astype(np.int64)))
        b, i = bad[0]
        raise AssertionError(f"int mode mismatch at query {b} rank {i}: gpu ({g_ids[b, i]}, {g_sc[b, i]}) "
                             f"oracle ({o_ids[b, i]}, {o_sc[b, i]}); {len(bad)} mismatches")


def check_f32_row(g_ids, g_sc, o_ids, o_sc, true_of_gpu, n_docs):
    """One query.  true_of_gpu[i] = oracle fp64 score of g_ids[i]."""
    k = len(g_ids)
    n_real = min(k, n_docs)
    # padding slots (k > N)
    assert np.all(g_ids[n_real:] == -1) and np.all(np.isneginf(g_sc[n_real:]))
    gi, gs, ts = g_ids[:n_real], g_sc[:n_real].astype(np.float64), np.asarray(true_of_gpu[:n_real], np.float64)
    # (1) structure
    assert gi.min(initial=0) >= 0 and gi.max(initial=0) < n_docs, "id out of range"
    assert len(np.unique(gi)) == n_real, "duplicate ids"
    d = np.diff(g_sc[:n_real])
    assert np.all(d <= 0), "gpu scores not sorted descending"
    eq = np.nonzero(d == 0)[0]
    assert np.all(gi[eq] < gi[eq + 1]), "ties not ordered by ascending doc id"
    # (2) values
    err = np.abs(gs - ts)
    assert np.all(err <= tol(ts)), f"score error {err.max()} exceeds tolerance"
    # (3) set
    oi, os_ = o_ids[:n_real], o_sc[:n_real]
    tau = os_[-1]
    must = oi[os_ > tau + 2 * tol(tau)]
    assert np.all(np.isin(must, gi)), "a clearly-top-k document is missing"
    assert np.all(ts >= tau - 2 * tol(tau)), "a returned document is clearly below the k-th score"
    # (4) order
    assert np.all(ts[:-1] >= ts[1:] - 2 * tol(ts[1:])), "returned order contradicts true scores"
    return float((err / np.maximum(np.abs(ts), 1e-30)).max(initial=0.0)), int(n_real - np.isin(gi, oi).sum())


def check_f32(g_ids, g_sc, o_ids, o_sc, true_scores_fn, n_docs):
    """All queries.  true_scores_fn(b, ids) -> oracle fp64 scores of those docs for query b."""
    g_ids, g_sc = np.asarray(g_ids), np.asarray(g_sc)
    assert g_ids.shape == o_ids.shape
    worst, subs = 0.0, 0
    for b in range(g_ids.shape[0]):
        n_real = min(g_ids.shape[1], n_docs)
        t = true_scores_fn(b, g_ids[b, :n_real])
        w, s = check_f32_row(g_ids[b], g_sc[b], o_ids[b], o_sc[b], t, n_docs)
        worst, subs = max(worst, w), subs + s
    return worst, subs
