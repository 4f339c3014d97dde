"""Measures both scoring paths over a grid of (collection size, batch size, query length) on the current GPU — the data the
constants of ``gs_dispatch_model`` (GS_ALGO_AUTO) were fitted to.

    python -m paper_2606_26441_b200.tune_dispatch [out.csv]

Writes one CSV row per grid point: n_docs, doc_nnz, B, q_nnz, term_ms, doc_ms, winner (median of 7 searches after 3 warm-up
searches, CUDA events, k = 10, fp32).  ``profiles/r02_dispatch_sweep.csv`` is the B200 run the shipped constants come from.
"""
from __future__ import annotations

import csv
import sys

import numpy as np


def main(out_path: str) -> None:
    import torch

    from . import binding as gs
    from . import workload as wl

    d = torch.device("cuda:0")

    def dev(c):
        return [torch.from_numpy(np.ascontiguousarray(a)).to(d) for a in (c.indptr, c.terms, c.weights)]

    def timeit(ix, q, algo):
        qd = dev(q)
        for _ in range(3):
            ix.search(*qd, 10, algo=algo)
        torch.cuda.synchronize()
        ts = []
        for _ in range(7):
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record()
            ix.search(*qd, 10, algo=algo)
            b.record()
            torch.cuda.synchronize()
            ts.append(a.elapsed_time(b))
        return float(np.median(ts))

    rows = []
    for n_docs, doc_mu in [(20000, 120), (100000, 120), (1000000, 120), (100000, 20)]:
        docs = wl.make_rows(n_docs, seed=0, stream=wl.STREAM_DOCS, mu=doc_mu, sigma=doc_mu / 3, lo=max(2, doc_mu // 6), hi=doc_mu * 4)
        ix = gs.Index.from_numpy(docs, wl.VOCAB)
        for B in (1, 16, 64, 256):
            for qn in (25, 200, 1000, 4000):
                q = wl.make_rows(B, seed=0, stream=wl.STREAM_QUERIES, mu=qn, sigma=0.0, lo=qn, hi=qn)
                t, dd = timeit(ix, q, "term"), timeit(ix, q, "doc")
                rows.append([n_docs, doc_mu, B, qn, round(t, 4), round(dd, 4), "term" if t <= dd else "doc"])
                print(rows[-1], flush=True)
        ix.close()
    with open(out_path, "w", newline="") as f:
        w = csv.writer(f)
        w.writerow(["n_docs", "doc_nnz", "B", "q_nnz", "term_ms", "doc_ms", "winner"])
        w.writerows(rows)


if __name__ == "__main__":
    main(sys.argv[1] if len(sys.argv) > 1 else "dispatch_sweep.csv")
