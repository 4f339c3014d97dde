#!/usr/bin/env python
"""Writes the paper-scale golden top-k lists used by tests/test_gpu_golden.py.

    python tests/golden/make_paper_golden.py [--only paper_f32,paper_u8,skew_f32,skew_u8] [--threads T]

Calls ONLY `oracle/` (exhaustive merge scoring + full sort: Eq. 4, top-k over all N
documents L61/L125, ties by lower doc id) on inputs from the seeded generator
(`paper_2606_26441_b200.workload`, no method arithmetic).  Nothing here touches the CUDA path.

Output, one compressed .npz per case under tests/golden/ (last pin row: "cached as a golden file
keyed by generator checksum"):

    paper_topk_f32.npz  BASELINE.json configs[2]: 8.8M docs (Zipf 1.1), all 500 queries, k=1000 -> ids int32, scores float64
    paper_topk_u8.npz   configs[3]: the uint8 twin, all 500 queries, k=10                    -> ids int32, scores int32
    skew_topk_f32.npz   configs[4]: 8.8M docs with Zipf 1.3 term ids, 64 queries (5..256 terms), k=10
    skew_topk_u8.npz    the uint8 twin of configs[4]

Each file also stores the 64-bit generator checksums of the document and query arrays it was computed from; the test
regenerates the inputs, compares the checksums and only then compares the results.  Cost: about 6 core-seconds per
query at 8.8M docs (config 2/3), more for the long queries of config 4.
"""
import argparse
import os
import sys
import time

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import oracle                                          # noqa: E402
from paper_2606_26441_b200 import workload as wl      # noqa: E402

# case -> (docs config, queries config, number of queries, k, uint8?)
CASES = {
    "paper_f32": ("paper", "paper", 500, 1000, False),
    "paper_u8": ("paper", "paper", 500, 10, True),
    "skew_f32": ("skew_b32", "skew_b32", 64, 10, False),
    "skew_u8": ("skew_b32", "skew_b32", 64, 10, True),
}
FILES = {"paper_f32": "paper_topk_f32.npz", "paper_u8": "paper_topk_u8.npz", "skew_f32": "skew_topk_f32.npz",
         "skew_u8": "skew_topk_u8.npz"}


def checksums(docs, queries):
    return np.array([wl.checksum(docs.indptr), wl.checksum(docs.terms), wl.checksum(docs.weights),
                     wl.checksum(queries.indptr), wl.checksum(queries.terms), wl.checksum(queries.weights)], dtype=np.uint64)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--only", default=",".join(CASES))
    ap.add_argument("--threads", type=int, default=0)
    ap.add_argument("--docs", type=int, default=None, help="debug: first N docs only (the file name gets a suffix)")
    args = ap.parse_args()
    cache = {}
    for case in [c for c in args.only.split(",") if c]:
        dcfg, qcfg, nq, k, u8 = CASES[case]
        t0 = time.perf_counter()
        if dcfg not in cache:
            cache.clear()
            cache[dcfg] = wl.make_docs(dcfg, n_docs=args.docs)
        docs = cache[dcfg]
        queries = wl.make_queries(qcfg, n_queries=nq)
        if u8:
            docs, queries = docs.to_u8(), queries.to_u8()
        R_d, R_q = oracle.as_rows(docs, wl.VOCAB), oracle.as_rows(queries, wl.VOCAB)
        t1 = time.perf_counter()
        ids, sc = oracle.search(R_q, R_d, k, nthreads=args.threads)
        t2 = time.perf_counter()
        name = FILES[case] if args.docs is None else FILES[case].replace(".npz", f"_first{args.docs}.npz")
        np.savez_compressed(os.path.join(HERE, name), ids=ids, scores=sc, checksums=checksums(docs, queries),
                            n_docs=np.int64(docs.rows), k=np.int64(k), vocab=np.int64(wl.VOCAB))
        print(f"{case}: {docs.rows} docs x {nq} queries, k={k}: generate+canonicalise {t1 - t0:.1f} s, oracle {t2 - t1:.1f} s "
              f"({oracle.max_threads()} threads) -> {name}", flush=True)
        del R_d, R_q


if __name__ == "__main__":
    main()
