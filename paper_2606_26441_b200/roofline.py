"""Byte / work accounting for the roofline lines of bench.py.

Pure arithmetic on sizes — no scoring.  Two families of models:

* the PAPER's models (Table 7), kept so that our numbers can be put next to
  its "% of peak" figures with the same convention (pinned by tests/test_roofline_models.py against the
  values the paper prints):
    scatter-add      bytes = B * q_bar * L_bar * 8            (4 B doc id + 4 B score per posting touched)
    doc-parallel     bytes = B * N * k_bar * 12               (4 B term id + 4 B weight + 4 B query lookup,
                                                               forward index re-read for EVERY query)
* OUR kernels' algorithmic bytes (what the method must move at least once per launch):
    term-parallel    bytes = (4 + w) * U                      U = postings of the batch's DISTINCT terms
    doc-parallel     bytes = passes * (8*(N+1) + (4+w)*P)     passes = ceil(B / query tile): the forward
                                                               index is streamed once per query TILE
  with w = 4 (fp32 weights) or 1 (uint8 impacts).
"""
from __future__ import annotations

import math

import numpy as np


def weight_bytes(wtype: str) -> int:
    return 4 if wtype == "f32" else 1


# ---- the paper's models -----------------------------------------------------------------------------
def paper_scatter_entries_per_query(q_bar: float, L_bar: float) -> float:
    """L181: q * L posting entries touched per query."""
    return q_bar * L_bar


def paper_scatter_bytes(B: int, q_bar: float, L_bar: float) -> float:
    """L172: B * q_bar * L_bar * 8 bytes per batch."""
    return B * q_bar * L_bar * 8.0


def paper_doc_entries_per_query(N: int, k_bar: float) -> float:
    """L181: N * k forward-index entries per query."""
    return N * k_bar


def paper_doc_bytes(B: int, N: int, k_bar: float) -> float:
    """L174 / Table 7: B * N * k_bar * 12 bytes per batch."""
    return B * N * k_bar * 12.0


def effective_gbps(nbytes: float, ms: float) -> float:
    return nbytes / (ms * 1e-3) / 1e9


# ---- our kernels ------------------------------------------------------------------------------------
def batch_term_stats(list_lengths: np.ndarray, query_terms: np.ndarray) -> dict:
    """U = postings of the distinct terms of the batch, W = postings counted once per (query, term)."""
    L = np.asarray(list_lengths, dtype=np.int64)
    t = np.asarray(query_terms)
    t = t[(t >= 0) & (t < L.shape[0])]
    return {"U": int(L[np.unique(t)].sum()), "W": int(L[t].sum()), "distinct_terms": int(np.unique(t).shape[0])}


def forward_index_bytes(N: int, P: int, wtype: str) -> int:
    return 8 * (N + 1) + (4 + weight_bytes(wtype)) * P


def doc_parallel_bytes(N: int, P: int, wtype: str, B: int, query_tile: int, sample_share: float = 0.0) -> float:
    passes = math.ceil(B / max(query_tile, 1))
    return passes * forward_index_bytes(N, P, wtype) * (1.0 + sample_share)


def term_parallel_bytes(U: int, wtype: str, sample_share: float = 0.0) -> float:
    return (4 + weight_bytes(wtype)) * U * (1.0 + sample_share)
