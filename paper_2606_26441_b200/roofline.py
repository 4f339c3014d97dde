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
    doc-parallel     bytes = sum over passes of 8*(N+1) + (4+w)*P_tail + w*N*h_pass
                                                               passes = ceil(B / query tile): the forward index is
                                                               streamed once per query TILE; it is a hybrid of a CSR
                                                               holding the P_tail postings without a dense strip and
                                                               of H strips (w bytes per doc each), of which a pass
                                                               reads the h_pass ones some query of its tile uses
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


def forward_index_bytes(N: int, P_tail: int, wtype: str, strips: int = 0) -> int:
    """One pass over the hybrid forward index: one row pointer per block of 32 documents + the tail block CSR
    (`P_tail` slots: postings plus the padding of every block to 128) + `strips` dense strips of N entries."""
    w = weight_bytes(wtype)
    return 8 * ((N + 31) // 32 + 1) + (4 + w) * P_tail + w * N * strips


def strips_per_pass(query_indptr: np.ndarray, query_terms: np.ndarray, head_terms: np.ndarray, query_tile: int) -> list:
    """For every pass (tile of `query_tile` consecutive queries): how many strip terms its queries contain."""
    indptr = np.asarray(query_indptr, dtype=np.int64)
    B = indptr.shape[0] - 1
    head = np.asarray(head_terms)
    out = []
    for a in range(0, B, max(query_tile, 1)):
        b = min(B, a + query_tile)
        t = np.asarray(query_terms[indptr[a]:indptr[b]])
        out.append(int(np.intersect1d(t, head).shape[0]))
    return out


def doc_parallel_bytes(N: int, P_tail: int, wtype: str, B: int, query_tile: int, sample_share: float = 0.0,
                       strips_by_pass=None) -> float:
    passes = math.ceil(B / max(query_tile, 1))
    if strips_by_pass is None:
        strips_by_pass = [0] * passes
    assert len(strips_by_pass) == passes
    return sum(forward_index_bytes(N, P_tail, wtype, h) for h in strips_by_pass) * (1.0 + sample_share)


def term_parallel_bytes(U: int, wtype: str, sample_share: float = 0.0) -> float:
    return (4 + weight_bytes(wtype)) * U * (1.0 + sample_share)


# ---- term-parallel kernel: the shared-memory roof ----------------------------------------------------
# The term-parallel kernel is not HBM bound by construction (it reads each posting of the batch's terms from
# HBM/L2 and then does one shared-memory access or read-modify-write per multiply-add): its roof is the
# shared-memory pipeline.  SM counts and clocks: /opt/skills/guides/B200_PROFILING.md (148 SMs, 1965 MHz);
# 32 banks x 4 bytes per SM per clock is the architectural shared-memory width.
B200_SMS = 148
SMEM_BYTES_PER_CLK_PER_SM = 128


def smem_peak_gbs(sm_mhz: float = 1965.0, sms: int = B200_SMS) -> float:
    """Shared-memory bandwidth of the chip in GB/s: SMs x 128 B/clk x clock (37 226 GB/s at 1965 MHz)."""
    return sms * SMEM_BYTES_PER_CLK_PER_SM * sm_mhz * 1e6 / 1e9


def head_tail_work(list_lengths: np.ndarray, query_terms: np.ndarray, head_terms: np.ndarray) -> dict:
    """Useful multiply-adds of a batch split into head (dense-strip) terms and tail (scattered) terms."""
    L = np.asarray(list_lengths, dtype=np.int64)
    t = np.asarray(query_terms)
    t = t[(t >= 0) & (t < L.shape[0])]
    is_head = np.zeros(L.shape[0], dtype=bool)
    is_head[np.asarray(head_terms, dtype=np.int64)] = True
    return {"W_head": int(L[t[is_head[t]]].sum()), "W_tail": int(L[t[~is_head[t]]].sum())}


def term_parallel_smem_bytes(W_head: int, W_tail: int, cell_rows: int, tile_docs: int, sample_share: float = 0.0) -> float:
    """Algorithmic shared-memory traffic of the term-parallel kernel per batch:
    4 B per head multiply-add (the strip value read from the staged strip), 8 B per tail multiply-add (accumulator
    read + write), and per (doc tile, query) cell row 4*Ts to zero it and 4*Ts to read it back."""
    return (4.0 * W_head + 8.0 * W_tail + 8.0 * cell_rows * tile_docs) * (1.0 + sample_share)
