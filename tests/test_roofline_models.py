"""The byte-accounting conventions of paper_2606_26441_b200/roofline.py against the numbers the paper prints
(tests/golden/paper_byte_models.json: PAPER.md L172-181 and Table 7).  CPU only."""
import json
import os

import numpy as np
import pytest

from paper_2606_26441_b200 import roofline as rf

G = json.load(open(os.path.join(os.path.dirname(__file__), "golden", "paper_byte_models.json")))


def test_paper_scatter_model():
    assert abs(rf.paper_scatter_entries_per_query(G["q_bar"], G["L_bar"]) - G["scatter_entries_per_query"]) <= G["scatter_entries_tol"]
    gb = rf.paper_scatter_bytes(G["B"], G["q_bar"], G["L_bar"]) / 1e9
    assert abs(gb - G["scatter_bytes_GB"]) <= G["scatter_bytes_tol_GB"]
    gbps = rf.effective_gbps(rf.paper_scatter_bytes(G["B"], G["q_bar"], G["L_bar"]), G["scatter_ms"])
    assert abs(gbps - G["scatter_GBps"]) <= G["scatter_GBps_tol"]
    assert abs(100 * gbps / G["h100_peak_GBps"] - G["scatter_pct"]) <= G["scatter_pct_tol"]


def test_paper_doc_parallel_model():
    assert rf.paper_doc_entries_per_query(G["N"], G["k_bar_model"]) == G["doc_entries_per_query"]
    b = rf.paper_doc_bytes(G["B"], G["N"], G["k_bar_measured"])
    assert abs(b / 1e9 - G["doc_bytes_GB"]) <= G["doc_bytes_tol_GB"]
    gbps = rf.effective_gbps(b, G["doc_ms"])
    assert abs(gbps - G["doc_GBps"]) <= G["doc_GBps_tol"]
    assert abs(100 * gbps / G["h100_peak_GBps"] - G["doc_pct"]) <= G["doc_pct_tol"]
    ratio = rf.paper_doc_entries_per_query(G["N"], G["k_bar_model"]) / rf.paper_scatter_entries_per_query(G["q_bar"], G["L_bar"])
    assert abs(ratio - G["work_ratio"]) <= G["work_ratio_tol"]


def test_our_models_closed_forms():
    L = np.array([10, 0, 7, 3], np.int64)
    q_terms = np.array([0, 2, 2, 3, 9, -1], np.int32)           # out-of-range ids contribute nothing
    st = rf.batch_term_stats(L, q_terms)
    assert st == {"U": 20, "W": 27, "distinct_terms": 3}
    assert rf.term_parallel_bytes(20, "f32") == 160 and rf.term_parallel_bytes(20, "u8") == 100
    # 70 documents = 3 blocks of 32 -> 4 row pointers; 128 slots (postings + block padding)
    assert rf.forward_index_bytes(70, 128, "f32") == 8 * 4 + 8 * 128
    assert rf.forward_index_bytes(70, 128, "u8") == 8 * 4 + 5 * 128
    assert rf.forward_index_bytes(64, 0, "f32") == 8 * 3 and rf.forward_index_bytes(65, 0, "f32") == 8 * 4
    assert rf.doc_parallel_bytes(70, 128, "f32", B=500, query_tile=16) == 32 * (32 + 1024)
    assert rf.doc_parallel_bytes(70, 128, "f32", B=1, query_tile=16, sample_share=0.5) == 1.5 * 1056
    # hybrid forward index: tail slots + strips read by the pass (4 B or 1 B per doc each)
    assert rf.forward_index_bytes(3, 5, "f32", strips=2) == 16 + 40 + 24
    assert rf.forward_index_bytes(3, 5, "u8", strips=2) == 16 + 25 + 6
    indptr = np.array([0, 2, 3, 6], np.int64)
    terms = np.array([5, 1, 9, 1, 2, 7], np.int32)
    assert rf.strips_per_pass(indptr, terms, np.array([1, 2, 3]), query_tile=2) == [1, 2]
    assert rf.doc_parallel_bytes(3, 5, "f32", B=3, query_tile=2, strips_by_pass=[1, 2]) == (16 + 40 + 12) + (16 + 40 + 24)


def test_term_parallel_shared_memory_roof():
    assert rf.smem_peak_gbs(1965.0) == pytest.approx(148 * 128 * 1.965e9 / 1e9)
    L = np.array([10, 0, 7, 3], np.int64)
    q_terms = np.array([0, 2, 2, 3, 9, -1], np.int32)
    ht = rf.head_tail_work(L, q_terms, np.array([0, 3]))
    assert ht == {"W_head": 13, "W_tail": 14}                    # head: terms 0 and 3 once each; tail: term 2 twice
    assert ht["W_head"] + ht["W_tail"] == rf.batch_term_stats(L, q_terms)["W"]
    assert rf.term_parallel_smem_bytes(13, 14, cell_rows=6, tile_docs=512) == 4 * 13 + 8 * 14 + 8 * 6 * 512
    assert rf.term_parallel_smem_bytes(13, 14, 6, 512, sample_share=0.5) == 1.5 * (4 * 13 + 8 * 14 + 8 * 6 * 512)
