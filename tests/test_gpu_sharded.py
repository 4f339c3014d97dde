"""Document sharding + device-side merge (gs_merge_topk; §6.7) — `-m gpu`.

The shards of a collection are indexed and searched one after the other on ONE GPU (nothing here waits on another
rank); their [B, k] lists are merged by gs_merge_topk and the result must equal the oracle's exhaustive search of the
WHOLE collection: bit-exact in integer mode (ties across shard boundaries included), within the fp32 rules of
tests/parity.py otherwise.
"""
import numpy as np
import pytest

import oracle
from paper_2606_26441_b200 import sharded
from paper_2606_26441_b200 import workload as wl
import parity
from test_gpu_parity import compare, csr_from_dicts, dev, gs  # noqa: F401  (gs is the module fixture)

pytestmark = pytest.mark.gpu


def search_sharded(gs, docs, queries, vocab, k, ranges, **opt):
    import torch
    ids_l, sc_l = [], []
    for lo, hi in ranges:
        ix = gs.Index.from_numpy(docs.slice_rows(lo, hi), vocab)
        ids, sc = ix.search(*dev(queries), k, **opt)
        ids_l.append(ids)
        sc_l.append(sc)
        ix.close()
    ids, sc = gs.merge_topk(torch.stack(ids_l).contiguous(), torch.stack(sc_l).contiguous(), k,
                            doc_bases=[lo for lo, _ in ranges])
    return ids.cpu().numpy(), sc.cpu().numpy()


@pytest.mark.parametrize("mode", ["f32", "u8"])
@pytest.mark.parametrize("world,k", [(2, 10), (3, 100), (8, 1000)])
def test_sharded_search_equals_the_single_index(gs, mode, world, k):
    docs = wl.make_docs("mid", n_docs=30_011)
    queries = wl.make_queries("mid", n_queries=24)
    if mode == "u8":
        docs, queries = docs.to_u8(), queries.to_u8()
    ranges = sharded.shard_ranges(docs.rows, world)
    ids, sc = search_sharded(gs, docs, queries, wl.VOCAB, k, ranges, algo="term")
    compare(gs, docs, queries, wl.VOCAB, k, ids, sc)


def test_ties_across_shard_boundaries_and_short_shards(gs):
    """Closed form: every doc holds term 0 with the u8 weight (d mod 7) + 1, query = {0: 1}: the ranking is known
    analytically (score desc, lower id first), ties span all shards.  Shards of 5 docs with k = 12 return padded lists."""
    n, k = 33, 12
    docs = csr_from_dicts([{0: (d % 7) + 1} for d in range(n)], np.uint8)
    queries = csr_from_dicts([{0: 1}, {}], np.uint8)
    ranges = sharded.shard_ranges(n, 7)
    assert max(hi - lo for lo, hi in ranges) < k
    ids, sc = search_sharded(gs, docs, queries, 4, k, ranges, algo="term")
    order = sorted(range(n), key=lambda d: (-((d % 7) + 1), d))[:k]
    assert ids[0].tolist() == order and sc[0].tolist() == [(d % 7) + 1 for d in order]
    assert ids[1].tolist() == list(range(k)) and sc[1].tolist() == [0] * k          # empty query: ids 0..k-1, score 0
    compare(gs, docs, queries, 4, k, ids, sc)


def test_union_smaller_than_k_is_padded(gs):
    import torch
    d = torch.device("cuda:0")
    ids = torch.tensor([[[4, 1, -1]], [[0, -1, -1]]], dtype=torch.int32, device=d)             # 2 lists, 1 query, k_in 3
    sc = torch.tensor([[[2.0, 2.0, 0.0]], [[2.0, 0.0, 0.0]]], dtype=torch.float32, device=d)
    o_ids, o_sc = gs.merge_topk(ids, sc, 5, doc_bases=[0, 10])
    assert o_ids.cpu().tolist() == [[1, 4, 10, -1, -1]]
    assert o_sc.cpu().tolist()[0][:3] == [2.0, 2.0, 2.0] and all(np.isneginf(o_sc.cpu().numpy()[0][3:]))
    with pytest.raises(gs.GsError):
        gs.merge_topk(ids, sc, 0)


def test_sharded_index_without_a_process_group(gs):
    """ShardedIndex on one process: the 'exchange' is the identity, the merge re-bases the local ids of the rank's shard."""
    docs = wl.make_docs("tiny", n_docs=2_000)
    queries = wl.make_queries("tiny", n_queries=5)
    ranges = sharded.shard_ranges(docs.rows, 2)
    ix = gs.Index.from_numpy(docs.slice_rows(*ranges[1]), wl.VOCAB)
    si = sharded.ShardedIndex(ix, ranges, 1)
    ids, sc = si.search(*dev(queries), 10)
    l_ids, l_sc = ix.search(*dev(queries), 10)
    assert np.array_equal(ids.cpu().numpy(), l_ids.cpu().numpy() + ranges[1][0])
    assert np.array_equal(sc.cpu().numpy(), l_sc.cpu().numpy())
    ix.close()
