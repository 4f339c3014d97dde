"""Host logic of document sharding on CPU: two processes over gloo (§6.7).

What runs here is the part of `paper_2606_26441_b200.sharded` that is not a kernel: the doc-id ranges and the exchange
(all-gather of the per-rank [B, k] lists, rank order = shard order).  The local searches are stood in for by the
oracle on each rank's shard (test infrastructure: there is no GPU here), and the merge by a few lines of numpy below;
the merged lists must equal the oracle's search of the whole collection.  The CUDA merge itself (gs_merge_topk) is
checked against the oracle in tests/test_gpu_sharded.py.
"""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

import oracle
from paper_2606_26441_b200 import sharded
from paper_2606_26441_b200 import workload as wl

WORLD, N_DOCS, B, K = 2, 1501, 6, 20


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank: int, port: int, out_dir: str):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(WORLD))
    dist.init_process_group("gloo", rank=rank, world_size=WORLD)
    try:
        docs = wl.make_docs("tiny", n_docs=N_DOCS).to_u8()
        queries = wl.make_queries("tiny", n_queries=B).to_u8()
        ranges = sharded.shard_ranges(N_DOCS, dist.get_world_size())
        lo, hi = ranges[rank]
        ids, sc = oracle.search(oracle.as_rows(queries, wl.VOCAB), oracle.as_rows(docs.slice_rows(lo, hi), wl.VOCAB), K)
        all_ids, all_sc = sharded.gather_lists(torch.from_numpy(ids.astype(np.int32)), torch.from_numpy(sc.astype(np.int32)), dist)
        np.savez(os.path.join(out_dir, f"g{rank}.npz"), ids=all_ids.numpy(), sc=all_sc.numpy(), ranges=np.array(ranges))
        dist.barrier()
    finally:
        dist.destroy_process_group()


def _merge(all_ids, all_sc, bases, k):
    out_i, out_s = [], []
    for b in range(all_ids.shape[1]):
        pairs = [(-int(all_sc[l, b, j]), int(all_ids[l, b, j]) + bases[l])
                 for l in range(all_ids.shape[0]) for j in range(all_ids.shape[2]) if all_ids[l, b, j] >= 0]
        pairs.sort()
        out_i.append([p[1] for p in pairs[:k]])
        out_s.append([-p[0] for p in pairs[:k]])
    return np.array(out_i), np.array(out_s)


def test_two_shards_over_gloo(tmp_path):
    mp.spawn(_worker, args=(_free_port(), str(tmp_path)), nprocs=WORLD, join=True)
    docs = wl.make_docs("tiny", n_docs=N_DOCS).to_u8()
    queries = wl.make_queries("tiny", n_queries=B).to_u8()
    o_ids, o_sc = oracle.search(oracle.as_rows(queries, wl.VOCAB), oracle.as_rows(docs, wl.VOCAB), K)
    for rank in range(WORLD):
        z = np.load(tmp_path / f"g{rank}.npz")
        assert z["ids"].shape == (WORLD, B, K) and z["ranges"].tolist() == [[0, 751], [751, 1501]]
        m_ids, m_sc = _merge(z["ids"], z["sc"], [int(r[0]) for r in z["ranges"]], K)
        assert np.array_equal(m_ids, o_ids) and np.array_equal(m_sc, o_sc)      # every rank holds the same gathered lists


def test_shard_ranges_and_single_process_gather():
    assert sharded.shard_ranges(10, 3) == [(0, 4), (4, 7), (7, 10)]
    assert sharded.shard_ranges(2, 4) == [(0, 1), (1, 2), (2, 2), (2, 2)]
    assert sharded.shard_ranges(0, 2) == [(0, 0), (0, 0)]
    r = sharded.shard_ranges(8_800_000, 8)
    assert r[0] == (0, 1_100_000) and r[-1][1] == 8_800_000 and all(a[1] == b[0] for a, b in zip(r, r[1:]))
    with pytest.raises(ValueError):
        sharded.shard_ranges(5, 0)
    ids, sc = torch.zeros((3, 4), dtype=torch.int32), torch.ones((3, 4))
    a, s = sharded.gather_lists(ids, sc)                                         # no process group: one list
    assert a.shape == (1, 3, 4) and s.shape == (1, 3, 4)
