"""N>1 path on CPU: two processes over the gloo backend (DESIGN.md §8 "replicas only").

Covers what `bench.py --gpus N` does across ranks: every rank draws its own, disjoint slice of the seeded query
stream (the slices tile the stream a single process would draw), the only collective is one MAX reduction of the
elapsed time, and the reported throughput counts the queries of all replicas over the slowest replica's time.
"""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2606_26441_b200 import replicas
from paper_2606_26441_b200 import workload as wl

WORLD = 2
BATCH = 7


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank: int, port: int, out_dir: str):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(WORLD))
    dist.init_process_group("gloo", rank=rank, world_size=WORLD)
    try:
        r0, r1 = replicas.query_rows(rank, BATCH)
        q = wl.make_queries("tiny", n_queries=BATCH, row0=r0)
        np.savez(os.path.join(out_dir, f"q{rank}.npz"), indptr=q.indptr, terms=q.terms, weights=q.weights, rows=np.array([r0, r1]))
        elapsed = 10.0 + 5.0 * rank                              # rank 1 is the slow replica
        mx = replicas.max_over_ranks(elapsed, dist, "cpu")
        qps = replicas.aggregate_qps(dist.get_world_size(), BATCH, 3, mx)
        np.save(os.path.join(out_dir, f"r{rank}.npy"), np.array([mx, qps]))
        dist.barrier()
    finally:
        dist.destroy_process_group()


def test_two_replicas_over_gloo(tmp_path):
    mp.spawn(_worker, args=(_free_port(), str(tmp_path)), nprocs=WORLD, join=True)
    whole = wl.make_queries("tiny", n_queries=WORLD * BATCH)
    seen = []
    for rank in range(WORLD):
        z = np.load(tmp_path / f"q{rank}.npz")
        r0, r1 = z["rows"]
        assert (r0, r1) == (rank * BATCH, (rank + 1) * BATCH)
        ref = whole.slice_rows(int(r0), int(r1))
        assert np.array_equal(z["indptr"], ref.indptr) and np.array_equal(z["terms"], ref.terms)
        assert np.array_equal(z["weights"], ref.weights)
        seen.append((int(r0), int(r1)))
        mx, qps = np.load(tmp_path / f"r{rank}.npy")
        assert mx == 15.0                                        # MAX over ranks, identical on every rank
        assert qps == pytest.approx(WORLD * BATCH * 3 / 15e-3)
    assert seen == [(0, BATCH), (BATCH, 2 * BATCH)]              # disjoint, contiguous


def test_single_process_is_identity():
    assert replicas.max_over_ranks(3.5) == 3.5
    assert replicas.max_over_ranks(3.5, dist) == 3.5             # no process group initialised
    assert replicas.query_rows(0, 500) == (0, 500) and replicas.query_rows(3, 500) == (1500, 2000)
    with pytest.raises(ValueError):
        replicas.query_rows(-1, 5)
    assert replicas.aggregate_qps(8, 500, 10, 40.0) == pytest.approx(8 * 500 * 10 / 0.04)
