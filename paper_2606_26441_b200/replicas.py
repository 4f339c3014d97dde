"""Host logic of the multi-GPU path: "replicas only".

BASELINE.json's north_star fixes one GPU, no sharding and no collectives: the 8.8M-document index (about
20 GB) fits one B200 many times over.  `bench.py --gpus N` therefore runs N independent replicas, one process
per GPU; every replica indexes the same collection and searches ITS OWN batch of B queries.  The only
cross-rank traffic is one scalar MAX reduction of the elapsed time, outside the timed region.
This module holds that logic (no scoring arithmetic) so that it can be tested on CPU with the gloo backend.
"""
from __future__ import annotations


def query_rows(rank: int, batch: int) -> tuple:
    """Rows [row0, row0 + batch) of the seeded query stream that replica `rank` searches (disjoint across ranks)."""
    if rank < 0 or batch < 0:
        raise ValueError("rank and batch must be non-negative")
    return rank * batch, (rank + 1) * batch


def max_over_ranks(value: float, dist=None, device=None) -> float:
    """MAX over all ranks of a host scalar (elapsed time); identity without an initialised process group."""
    if dist is None or not dist.is_available() or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(value)
    import torch
    t = torch.tensor([float(value)], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_qps(world: int, batch: int, steps: int, max_ms: float) -> float:
    """Whole-job throughput: the queries ALL replicas answered divided by the slowest replica's time."""
    return world * batch * steps / (max_ms * 1e-3)
