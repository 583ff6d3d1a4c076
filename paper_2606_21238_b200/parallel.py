"""Multi-GPU plumbing: REPLICAS ONLY.

The ARC directory is one serial state machine per cache, and the paper's own architecture has "a module
that does per-GPU memory management and eviction" under a router; collaborative multi-GPU
caching is future work.  N GPUs therefore means N independent handles, one process per
GPU, each fed its own request stream.  There is no data-path collective; torch.distributed is used only
to line the ranks up (barrier) and to combine the measurement (max of the device time, sums of the units).
"""
from __future__ import annotations


def replica_seed(base_seed: int, rank: int) -> int:
    """Every replica serves its own seeded trace (rank 0 keeps the single-GPU trace)."""
    return int(base_seed) + 1000003 * int(rank)


def barrier(dist) -> None:
    if dist is not None and dist.is_initialized():
        dist.barrier()


def reduce_timing(dist, torch, ms: float, n_access: int, n_tokens: int, n_req: int, device=None):
    """-> (max over ranks of ms, sum of accesses, sum of tokens, sum of requests)."""
    if dist is None or not dist.is_initialized():
        return float(ms), int(n_access), int(n_tokens), int(n_req)
    if device is None:
        device = torch.device("cuda", torch.cuda.current_device()) if dist.get_backend() == "nccl" else torch.device("cpu")
    t = torch.tensor([float(ms)], dtype=torch.float64, device=device)
    s = torch.tensor([int(n_access), int(n_tokens), int(n_req)], dtype=torch.int64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(s, op=dist.ReduceOp.SUM)
    return float(t.item()), int(s[0].item()), int(s[1].item()), int(s[2].item())


def route_requests(first_block_keys, world: int):
    """Prefix-affinity routing helper: request -> replica by its first block's key, so
    that requests sharing a document prefix land on the same cache.  Host-side, numpy uint64 in, int64 out."""
    import numpy as np

    k = np.asarray(first_block_keys, dtype=np.uint64)
    return ((k >> np.uint64(33)) % np.uint64(max(1, world))).astype(np.int64)
