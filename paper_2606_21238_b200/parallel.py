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


# ---------------------------------------------------------------------------------------------------------------------
# NEXT-4: prefix-affinity sharding.  The paper's deployment context is a router in front of per-GPU
# cache managers (collaborative caching is future work).  N shards = N independent caches;
# a request goes to the shard chosen by the key of its FIRST block, so that all requests sharing a document or a
# conversation prefix meet in the same cache.  This is a different system from one cache of N x the capacity and is not
# bit-comparable to it; each shard is bit-comparable to an oracle fed the same sub-stream.  No data-path collective.

def first_block_offsets(offsets, block_size: int = 16):
    """offsets of the sub-batch holding only the first full block of every request (empty for shorter requests)."""
    import numpy as np

    o = np.asarray(offsets, dtype=np.int64)
    has = (o[1:] - o[:-1]) >= block_size
    return o[:-1], has


def split_batch(offsets, dst, shard: int):
    """-> (indices of the requests routed to `shard`, their offsets rebased to a packed sub-batch, the token slices)."""
    import numpy as np

    o = np.asarray(offsets, dtype=np.int64)
    idx = np.flatnonzero(np.asarray(dst) == shard)
    lens = o[idx + 1] - o[idx]
    sub = np.zeros(len(idx) + 1, dtype=np.int64)
    sub[1:] = np.cumsum(lens)
    return idx, sub, [(int(o[i]), int(o[i + 1])) for i in idx]


class ShardedArc:
    """`world` caches with prefix-affinity routing.  With `rank` given (one process per GPU) only the local shard lives
    here and `step` serves the local share of the batch; with rank=None all shards live in this process (single-GPU
    simulation, used by the tests)."""

    def __init__(self, capacity_blocks_per_shard: int, world: int, rank=None, block_size: int = 16, policy: int = 0):
        from . import arc as A

        self._A = A
        self.world, self.rank, self.B = int(world), rank, block_size
        shards = range(self.world) if rank is None else [int(rank)]
        self.caches = {s: A.ArcCache(capacity_blocks_per_shard, block_size, policy) for s in shards}

    def route(self, tokens, offsets):
        """Destination shard of every request: by its first block's key, computed by ONE kernel on the device
        (arc_route_requests); requests without a full block go to shard 0 (they make no access anywhere).  The result comes
        back to the host (4 bytes per request) because arc_step takes its batch layout from host offsets."""
        import numpy as np

        return self._A.route_requests(tokens, np.asarray(offsets, dtype=np.int64), self.world, self.B).cpu().numpy().astype(np.int64)

    def step(self, tokens, offsets):
        """-> {shard: (request indices, StepResult)} for the shards that live in this process."""
        import torch

        dst = self.route(tokens, offsets)
        out = {}
        for s, cache in self.caches.items():
            idx, sub, slices = split_batch(offsets, dst, s)
            sub_tokens = torch.cat([tokens[a:b] for a, b in slices]) if slices else tokens[:0]
            out[s] = (idx, cache.step(sub_tokens.contiguous(), sub))
        return out

    def stats(self, dist=None, torch=None):
        """Counters summed over the local shards and, with an initialised process group, over all ranks."""
        keys = [k for k in self._A.STAT_FIELDS if k not in ("p", "capacity_blocks")]
        tot = {k: 0 for k in keys}
        for c in self.caches.values():
            st = c.stats()
            for k in keys:
                tot[k] += st[k]
        return aggregate_counters(dist, torch, tot)

    def close(self):
        for c in self.caches.values():
            c.close()


def aggregate_counters(dist, torch, counters: dict, device=None) -> dict:
    """One all-reduce (SUM) of a dict of integer counters over the ranks; a pass-through without a process group."""
    if dist is None or not dist.is_initialized():
        return dict(counters)
    if device is None:
        device = torch.device("cuda", torch.cuda.current_device()) if dist.get_backend() == "nccl" else torch.device("cpu")
    keys = sorted(counters)
    t = torch.tensor([int(counters[k]) for k in keys], dtype=torch.int64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return {k: int(v) for k, v in zip(keys, t.tolist())}
