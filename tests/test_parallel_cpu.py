"""world_size-2 gloo test of the replicas-only plumbing (paper_2606_21238_b200.parallel) on CPU."""
import os
import socket

import numpy as np
import pytest

torch = pytest.importorskip("torch")
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2606_21238_b200 import parallel as P
from paper_2606_21238_b200 import workloads as W


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, q):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    # each replica serves its own seeded trace: different seeds, deterministic per rank
    tr = W.make_trace(1, seed=P.replica_seed(0, rank), scale=0.02)
    n_acc = n_tok = n_req = 0
    for tokens, offsets in tr.steps():
        n_acc += int((np.diff(offsets) // 16).sum())
        n_tok += len(tokens)
        n_req += len(offsets) - 1
    P.barrier(dist)
    out = P.reduce_timing(dist, torch, 10.0 * (rank + 1), n_acc, n_tok, n_req)
    agg = P.aggregate_counters(dist, torch, {"accesses": n_acc, "requests": n_req})
    assert agg["accesses"] == out[1] and agg["requests"] == out[3]
    q.put((rank, (n_acc, n_tok, n_req), out))
    dist.destroy_process_group()


def test_replicas_reduce_world2():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    got = sorted(q.get(timeout=120) for _ in range(2))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    (r0, mine0, out0), (r1, mine1, out1) = got
    assert out0 == out1                                        # every rank sees the same reduction
    assert out0[0] == 20.0                                     # max over ranks of the time
    assert out0[1:] == tuple(a + b for a, b in zip(mine0, mine1))   # sums of the units
    assert mine0 != mine1                                      # the replicas really serve different traces


def test_single_process_passthrough_and_routing():
    assert P.reduce_timing(None, torch, 3.5, 1, 2, 3) == (3.5, 1, 2, 3)
    assert P.replica_seed(7, 0) == 7 and P.replica_seed(7, 1) != 7
    keys = np.random.default_rng(0).integers(2, 2**63, size=10000, dtype=np.uint64)
    dst = P.route_requests(keys, 8)
    assert dst.min() >= 0 and dst.max() < 8
    assert np.array_equal(dst, P.route_requests(keys, 8))      # deterministic: same prefix -> same replica
    assert np.bincount(dst, minlength=8).min() > 1000          # and roughly balanced


def test_split_batch_partitions_the_requests():
    rng = np.random.default_rng(1)
    lens = rng.integers(0, 90, size=40)
    offsets = np.concatenate([[0], np.cumsum(lens)]).astype(np.int64)
    dst = rng.integers(0, 3, size=40)
    seen = []
    for s in range(3):
        idx, sub, slices = P.split_batch(offsets, dst, s)
        assert np.array_equal(np.diff(sub), lens[idx]) and len(slices) == len(idx)
        assert all(b - a == lens[i] for (a, b), i in zip(slices, idx))
        seen += idx.tolist()
    assert sorted(seen) == list(range(40))
    starts, has = P.first_block_offsets(offsets)
    assert np.array_equal(has, lens >= 16) and np.array_equal(starts, offsets[:-1])
