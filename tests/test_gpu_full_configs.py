"""Parity at BASELINE.json's full sizes, in the launch configuration bench.py times (default K3 machine, buffers
reserved, steps enqueued on the current stream): every output array of every step against the oracle, then the
counters and the four lists.  Configs 2 and 3 run their whole trace; 4 and 5 a prefix of it here (1,000 and 250 of 1,954 steps: 82 M and 75 M
accesses; the state machine is sequential, so the oracle cannot skip ahead and a slice is always a prefix).  Their WHOLE
traces (160 M and 600 M accesses) are compared step by step with tests/full_trace_parity.py; the logs of those runs are
in profiles/r02_full_trace_parity.md."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

from oracle import oracle as O
from paper_2606_21238_b200 import workloads as W

OUT_KEYS = ("prefix_len", "blk_off", "cls", "block_id", "evicted_id", "p_after", "alloc_ids", "evict_ids")
STAT_KEYS = ("steps", "requests", "tokens_seen", "tokens_hashed", "accesses", "hit_t1", "hit_t2", "ghost_b1", "ghost_b2",
             "miss", "evict_t1", "evict_t2", "drop_b1", "drop_b2", "fresh_ids_used", "prefix_hit_tokens", "t1", "t2",
             "b1", "b2", "p")


@pytest.mark.parametrize("config,max_steps,policy", [(2, None, 0), (2, 300, 1), (2, None, 2), (3, None, 0), (3, 400, 2), (4, 1000, 0), (4, 60, 1), (5, 250, 0)])
def test_full_size_config(config, max_steps, policy):
    if not torch.cuda.is_available():
        pytest.fail("-m gpu tests need a CUDA device")
    from paper_2606_21238_b200 import arc as A

    A.load_library()
    tr = W.make_trace(config, seed=0)
    c = tr.info.capacity_blocks
    gc, oc = A.ArcCache(c, 16, policy), O.OracleCache(c, 16, policy)
    n_steps = n_acc = 0
    for tokens, offsets in tr.steps(max_steps=max_steps):
        g = gc.step(torch.from_numpy(tokens).cuda(), offsets).to_host()
        o = oc.step(tokens, offsets)
        assert g["n_access"] == o["n_access"]
        for k in OUT_KEYS:
            assert np.array_equal(g[k], o[k]), f"config {config} policy {policy} step {n_steps}: {k} differs"
        n_steps += 1
        n_acc += o["n_access"]
    gs, os_ = gc.stats(), oc.stats()
    for k in STAT_KEYS:
        assert gs[k] == os_[k], f"config {config}: stat {k}: gpu {gs[k]} oracle {os_[k]}"
    gl, ol = gc.debug_lists(), oc.lists()
    for n in ("T1", "T2", "B1", "B2"):
        assert np.array_equal(gl[n][0], ol[n][0]) and np.array_equal(gl[n][1], ol[n][1]), f"config {config}: list {n}"
    assert n_steps > 0 and n_acc > 0
    if config in (2, 3) and max_steps is None:
        assert n_steps == tr.info.n_steps
    gc.close()


@pytest.mark.parametrize("policy", [0, 1, 2])
def test_windowed_zipf_batch1(policy):
    """The paper-shaped workload at batch size 1: 3,072 one-request steps, every output and
    the T1 ratio trajectory against the oracle."""
    from paper_2606_21238_b200 import arc as A

    c = 30000 // 16                                  # the paper's smallest cache size, 30K tokens
    tr = W.make_windowed_zipf(c, seed=0)
    gc, oc = A.ArcCache(c, 16, policy), O.OracleCache(c, 16, policy)
    n = 0
    for i, (tokens, offsets) in enumerate(tr.steps()):
        if int((np.diff(offsets) // 16).max()) > c:
            continue
        g = gc.step(torch.from_numpy(tokens).cuda(), offsets).to_host()
        o = oc.step(tokens, offsets)
        for k in OUT_KEYS:
            assert np.array_equal(g[k], o[k]), f"policy {policy} request {i}: {k}"
        if i % 64 == 0:
            gs, os_ = gc.stats(), oc.stats()
            assert (gs["t1"], gs["t2"], gs["b1"], gs["b2"], gs["p"]) == (os_["t1"], os_["t2"], os_["b1"], os_["b2"], os_["p"])
        n += 1
    assert n > 2500
    gs, os_ = gc.stats(), oc.stats()
    for k in STAT_KEYS:
        assert gs[k] == os_[k], k
    gc.close()


def test_report_tool_runs():
    from paper_2606_21238_b200 import report

    rep = report.run([30000], seed=0, policies=(0, 1), sample_every=256)
    assert len(rep["runs"]) == 2
    arc, lru = rep["runs"]
    assert arc["policy"] == "ARC" and lru["policy"] == "LRU"
    assert 0.0 < lru["block_hit_rate"] <= arc["block_hit_rate"] + 0.02 < 1.0
    assert all(0.0 <= x <= 1.0 for x in arc["t1_ratio_every_256_requests"])


def test_prefix_affinity_shards_match_per_shard_oracles():
    """NEXT-4: four shards in one process; routing by the first block's key computed on the GPU must equal the routing
    computed from the oracle's keys, and every shard must match an oracle fed the same sub-stream."""
    from paper_2606_21238_b200 import parallel as P

    world, c = 4, 48
    sh = P.ShardedArc(c, world, rank=None)
    oracles = [O.OracleCache(c, 16, 0) for _ in range(world)]
    tr = W.make_trace(1, seed=2)
    for step, (tokens, offsets) in enumerate(tr.steps(max_steps=60)):
        keys, blk_off = O.hash_blocks(tokens, offsets)
        nb = np.diff(blk_off)
        want_dst = np.zeros(len(nb), dtype=np.int64)
        want_dst[nb > 0] = P.route_requests(keys[blk_off[:-1][nb > 0]], world)
        dev_tokens = torch.from_numpy(tokens).cuda()
        assert np.array_equal(sh.route(dev_tokens, offsets), want_dst)
        res = sh.step(dev_tokens, offsets)
        for s in range(world):
            idx, sub, slices = P.split_batch(offsets, want_dst, s)
            sub_tokens = np.concatenate([tokens[a:b] for a, b in slices]) if slices else np.zeros(0, np.int32)
            o = oracles[s].step(sub_tokens, sub)
            gi, g = res[s]
            assert np.array_equal(gi, idx)
            g = g.to_host()
            for k in OUT_KEYS:
                assert np.array_equal(g[k], o[k]), f"step {step} shard {s}: {k}"
    tot = sh.stats()
    assert tot["accesses"] == sum(o.stats()["accesses"] for o in oracles)
    assert tot["hit_t1"] + tot["hit_t2"] == sum(o.stats()["hit_t1"] + o.stats()["hit_t2"] for o in oracles)
    sh.close()


def _sharded_rank_worker(rank, world, port, q):
    import os

    import torch.distributed as dist

    os.environ["MASTER_ADDR"], os.environ["MASTER_PORT"] = "127.0.0.1", str(port)
    torch.cuda.set_device(rank)
    dist.init_process_group("nccl", rank=rank, world_size=world, device_id=torch.device("cuda", rank))
    from paper_2606_21238_b200 import parallel as P

    c = 48
    sh = P.ShardedArc(c, world, rank=rank)
    oc = O.OracleCache(c, 16, 0)
    tr = W.make_trace(1, seed=2)
    ok = True
    for tokens, offsets in tr.steps(max_steps=40):
        dev_tokens = torch.from_numpy(tokens).cuda()
        dst = sh.route(dev_tokens, offsets)
        (idx, g), = sh.step(dev_tokens, offsets).values()
        _, sub, slices = P.split_batch(offsets, dst, rank)
        sub_tokens = np.concatenate([tokens[a:b] for a, b in slices]) if slices else np.zeros(0, np.int32)
        o = oc.step(sub_tokens, sub)
        g = g.to_host()
        ok = ok and all(np.array_equal(g[k], o[k]) for k in OUT_KEYS)
    tot = sh.stats(dist, torch)                               # one all-reduce over NCCL
    q.put((rank, ok, tot["accesses"], oc.stats()["accesses"]))
    sh.close()
    dist.destroy_process_group()


def test_prefix_affinity_shards_one_process_per_gpu_over_nccl():
    """NEXT-4 as it would be deployed: one process per GPU, every rank owns one shard, routing on the device, counters
    summed with one NCCL all-reduce.  Needs two GPUs; on a one-GPU box it is skipped (visibly)."""
    if torch.cuda.device_count() < 2:
        pytest.skip(f"needs >= 2 CUDA devices, this box has {torch.cuda.device_count()}: the one-process-per-GPU mode has not run on hardware")
    import socket

    import torch.multiprocessing as mp

    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_sharded_rank_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    got = sorted(q.get(timeout=300) for _ in range(2))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert all(ok for _, ok, _, _ in got)
    assert got[0][2] == got[1][2] == got[0][3] + got[1][3]    # the all-reduced total is the sum of the shards' oracles
