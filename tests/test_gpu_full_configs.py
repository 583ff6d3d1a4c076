"""Parity at BASELINE.json's full sizes, in the launch configuration bench.py times (default K3 machine, buffers
reserved, steps enqueued on the current stream): every output array of every step against the oracle, then the
counters and the four lists.  Configs 2 and 3 run their whole trace; 4 and 5 a prefix of it (their full traces are
160 M and 600 M accesses; the prefix still fills the cache, evicts, adapts p and exercises the maintenance kernels)."""
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


@pytest.mark.parametrize("config,max_steps,policy", [(2, None, 0), (2, 300, 1), (2, None, 2), (3, None, 0), (3, 400, 2), (4, 500, 0), (4, 60, 1), (5, 120, 0)])
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
