"""Parity of the CUDA path against the CPU oracle, bit-exact, through the C ABI (-m gpu)."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

from oracle import oracle as O
from paper_2606_21238_b200 import workloads as W

OUT_KEYS = ("prefix_len", "blk_off", "cls", "block_id", "evicted_id", "p_after", "alloc_ids", "evict_ids")
STAT_KEYS = ("steps", "requests", "tokens_seen", "tokens_hashed", "accesses", "hit_t1", "hit_t2", "ghost_b1", "ghost_b2",
             "miss", "evict_t1", "evict_t2", "drop_b1", "drop_b2", "fresh_ids_used", "prefix_hit_tokens", "t1", "t2",
             "b1", "b2", "p", "capacity_blocks", "block_size", "policy")


@pytest.fixture(scope="module")
def arc():
    if not torch.cuda.is_available():
        pytest.fail("-m gpu tests need a CUDA device")
    from paper_2606_21238_b200 import arc as A
    A.load_library()   # fails loudly if the extension is missing
    return A


def dev(tokens):
    return torch.from_numpy(np.ascontiguousarray(tokens, dtype=np.int32)).cuda()


def assert_same_step(g, o, ctx=""):
    assert g["n_access"] == o["n_access"], ctx
    for k in OUT_KEYS:
        assert np.array_equal(g[k], o[k]), f"{ctx}: {k} differs at {np.flatnonzero(np.asarray(g[k]) != np.asarray(o[k]))[:8] if len(g[k]) == len(o[k]) else (len(g[k]), len(o[k]))}"


def assert_same_state(gc, oc, ctx=""):
    gs, os_ = gc.stats(), oc.stats()
    for k in STAT_KEYS:
        assert gs[k] == os_[k], f"{ctx}: stat {k}: gpu {gs[k]} oracle {os_[k]}"
    gl, ol = gc.debug_lists(), oc.lists()
    for n in ("T1", "T2", "B1", "B2"):
        assert np.array_equal(gl[n][0], ol[n][0]), f"{ctx}: list {n} keys differ"
        assert np.array_equal(gl[n][1], ol[n][1]), f"{ctx}: list {n} block ids differ"


def run_trace(arc, steps, c, policy, machine, check_every=1, ctx=""):
    gc, oc = arc.ArcCache(c, 16, policy), O.OracleCache(c, 16, policy)
    gc.set_machine(machine)
    for i, (tokens, offsets) in enumerate(steps):
        g = gc.step(dev(tokens), offsets)
        o = oc.step(tokens, offsets)
        if i % check_every == 0:
            assert_same_step(g.to_host(), o, f"{ctx} step {i}")
    assert_same_state(gc, oc, ctx)
    gc.close()
    return oc.stats()


# ------------------------------------------------------------------------------------------- K1

def test_hash_parity_edge_requests(arc):
    rng = np.random.default_rng(0)
    lens = [0, 1, 15, 16, 17, 31, 32, 33, 47, 16 * 31, 16 * 32, 16 * 33 + 5, 16 * 2048, 16 * 2049 + 15, 0, 100]
    reqs = [rng.integers(-3, 128000, size=n).astype(np.int32) for n in lens]
    tokens, offsets = W.pack_requests(reqs)
    want, _ = O.hash_blocks(tokens, offsets)
    got = arc.hash_blocks(dev(tokens), offsets).cpu().numpy().view(np.uint64)
    assert np.array_equal(got, want)


@pytest.mark.parametrize("shift", [0, 1, 2, 3])
def test_hash_parity_misaligned_base(arc, shift):
    rng = np.random.default_rng(1)
    reqs = [rng.integers(0, 32000, size=int(n)).astype(np.int32) for n in rng.integers(1, 700, size=50)]
    tokens, offsets = W.pack_requests(reqs)
    want, _ = O.hash_blocks(tokens, offsets)
    buf = torch.zeros(len(tokens) + 8, dtype=torch.int32, device="cuda")
    buf[shift:shift + len(tokens)] = dev(tokens)
    got = arc.hash_blocks(buf[shift:], offsets).cpu().numpy().view(np.uint64)   # base pointer 4*shift bytes off 16-B alignment
    assert np.array_equal(got, want)


@pytest.mark.parametrize("config", [1, 2, 3])
def test_hash_parity_configs(arc, config):
    tr = W.make_trace(config, seed=0, scale=0.02 if config > 1 else 1.0)
    for i, (tokens, offsets) in enumerate(tr.steps(max_steps=6)):
        want, _ = O.hash_blocks(tokens, offsets)
        got = arc.hash_blocks(dev(tokens), offsets).cpu().numpy().view(np.uint64)
        assert np.array_equal(got, want), (config, i)


def test_hash_on_two_streams_and_from_device_offsets(arc):
    """arc_hash_blocks keeps no shared scratch: calls on two streams that overlap (different request mixes, many calls in
    flight, more than the scratch ring holds) all give the oracle's keys; arc_hash_blocks_device (offsets already on the
    device, the caller's ticket scratch zeroed once) gives the same keys call after call."""
    rng = np.random.default_rng(77)
    jobs = []
    for j in range(24):
        n_req = int(rng.integers(1, 3000 if j % 3 == 0 else 40))
        lens = rng.integers(0, 2000 if j % 2 else 300, size=n_req)
        reqs = [rng.integers(0, 128000, size=int(n)).astype(np.int32) for n in lens]
        tokens, offsets = W.pack_requests(reqs)
        want, blk_off = O.hash_blocks(tokens, offsets)
        jobs.append((dev(tokens), offsets, want, blk_off))
    s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
    outs = []
    for j, (t, o, want, _) in enumerate(jobs):
        outs.append(arc.hash_blocks(t, o, stream=(s1 if j % 2 else s2)))
    torch.cuda.synchronize()
    for (t, o, want, _), got in zip(jobs, outs):
        assert np.array_equal(got.cpu().numpy().view(np.uint64), want)
    ticket = torch.zeros(2, dtype=torch.int32, device="cuda")
    for rep in range(2):
        for t, o, want, blk_off in jobs[:8]:
            if len(want) == 0:
                continue
            items = arc.hash_items(o)
            out = torch.empty(len(want), dtype=torch.int64, device="cuda")
            arc.hash_blocks_device(t, torch.from_numpy(items.view(np.uint8)).cuda(), len(items), int(o[0]), int(o[-1]), out, ticket)
            assert np.array_equal(out.cpu().numpy().view(np.uint64), want)
    assert int(ticket.abs().sum()) == 0


# ------------------------------------------------------------------------------- whole arc_step

@pytest.mark.parametrize("machine", [0, 1, 2, 3, 4, 5])
@pytest.mark.parametrize("policy", [0, 1, 2])
def test_config1_full_trace(arc, policy, machine):
    """BASELINE.json configs[0]: c = 64, 2,000 requests, 8 per step, ARC and LRU, every output of every step."""
    tr = W.make_trace(1, seed=0)
    st = run_trace(arc, tr.steps(), 64, policy, machine, ctx=f"config1 policy {policy} machine {machine}")
    assert st["requests"] == 2000


@pytest.mark.parametrize("machine", [0, 1, 2, 3, 4, 5])
@pytest.mark.parametrize("config,scale,max_steps", [(2, 0.06, 40), (3, 0.03, 40), (4, 0.004, 8)])
def test_larger_configs_scaled(arc, config, scale, max_steps, machine):
    tr = W.make_trace(config, seed=0, scale=scale)
    if machine == 1 and config == 4:
        max_steps = 3
    run_trace(arc, tr.steps(max_steps=max_steps), tr.info.capacity_blocks, 0, machine, ctx=f"config{config} m{machine}")


@pytest.mark.parametrize("policy", [0, 1, 2])
def test_config2_lru_and_small_cache_pressure(arc, policy):
    """Config-2 shaped requests against a cache of 600 blocks: constant eviction, ghost churn, pin fallbacks."""
    tr = W.make_trace(2, seed=5, scale=0.01)
    reqs = [r[:16 * 500 + 7] for r in tr.requests(max_requests=300)]
    steps = [W.pack_requests(reqs[s:s + 16]) for s in range(0, len(reqs), 16)]
    run_trace(arc, steps, 600, policy, 0, ctx=f"pressure policy {policy}")


@pytest.mark.parametrize("machine", [0, 1, 2, 3, 4, 5])
@pytest.mark.parametrize("c", [1, 2, 3, 5, 8])
def test_tiny_caches_prefix_trees(arc, c, machine):
    """Adversarial micro-traces: duplicate requests inside one step, keys dropped from a ghost list and
    re-accessed in the same step, requests of exactly c blocks, empty and sub-block requests."""
    rng = np.random.default_rng(100 + c)
    for policy in (0, 1, 2):
        gc, oc = arc.ArcCache(c, 16, policy), O.OracleCache(c, 16, policy)
        gc.set_machine(machine)
        table = rng.integers(0, 1000, size=(3, 2, 16), dtype=np.int32)    # a tree that lasts: prefixes shared ACROSS steps too
        for step in range(60):
            reqs = W.prefix_tree_requests(rng, n_requests=int(rng.integers(1, 12)), block_size=16, branching=2, depth=3,
                                          max_blocks=c)
            reqs += [_tree_request(rng, table, c) for _ in range(int(rng.integers(0, 5)))]
            if step % 7 == 3:
                reqs += [reqs[0], reqs[0]]                                # duplicates inside the step
            if step % 5 == 1:
                reqs.insert(1, np.zeros(0, np.int32))                     # empty request
                reqs.append(np.arange(9, dtype=np.int32))                 # shorter than one block
            tokens, offsets = W.pack_requests(reqs)
            assert_same_step(gc.step(dev(tokens), offsets).to_host(), oc.step(tokens, offsets), f"c={c} p={policy} step {step}")
        assert_same_state(gc, oc, f"c={c} policy {policy}")
        gc.close()


def test_step_partition_invariance_on_gpu(arc):
    tr = W.make_trace(1, seed=3)
    reqs = list(tr.requests(max_requests=160))
    outs = []
    for rps in (1, 7, 160):
        gc = arc.ArcCache(64)
        acc = {k: [] for k in ("prefix_len", "cls", "block_id", "evicted_id", "p_after", "alloc_ids", "evict_ids")}
        for s in range(0, len(reqs), rps):
            tokens, offsets = W.pack_requests(reqs[s:s + rps])
            h = gc.step(dev(tokens), offsets).to_host()
            for k in acc:
                acc[k] += h[k].tolist()
        outs.append(acc)
        gc.close()
    assert outs[0] == outs[1] == outs[2]


def test_errors_leave_state_unchanged(arc):
    gc, oc = arc.ArcCache(4), O.OracleCache(4)
    toks = np.arange(48, dtype=np.int32)
    assert_same_step(gc.step(dev(toks), [0, 48]).to_host(), oc.step(toks, [0, 48]))
    big = np.arange(16 * 5, dtype=np.int32)
    with pytest.raises(arc.ArcError) as e:
        gc.step(dev(big), [0, 80])
    assert e.value.code == arc.ERR_REQUEST_TOO_LARGE == oc.step(big, [0, 80])
    with pytest.raises(arc.ArcError) as e:
        gc.step(dev(toks), np.array([0, 32, 16]))
    assert e.value.code == arc.ERR_INVALID_ARG == oc.step(toks, [0, 32, 16])
    assert_same_state(gc, oc, "after errors")
    assert_same_step(gc.step(dev(toks[:40]), [0, 0, 15, 15, 40]).to_host(), oc.step(toks[:40], [0, 0, 15, 15, 40]))
    assert_same_step(gc.step(dev(toks[:0]), [0]).to_host(), oc.step(toks[:0], [0]))
    assert_same_state(gc, oc, "after empty steps")
    for bad in ((0, 16, 0), (4, 15, 0), (4, 16, 3), (4, 16, 9)):
        with pytest.raises(arc.ArcError):
            arc.ArcCache(*bad)
    gc.close()
    gc.close()   # double destroy is a no-op


def test_growth_reset_and_host_entry(arc):
    """Steps larger than the initial buffers (lazy growth with a live directory), arc_reset, arc_step_host."""
    rng = np.random.default_rng(9)
    c = 300
    gc, oc = arc.ArcCache(c), O.OracleCache(c)
    docs = [rng.integers(0, 32000, size=16 * 40, dtype=np.int32) for _ in range(30)]
    for n_req in (10, 40, 200, 700, 90):      # 700 x 40 = 28,000 blocks > the initial 4,096
        reqs = [docs[int(i)] for i in rng.integers(0, 30, size=n_req)]
        tokens, offsets = W.pack_requests(reqs)
        assert_same_step(gc.step(dev(tokens), offsets).to_host(), oc.step(tokens, offsets), f"growth n_req={n_req}")
    assert_same_state(gc, oc, "growth")
    gc.reset()
    oc = O.OracleCache(c)
    for n_req in (5, 50):
        reqs = [docs[int(i)] for i in rng.integers(0, 30, size=n_req)]
        tokens, offsets = W.pack_requests(reqs)
        h = gc.step_host(tokens, offsets)
        o = oc.step(tokens, offsets)
        for k in ("prefix_len", "alloc_ids", "evict_ids"):
            assert np.array_equal(h[k], o[k]), k
    assert_same_state(gc, oc, "after reset + step_host")
    assert gc.launch_count() > 0
    gc.close()


def test_host_entry_pipelined(arc):
    """arc_step_host_async / arc_step_host_wait: three steps in flight, the fourth refused, results (prefix lengths,
    allocated and evicted IDs, in order) equal to the oracle's for every step; mixed with arc_step_host and arc_step."""
    rng = np.random.default_rng(123)
    c = 500
    gc, oc = arc.ArcCache(c), O.OracleCache(c)
    gc.reserve(64, 64 * 60)
    docs = [rng.integers(0, 32000, size=16 * int(n) + int(rng.integers(0, 16)), dtype=np.int32) for n in rng.integers(1, 60, size=40)]
    def batch():
        reqs = [np.concatenate([docs[int(i)], rng.integers(0, 32000, size=int(rng.integers(0, 40)), dtype=np.int32)]) for i in rng.integers(0, 40, size=int(rng.integers(1, 30)))]
        return W.pack_requests(reqs)
    pinned = []
    want = {}
    inflight = []
    for step in range(60):
        tokens, offsets = batch()
        buf = torch.from_numpy(tokens).pin_memory()
        pinned.append(buf)
        t = gc.step_host_async(buf.numpy(), offsets)
        want[t] = oc.step(tokens, offsets)
        inflight.append(t)
        if len(inflight) == 3:
            tk2, of2 = batch()
            with pytest.raises(arc.ArcError):                      # a fourth step in flight is refused, nothing changes
                gc.step_host_async(tk2, of2)
            gc._inflight.pop(max(gc._inflight), None) if len(gc._inflight) > 3 else None
        while len(inflight) > int(rng.integers(0, 3)):
            tk = inflight.pop(0)
            r, o = gc.step_host_wait(tk), want.pop(tk)
            for k in ("prefix_len", "alloc_ids", "evict_ids"):
                assert np.array_equal(r[k], o[k]), (step, k)
            assert r["d2h_bytes"] == 4 * (3 + len(o["prefix_len"]) + len(o["alloc_ids"]) + len(o["evict_ids"]))
    for tk in inflight:
        r, o = gc.step_host_wait(tk), want.pop(tk)
        assert np.array_equal(r["alloc_ids"], o["alloc_ids"])
    tokens, offsets = batch()
    h = gc.step_host(tokens, offsets)
    o = oc.step(tokens, offsets)
    assert np.array_equal(h["evict_ids"], o["evict_ids"]) and np.array_equal(h["prefix_len"], o["prefix_len"])
    tokens, offsets = batch()
    assert_same_step(gc.step(dev(tokens), offsets).to_host(), oc.step(tokens, offsets), "arc_step after host steps")
    assert_same_state(gc, oc, "host entry")
    gc.close()


def test_maintenance_rebuild_and_compaction(arc):
    """Many small steps on one handle: the table rebuild and the ring compaction both trigger many times."""
    rng = np.random.default_rng(11)
    c = 128
    for policy in (0, 1):
        gc, oc = arc.ArcCache(c, 16, policy), O.OracleCache(c, 16, policy)
        docs = [rng.integers(0, 32000, size=16 * int(n), dtype=np.int32) for n in rng.integers(1, 40, size=60)]
        for step in range(400):
            reqs = [np.concatenate([docs[int(i)], rng.integers(0, 32000, size=int(rng.integers(0, 50)), dtype=np.int32)])
                    for i in rng.zipf(1.2, size=24) % 60]
            tokens, offsets = W.pack_requests(reqs)
            g = gc.step(dev(tokens), offsets)
            o = oc.step(tokens, offsets)
            if step % 20 == 0 or step > 390:
                assert_same_step(g.to_host(), o, f"maint policy {policy} step {step}")
        assert_same_state(gc, oc, f"maintenance policy {policy}")
        gc.close()


@pytest.mark.parametrize("machine", [0, 1, 2, 3, 4, 5])
@pytest.mark.parametrize("bits", [3, 6])
def test_equal_keys_inside_a_request(arc, machine, bits):
    """The same key several times inside one request (forced with the key-mask test hook; the 64-bit hash never does
    it): the second access is a hit on a block its own request has pinned.  Exercises the window cuts at repeated nodes."""
    rng = np.random.default_rng(40 + bits)
    mask = (1 << bits) - 1
    for policy in (0, 1, 2):
        c = 40
        gc, oc = arc.ArcCache(c, 16, policy), O.OracleCache(c, 16, policy)
        gc.set_machine(machine)
        gc.debug_set_key_mask(mask)
        for step in range(25):
            reqs = [rng.integers(0, 50, size=16 * int(rng.integers(1, c + 1)) + int(rng.integers(0, 16)), dtype=np.int32)
                    for _ in range(int(rng.integers(1, 6)))]
            tokens, offsets = W.pack_requests(reqs)
            keys, blk_off = O.hash_blocks(tokens, offsets)
            keys = keys & np.uint64(mask)
            keys[keys < 2] += np.uint64(2)
            o = oc.step_keys([keys[blk_off[r]:blk_off[r + 1]] for r in range(len(reqs))])
            g = gc.step(dev(tokens), offsets).to_host()
            for k in OUT_KEYS:
                assert np.array_equal(g[k], o[k]), f"bits {bits} policy {policy} machine {machine} step {step}: {k}"
        gl, ol = gc.debug_lists(), oc.lists()
        for n in ("T1", "T2", "B1", "B2"):
            assert np.array_equal(gl[n][0], ol[n][0]) and np.array_equal(gl[n][1], ol[n][1]), n
        gc.close()


def test_latency_histogram_of_the_by_the_book_machine(arc):
    """arc_debug_latency_hist: with machine 1 every access lands in exactly one bin of its class (counts per class equal
    the class counters), other machines leave it untouched."""
    tr = W.make_trace(1, seed=4, scale=0.2)
    gc = arc.ArcCache(64)
    gc.set_machine(1)
    for tokens, offsets in tr.steps():
        gc.step(dev(tokens), offsets)
    st, h = gc.stats(), gc.debug_latency_hist()
    assert h.sum() == st["accesses"] > 0
    assert [int(x) for x in h.sum(axis=1)] == [st["miss"], st["hit_t1"], st["hit_t2"], st["ghost_b1"], st["ghost_b2"]]
    gc.set_machine(3)
    for tokens, offsets in tr.steps(max_steps=5):
        gc.step(dev(tokens), offsets)
    assert gc.debug_latency_hist().sum() == h.sum()
    gc.close()


def test_probe_alone_is_a_consistent_map(arc):
    """K2 through arc_debug_probe: equal keys get equal nodes, different keys different nodes, lookups repeat."""
    g = torch.Generator(device="cuda")
    g.manual_seed(5)
    n = 300_000
    keys = torch.randint(2, 2 ** 62, (n,), dtype=torch.int64, device="cuda", generator=g)
    keys[1000:2000] = keys[0:1000]                      # duplicates inside one launch race for the same slot
    gc = arc.ArcCache(50_000)
    nodes = gc.debug_probe(keys).clone()
    torch.cuda.synchronize()
    assert torch.equal(nodes[1000:2000], nodes[0:1000])
    uniq_keys = torch.unique(keys).numel()
    assert torch.unique(nodes).numel() == uniq_keys
    again = gc.debug_probe(keys.flip(0))
    torch.cuda.synchronize()
    assert torch.equal(again.flip(0), nodes)
    gc.stats()                                          # no device-side error
    gc.close()


def test_probe_on_a_table_far_larger_than_l2(arc):
    """K2 at c = 16 M blocks (a 2 GiB table, 16 x the 126 MB L2; the size bench.py's probe leg times): 16 M random keys
    of which 1 M repeat inside the launch (they race for one slot and must share one node), every key found again at
    its node in a second launch in another order, as many nodes as distinct keys, no device-side error; and the
    random-sector ceiling kernel reads what the table holds."""
    n = 1 << 24
    g = torch.Generator(device="cuda")
    g.manual_seed(16)
    keys = torch.randint(2, 2 ** 62, (n,), dtype=torch.int64, device="cuda", generator=g)
    keys[5:5 + 4096:2] = keys[4:4 + 4096:2]              # duplicates inside one launch: adjacent (same warp, same instant) ...
    keys[n - (1 << 20):] = keys[:1 << 20]                # ... and far apart in the grid
    gc = arc.ArcCache(n)
    gc.reserve(1, n)
    nodes = gc.debug_probe(keys).clone()
    torch.cuda.synchronize()
    assert torch.equal(nodes[n - (1 << 20):], nodes[:1 << 20])
    assert torch.equal(nodes[5:5 + 4096:2], nodes[4:4 + 4096:2])
    n_keys = torch.unique(keys).numel()
    assert torch.unique(nodes).numel() == n_keys and int(nodes.min()) >= 0
    perm = torch.randperm(n, device="cuda", generator=g)
    again = gc.debug_probe(keys[perm].contiguous())
    torch.cuda.synchronize()
    assert torch.equal(again, nodes[perm])
    gc.stats()                                           # raises on a device-side error (node pool, bad node)
    gc.close()
    buf = torch.arange(1 << 22, dtype=torch.int32, device="cuda")          # 16 MiB = 2^19 sectors
    x = arc.debug_gather_sectors(keys[:4096], buf).cpu().numpy()
    k = keys[:4096].cpu().numpy().view(np.uint64)
    want = np.bitwise_xor.reduce(buf.cpu().numpy().reshape(-1, 8)[(k & np.uint64((1 << 19) - 1)).astype(np.int64)], axis=1)
    assert np.array_equal(x, want)


@pytest.mark.parametrize("machine", [0, 1, 2, 3, 4, 5])
def test_step_wide_pin_scope(arc, machine):
    """NEXT-3 (part): ARC_PIN_STEP.  Hand trace G's situation (an earlier request's block is still pinned when a later
    request of the same step needs a victim), the admission rule, and random steps on small caches, against the oracle."""
    X = np.arange(100, 164, dtype=np.int32)
    Y, Z = np.arange(500, 516, dtype=np.int32), np.arange(700, 716, dtype=np.int32)
    for scope in (arc.PIN_REQUEST, arc.PIN_STEP):
        gc, oc = arc.ArcCache(4), O.OracleCache(4)
        gc.set_machine(machine)
        gc.set_pin_scope(scope)
        oc.set_pin_scope(scope)
        for reqs in ([X], [X], [Y, Z]):
            tokens, offsets = W.pack_requests(reqs)
            assert_same_step(gc.step(dev(tokens), offsets).to_host(), oc.step(tokens, offsets), f"scope {scope}")
        assert_same_state(gc, oc, f"scope {scope}")
        t1 = gc.debug_lists()["T1"][0]
        assert len(t1) == (2 if scope == arc.PIN_STEP else 1)          # Y0 survives only under step-wide pins
        big, boff = W.pack_requests([np.arange(48, dtype=np.int32), np.arange(900, 932, dtype=np.int32)])   # 3 + 2 blocks > c
        if scope == arc.PIN_STEP:
            with pytest.raises(arc.ArcError) as e:
                gc.step(dev(big), boff)
            assert e.value.code == arc.ERR_REQUEST_TOO_LARGE == oc.step(big, boff)
            assert_same_state(gc, oc, "after the refused step")
        gc.close()
    rng = np.random.default_rng(17)
    for policy in (0, 1, 2):
        for c in (3, 6, 40):
            gc, oc = arc.ArcCache(c, 16, policy), O.OracleCache(c, 16, policy)
            gc.set_machine(machine)
            gc.set_pin_scope(arc.PIN_STEP)
            oc.set_pin_scope(arc.PIN_STEP)
            table = rng.integers(0, 1000, size=(4, 2, 16), dtype=np.int32)
            for step in range(50):
                reqs, left = [], c
                while left > 0 and rng.random() < 0.85:
                    r = _tree_request(rng, table, min(left, 6))
                    reqs.append(r)
                    left -= len(r) // 16
                tokens, offsets = W.pack_requests(reqs)
                assert_same_step(gc.step(dev(tokens), offsets).to_host(), oc.step(tokens, offsets), f"step scope p{policy} c{c} step {step}")
            assert_same_state(gc, oc, f"step scope p{policy} c{c}")
            gc.close()


@pytest.mark.parametrize("policy", [0, 1, 2])
def test_many_tiny_requests_and_cache_sized_requests(arc, policy):
    """Edge shapes: 20,000 requests of 0-2 blocks in one step (most of K3's windows are one or two accesses), then requests
    of exactly c blocks (everything resident is replaced by one request), then a hit on all of it."""
    rng = np.random.default_rng(61 + policy)
    c = 3000
    gc, oc = arc.ArcCache(c, 16, policy), O.OracleCache(c, 16, policy)
    base = rng.integers(0, 5000, size=(300, 32), dtype=np.int32)          # 300 two-block prefixes
    reqs = []
    for _ in range(20000):
        b = base[int(rng.integers(0, 300))]
        reqs.append(b[:int(rng.integers(0, 40))])                          # 0 .. 39 tokens: 0, 1 or 2 full blocks
    tokens, offsets = W.pack_requests(reqs)
    assert_same_step(gc.step(dev(tokens), offsets).to_host(), oc.step(tokens, offsets), "tiny requests")
    big1 = rng.integers(0, 5000, size=16 * c, dtype=np.int32)
    big2 = rng.integers(0, 5000, size=16 * c + 9, dtype=np.int32)
    for name, r in (("cache-sized", [big1]), ("another", [big2]), ("again", [big2]), ("first again", [big1])):
        tokens, offsets = W.pack_requests(r)
        assert_same_step(gc.step(dev(tokens), offsets).to_host(), oc.step(tokens, offsets), name)
    assert_same_state(gc, oc, "edge shapes")
    gc.close()


def _tree_request(rng, table, max_blocks):
    """A root-to-node path in a FIXED token-block tree (table[level, branch] = one block): requests drawn from the same
    table share prefixes, so hits, ghost hits and hold counts above one all occur."""
    depth, branching, B = table.shape
    nb = int(rng.integers(1, max_blocks + 1))
    path = rng.integers(0, branching, size=nb)
    if rng.random() < 0.5:
        path[: min(nb, 3)] = 0                         # a popular trunk
    toks = [table[min(l, depth - 1), int(b)] for l, b in enumerate(path)]
    toks.append(rng.integers(0, 1000, size=int(rng.integers(0, B)), dtype=np.int32))
    return np.concatenate(toks).astype(np.int32)


def _serving_loop(arc, gc, oc, rng, c, steps, ctx, table, max_req_blocks=6):
    """Random steps and random releases under ARC_PIN_HELD, GPU against the oracle; returns the requests still held."""
    live = []
    refused = 0
    for step in range(steps):
        assert gc.hold_units() == oc.hold_units() == sum(len(x) for x in live), ctx
        if live and (rng.random() < 0.45 or oc.hold_units() > c - 2):
            ids = live.pop(int(rng.integers(0, len(live))))
            ids = ids[rng.permutation(len(ids))]
            while live and rng.random() < 0.4:          # several requests in one call: shared blocks appear several times
                ids = np.concatenate([ids, live.pop(int(rng.integers(0, len(live))))])
            gc.release(ids)
            assert oc.release(ids) == 0, ctx
        else:
            reqs, left = [], c - oc.hold_units() + (2 if rng.random() < 0.1 else 0)   # now and then one step too many
            while left > 0 and rng.random() < 0.85:
                r = _tree_request(rng, table, min(left, max_req_blocks))
                reqs.append(r)
                left -= len(r) // 16
            tokens, offsets = W.pack_requests(reqs)
            o = oc.step(tokens, offsets)
            if isinstance(o, int):
                assert o == arc.ERR_REQUEST_TOO_LARGE
                with pytest.raises(arc.ArcError) as e:
                    gc.step(dev(tokens), offsets)
                assert e.value.code == arc.ERR_REQUEST_TOO_LARGE
                refused += 1
                continue
            g = gc.step(dev(tokens), offsets).to_host()
            assert_same_step(g, o, f"{ctx} step {step}")
            off = o["blk_off"]
            live += [o["block_id"][off[r]:off[r + 1]].copy() for r in range(len(reqs)) if off[r + 1] > off[r]]
        if step % 16 == 0:
            assert_same_state(gc, oc, f"{ctx} step {step}")
    assert_same_state(gc, oc, ctx)
    return live, refused


@pytest.mark.parametrize("machine", [0, 1, 2, 3, 4, 5])
@pytest.mark.parametrize("policy", [0, 1, 2])
def test_held_pins_and_release(arc, policy, machine):
    """NEXT-3: ARC_PIN_HELD and arc_release.  A serving loop - steps add holds, finished requests give
    them back in arbitrary order, several requests per call - on small and medium caches; the scope is entered on a cache
    that already has content and left again; everything bit-exact against the oracle, lists included."""
    rng = np.random.default_rng(900 + 10 * policy + machine)
    seen = dict(hit=0, ghost=0, refused=0)
    for c, steps, mrb, depth in ((5, 150, 3, 3), (24, 250, 6, 4), (300, 200, 40, 7), (3000, 60, 700, 12)):
        table = rng.integers(0, 1000, size=(depth, 2, 16), dtype=np.int32)
        gc, oc = arc.ArcCache(c, 16, policy), O.OracleCache(c, 16, policy)
        gc.set_machine(machine)
        ctx = f"held p{policy} m{machine} c{c}"
        for i in range(10):                               # default scope first: the cache has content when the scope changes
            tokens, offsets = W.pack_requests([_tree_request(rng, table, min(c, mrb)) for _ in range(3)])
            assert_same_step(gc.step(dev(tokens), offsets).to_host(), oc.step(tokens, offsets), f"{ctx} warm {i}")
        gc.set_pin_scope(arc.PIN_HELD)
        oc.set_pin_scope(2)
        live, refused = _serving_loop(arc, gc, oc, rng, c, steps, ctx, table, mrb)
        seen["refused"] += refused
        if live:                                          # the scope cannot change while holds are outstanding
            with pytest.raises(arc.ArcError):
                gc.set_pin_scope(arc.PIN_REQUEST)
            ids = np.concatenate(live)
            gc.release(ids)
            assert oc.release(ids) == 0
        assert gc.hold_units() == oc.hold_units() == 0
        assert_same_state(gc, oc, ctx + " all released")
        gs = gc.stats()
        assert gs["t1"] + gs["t2"] == len(gc.debug_lists()["T1"][0]) + len(gc.debug_lists()["T2"][0])   # everything is back in a ring
        seen["hit"] += gs["hit_t1"] + gs["hit_t2"]
        seen["ghost"] += gs["ghost_b1"] + gs["ghost_b2"]
        gc.set_pin_scope(arc.PIN_REQUEST)
        oc.set_pin_scope(0)
        for i in range(10):
            tokens, offsets = W.pack_requests([_tree_request(rng, table, min(c, mrb)) for _ in range(3)])
            assert_same_step(gc.step(dev(tokens), offsets).to_host(), oc.step(tokens, offsets), f"{ctx} after {i}")
        assert_same_state(gc, oc, ctx + " back in the request scope")
        gc.close()
    assert seen["hit"] > 100 and seen["refused"] > 0, seen     # the loop really shares prefixes and really hits the admission rule
    if policy != 1:
        assert seen["ghost"] > 0, seen


def test_held_pins_protect_blocks_and_bad_release_is_flagged(arc):
    """A held request survives any amount of traffic; releasing what is not held changes nothing and raises the sticky
    device error."""
    c = 64
    gc, oc = arc.ArcCache(c), O.OracleCache(c)
    gc.set_pin_scope(arc.PIN_HELD)
    oc.set_pin_scope(2)
    doc = np.arange(5000, 5000 + 16 * 20, dtype=np.int32)             # 20 blocks, held for the whole test
    off = np.array([0, len(doc)], np.int64)
    g0 = gc.step(dev(doc), off).to_host()
    assert_same_step(g0, oc.step(doc, off), "held doc")
    rng = np.random.default_rng(5)
    for i in range(60):                                               # 60 x 40 fresh blocks through the other 44 slots
        t = rng.integers(10 ** 6, 2 * 10 ** 6, size=16 * 40).astype(np.int32)
        o2 = np.array([0, len(t)], np.int64)
        g, o = gc.step(dev(t), o2).to_host(), oc.step(t, o2)
        assert_same_step(g, o, f"traffic {i}")
        assert not np.isin(g["evicted_id"], g0["block_id"]).any()     # never a held block
        gc.release(g["block_id"])
        assert oc.release(o["block_id"]) == 0
    g1 = gc.step(dev(doc), off).to_host()
    assert_same_step(g1, oc.step(doc, off), "held doc again")
    assert (g1["cls"] != 0).all() and np.array_equal(g1["block_id"], g0["block_id"]) and g1["prefix_len"][0] == len(doc)
    assert gc.hold_units() == 40
    with pytest.raises(arc.ArcError):
        gc.release(np.arange(41, dtype=np.int32))                     # more IDs than holds: refused on the host
    assert_same_state(gc, oc, "before the bad release")
    bad = np.concatenate([g0["block_id"][:3], g0["block_id"][:1], g0["block_id"][:1]])   # the first block three times: held twice
    assert oc.release(bad) == O.ERR_INVALID_ARG
    gc.release(bad)
    with pytest.raises(arc.ArcError):
        gc.stats()
    with pytest.raises(arc.ArcError):                                 # the host entry reports the sticky error too (no arc_stats needed)
        gc.step_host(np.zeros(0, np.int32), np.zeros(1, np.int64))
    gl, ol = gc.debug_lists(), oc.lists()
    for n in ("T1", "T2", "B1", "B2"):
        assert np.array_equal(gl[n][0], ol[n][0]), n                   # nothing changed
    gc.close()


def test_resumed_requests_chain_state_and_split_invariance(arc):
    """arc_step_resume: chain_state equals the oracle's for requests of every shape (empty, shorter
    than a block, many rounds, misaligned starts); a prompt sent in chunks that continue from the returned state gets
    the keys of the unsplit prompt (seen as hits on a cache that served the whole prompt), mixed in one step with new
    prompts; everything bit-exact against the oracle."""
    rng = np.random.default_rng(4242)
    c = 4096
    gc, oc = arc.ArcCache(c), O.OracleCache(c)
    lens = [0, 5, 16, 17, 31, 32, 16 * 33 + 3, 16 * 64, 16 * 100 + 15, 16 * 257 + 9]
    prompts = [rng.integers(0, 128000, size=n).astype(np.int32) for n in lens]
    tokens, offsets = W.pack_requests(prompts)
    g, o = gc.step(dev(tokens), offsets).to_host(), oc.step(tokens, offsets)
    assert_same_step(g, o, "whole prompts")
    assert np.array_equal(g["chain_state"], o["chain_state"])
    assert g["chain_state"][0] == g["chain_state"][1] == np.uint64(0x243F6A8885A308D3)      # no full block: S0
    whole_state = g["chain_state"].copy()
    # the same prompts in two chunks; chunk 1 may end inside a block, chunk 2 starts again at the block boundary
    cuts = [int(rng.integers(0, n // 16 + 1)) for n in lens]
    part1 = [p[:16 * k + (int(rng.integers(0, 16)) if 16 * k + 16 <= len(p) else 0)] for p, k in zip(prompts, cuts)]
    part2 = [p[16 * k:] for p, k in zip(prompts, cuts)]
    g2c, o2c = arc.ArcCache(c), O.OracleCache(c)
    t1, o1 = W.pack_requests(part1)
    ga, oa = g2c.step(dev(t1), o1).to_host(), o2c.step(t1, o1)
    assert_same_step(ga, oa, "chunk 1")
    assert np.array_equal(ga["chain_state"], oa["chain_state"])
    fresh = [rng.integers(0, 128000, size=16 * 7 + 3).astype(np.int32)]                       # a new prompt in the same step
    t2, o2 = W.pack_requests(part2 + fresh)
    chain = np.concatenate([ga["chain_state"], np.array([0x243F6A8885A308D3], np.uint64)])
    gb = g2c.step(dev(t2), o2, chain_in=chain).to_host()
    ob = o2c.step(t2, o2, chain_in=chain)
    assert_same_step(gb, ob, "chunk 2")
    assert np.array_equal(gb["chain_state"], ob["chain_state"])
    assert np.array_equal(gb["chain_state"][:-1], whole_state)
    # on the cache that served the unsplit prompts the chunks are hits from block 0 of each chunk on
    gh = gc.step(dev(t2), o2, chain_in=torch.from_numpy(chain.view(np.int64)).cuda()).to_host()
    oh = oc.step(t2, o2, chain_in=chain)
    assert_same_step(gh, oh, "chunks against the whole")
    nb2 = np.array([len(p) // 16 for p in part2])
    assert np.array_equal(gh["prefix_len"][:-1], 16 * nb2)
    assert_same_state(gc, oc, "resume")
    assert_same_state(g2c, o2c, "resume, chunked")
    gc.close(); g2c.close()


@pytest.mark.parametrize("policy", [0, 1, 2])
def test_decode_loop_with_held_pins(arc, policy):
    """The serving loop NEXT-3 describes: held pins, running sequences that grow by the tokens generated since the last
    step (one block when 16 have accumulated, nothing otherwise) from their stored chain state, new prompts arriving,
    finished sequences releasing every block they hold.  GPU against the oracle, outputs, chain states, lists."""
    rng = np.random.default_rng(600 + policy)
    c = 160
    table = rng.integers(0, 1000, size=(6, 2, 16), dtype=np.int32)
    gc, oc = arc.ArcCache(c, 16, policy), O.OracleCache(c, 16, policy)
    gc.set_pin_scope(arc.PIN_HELD)
    oc.set_pin_scope(2)
    S0 = np.uint64(0x243F6A8885A308D3)
    running = []                      # dicts: state (uint64), pending (tokens of the block being filled), ids (block IDs held)
    grown = 0
    for step in range(300):
        reqs, chain, owner = [], [], []
        for q in running:
            q["pending"] = np.concatenate([q["pending"], rng.integers(0, 50, size=int(rng.integers(3, 12))).astype(np.int32)])
            reqs.append(q["pending"]); chain.append(q["state"]); owner.append(q)
        budget = c - oc.hold_units() - sum(len(r) // 16 for r in reqs)
        while len(running) + (len(reqs) - len(running)) < 6 and budget > 12 and rng.random() < 0.5:
            r = _tree_request(rng, table, min(budget - 6, 24))
            q = dict(state=S0, pending=np.zeros(0, np.int32), ids=[], new=True)
            reqs.append(r); chain.append(S0); owner.append(q)
            budget -= len(r) // 16
        if not reqs:
            continue
        tokens, offsets = W.pack_requests(reqs)
        chain = np.array(chain, np.uint64)
        g = gc.step(dev(tokens), offsets, chain_in=chain).to_host()
        o = oc.step(tokens, offsets, chain_in=chain)
        assert_same_step(g, o, f"decode p{policy} step {step}")
        assert np.array_equal(g["chain_state"], o["chain_state"]), step
        off = g["blk_off"]
        for r, q in enumerate(owner):
            nb = int(off[r + 1] - off[r])
            q["state"] = g["chain_state"][r]
            q["ids"] += g["block_id"][off[r]:off[r + 1]].tolist()
            q["pending"] = reqs[r][16 * nb:]                  # the tokens of the block still being filled
            if q.pop("new", False):
                running.append(q)
            elif nb:
                grown += nb
        for q in list(running):                               # some sequences finish: all their holds go back in one call
            if rng.random() < 0.08 or oc.hold_units() > c - 30:
                running.remove(q)
                ids = np.array(q["ids"], np.int32)
                gc.release(ids)
                assert oc.release(ids) == 0
        assert gc.hold_units() == oc.hold_units()
        if step % 25 == 0:
            assert_same_state(gc, oc, f"decode p{policy} step {step}")
    assert grown > 50                                         # sequences really grew block by block
    assert_same_state(gc, oc, f"decode p{policy}")
    gc.close()


@pytest.mark.parametrize("shift", [0, 1, 2, 3])
def test_segmented_in_step_hashing(arc, shift):
    """Steps with few, long requests hash every request in 128-block segments (hash_segments_kernel + hash_fixup_kernel).
    Request lengths around the segment and round boundaries, a misaligned token buffer, continuation states: the keys
    (seen through the lists), the classes and the chain states equal the oracle's."""
    rng = np.random.default_rng(31 + shift)
    blocks = [128, 129, 127, 1, 0, 255, 256, 257, 33, 1023, 1024, 640]
    reqs = [rng.integers(0, 128000, size=16 * nb + int(rng.integers(0, 16))).astype(np.int32) for nb in blocks]
    tokens, offsets = W.pack_requests(reqs)
    buf = torch.zeros(len(tokens) + 8, dtype=torch.int32, device="cuda")
    buf[shift:shift + len(tokens)] = torch.from_numpy(tokens).cuda()
    view = buf[shift:shift + len(tokens)]                               # 4-byte aligned only for shift != 0
    c = 8192
    gc, oc = arc.ArcCache(c), O.OracleCache(c)
    chain = rng.integers(0, 2 ** 63, size=len(reqs)).astype(np.uint64)
    for rep, ci in enumerate((None, None, chain)):
        g = gc.step(view, offsets, chain_in=ci).to_host()
        o = oc.step(tokens, offsets, chain_in=ci)
        assert_same_step(g, o, f"segmented rep {rep}")
        assert np.array_equal(g["chain_state"], o["chain_state"]), rep
        assert_same_state(gc, oc, f"segmented rep {rep}")
    gc.close()
