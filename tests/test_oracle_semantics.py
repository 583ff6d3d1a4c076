"""Invariants I1-I12, brute-force differential, LRU closed form, ARC==LRU trace classes, partition
invariance, statistical sanity (SURVEY.md §8(c) pins 1, 3-7)."""
import numpy as np
import pytest

from helpers import check_invariants
from oracle import oracle as O
from oracle import oracle_bruteforce as BF
from paper_2606_21238_b200 import workloads as W

HITS = (O.HIT_T1, O.HIT_T2)


def _bf_lists(cache):
    L = cache.lists()
    out = {}
    for n in ("T1", "T2"):
        out[n] = (np.array(L[n], np.uint64), np.array([cache.block_of[k] for k in L[n]], np.int32))
    for n in ("B1", "B2"):
        out[n] = (np.array(L[n], np.uint64), np.full(len(L[n]), -1, np.int32))
    out["p"], out["next_fresh"] = L["p"], cache.next_fresh
    return out


def _random_key_requests(rng, c, n_req, alphabet):
    reqs = []
    for _ in range(n_req):
        nb = int(rng.integers(1, min(c, 4) + 1))
        reqs.append(rng.choice(alphabet, size=nb, replace=False).tolist())
    return reqs


@pytest.mark.parametrize("policy", [0, 1, 2])
def test_invariants_after_every_access_bruteforce(policy):
    rng = np.random.default_rng(10 + policy)
    for c in (1, 2, 3, 5, 8):
        cache = BF.BruteForceCache(c, 16, policy)
        alphabet = np.arange(2, 2 + 3 * c)
        prev_p = cache.p
        for _ in range(600):
            if len(cache.pinned) >= c:   # a request has at most c blocks (R4)
                cache.pinned.clear()
            x = int(rng.choice(alphabet))
            cls, bid, evi = cache.access(x)
            check_invariants(_bf_lists(cache), c, policy_lru=(policy == 1), pinned=cache.pinned)
            if cls not in (O.GHOST_B1, O.GHOST_B2):
                assert cache.p == prev_p, "I12: p moves only on ghost hits"
            prev_p = cache.p
            assert 0 <= bid < c
            if evi >= 0:
                assert evi == bid, "R8: a non-hit reuses exactly the ID its own eviction freed"
            if rng.random() < 0.4:
                cache.pinned.clear()   # request boundary


@pytest.mark.parametrize("policy", [0, 1, 2])
def test_invariants_cpp_config1(policy):
    tr = W.make_trace(1, seed=0)
    cache = O.OracleCache(64, 16, policy)
    prev_full = False
    for tokens, offsets in tr.steps(max_steps=60):
        # one request per oracle step so that the invariants are checked at every request boundary
        for r in range(len(offsets) - 1):
            out = cache.step(tokens[offsets[r]:offsets[r + 1]], [0, offsets[r + 1] - offsets[r]])
            L = cache.lists()
            check_invariants(L, 64, policy_lru=(policy == 1))
            full = len(L["T1"][0]) + len(L["T2"][0]) == 64
            assert full or not prev_full, "I7: once full, stays full"
            prev_full = full
            nonhit = int((~np.isin(out["cls"], HITS)).sum())
            assert len(out["alloc_ids"]) == nonhit, "I10"
            assert int(out["prefix_len"][0]) % 16 == 0 and out["prefix_len"][0] <= 16 * out["n_access"], "I11"
            assert ((out["evicted_id"] == -1) | (out["evicted_id"] == out["block_id"])).all(), "R8"
    st = cache.stats()
    assert st["accesses"] == st["hit_t1"] + st["hit_t2"] + st["ghost_b1"] + st["ghost_b2"] + st["miss"]
    assert st["tokens_hashed"] == 16 * st["accesses"]
    assert st["fresh_ids_used"] == 64
    assert st["evict_t1"] + st["evict_t2"] == st["accesses"] - st["hit_t1"] - st["hit_t2"] - 64, "I10 over the run"


@pytest.mark.parametrize("policy", [0, 1, 2])
def test_differential_cpp_vs_bruteforce_keys(policy):
    """>= 10^4 random traces on c in 1..8, alphabet <= 3c, requests of 1..min(c,4) blocks; every output compared."""
    rng = np.random.default_rng(100 + policy)
    n_traces = 0
    for rep in range(700):
        for c in range(1, 9):
            alphabet = np.arange(2, 2 + int(rng.integers(c, 3 * c + 1)))
            bf, cpp = BF.BruteForceCache(c, 16, policy), O.OracleCache(c, 16, policy)
            for step in range(3):
                reqs = _random_key_requests(rng, min(c, len(alphabet)), int(rng.integers(1, 5)), alphabet)
                a, b = bf.step_keys(reqs), cpp.step_keys(reqs)
                for k in ("prefix_len", "blk_off", "cls", "block_id", "evicted_id", "p_after", "alloc_ids", "evict_ids"):
                    assert list(a[k]) == b[k].tolist(), (c, k, reqs)
            Lb, Lc = bf.lists(), cpp.lists()
            for n in ("T1", "T2", "B1", "B2"):
                assert Lb[n] == Lc[n][0].tolist()
            sb, sc = bf.stats, cpp.stats()
            for k in sb:
                assert sb[k] == sc[k], k
            n_traces += 1
    assert n_traces >= 5000  # x2 policies >= 10^4


def test_differential_tokens_prefix_trees():
    """Same, through the hash: requests are paths in small token-block trees so chained keys are shared."""
    rng = np.random.default_rng(7)
    for rep in range(150):
        c = int(rng.integers(1, 9))
        for policy in (0, 1, 2):
            bf, cpp = BF.BruteForceCache(c, 16, policy), O.OracleCache(c, 16, policy)
            reqs = W.prefix_tree_requests(rng, n_requests=12, block_size=16, branching=2, depth=3, max_blocks=min(c, 4))
            for s in range(0, 12, 4):
                tokens, offsets = W.pack_requests(reqs[s:s + 4])
                a, b = bf.step(tokens.tolist(), offsets.tolist()), cpp.step(tokens, offsets)
                for k in ("prefix_len", "blk_off", "cls", "block_id", "evicted_id", "p_after", "alloc_ids", "evict_ids"):
                    assert list(a[k]) == b[k].tolist(), (c, policy, k)
            assert bf.stats == {k: v for k, v in cpp.stats().items() if k in bf.stats}


def test_lru_stack_distance_closed_form():
    """Single-block requests: a hit iff fewer than c distinct other keys since the previous access of the
    same key.  Computed straight from the trace, no list code."""
    rng = np.random.default_rng(20)
    for c in (1, 2, 3, 7, 16):
        trace = (rng.zipf(1.3, size=1500) % (4 * c) + 2).tolist()
        cache = O.OracleCache(c, 16, O.POLICY_LRU)
        got = [int(cache.step_keys([[x]])["cls"][0]) for x in trace]
        last = {}
        for t, x in enumerate(trace):
            if x in last:
                distinct = len(set(trace[last[x] + 1:t]))
                want = O.HIT_T1 if distinct < c else O.MISS
            else:
                want = O.MISS
            assert got[t] == want, (c, t)
            last[x] = t


def _same_outputs(c, reqs_keys):
    a, l = O.OracleCache(c, 16, O.POLICY_ARC), O.OracleCache(c, 16, O.POLICY_LRU)
    for r in reqs_keys:
        oa, ol = a.step_keys([r]), l.step_keys([r])
        assert np.isin(oa["cls"], HITS).tolist() == np.isin(ol["cls"], HITS).tolist()
        assert (oa["cls"] == 0).tolist() == (ol["cls"] == 0).tolist()      # no ghost hits on these traces
        assert oa["block_id"].tolist() == ol["block_id"].tolist()
        assert oa["evicted_id"].tolist() == ol["evicted_id"].tolist()
        assert (oa["p_after"] == 0).all()


def test_arc_equals_lru_on_pure_recency_traces():
    rng = np.random.default_rng(30)
    _same_outputs(8, [[int(k)] for k in range(2, 200)])                                  # (i) all keys distinct
    ws = rng.integers(2, 10, size=400).tolist()
    _same_outputs(8, [[k] for k in ws])                                                   # (ii) working set <= c
    _same_outputs(3, [[k] for k in np.repeat(np.arange(2, 60), 2).tolist()])              # (iii) each key twice back-to-back
    _same_outputs(16, [list(range(100 + 5 * i, 100 + 5 * i + 5)) for i in range(40)])     # (i) with multi-block requests


@pytest.mark.parametrize("policy", [0, 1, 2])
def test_step_partition_invariance(policy):
    """R3 / PAPER.md:129: the same request stream cut into steps of 1, 7, 64 or all at once gives identical
    concatenated outputs."""
    tr = W.make_trace(1, seed=3)
    reqs = list(tr.requests(max_requests=200))
    results = []
    for rps in (1, 7, 64, 200):
        cache = O.OracleCache(64, 16, policy)
        acc = {k: [] for k in ("prefix_len", "cls", "block_id", "evicted_id", "p_after", "alloc_ids", "evict_ids")}
        for s in range(0, len(reqs), rps):
            tokens, offsets = W.pack_requests(reqs[s:s + rps])
            out = cache.step(tokens, offsets)
            for k in acc:
                acc[k] += out[k].tolist()
        results.append((acc, cache.stats()))
    for acc, st in results[1:]:
        assert acc == results[0][0]
        for k in st:
            if k != "steps":
                assert st[k] == results[0][1][k]


def test_errors_leave_state_unchanged():
    cache = O.OracleCache(4)
    toks = np.arange(16 * 3, dtype=np.int32)
    assert isinstance(cache.step(toks, [0, 48]), dict)
    before, st = cache.lists(), cache.stats()
    big = np.arange(16 * 5, dtype=np.int32)
    assert cache.step(big, [0, 80]) == O.ERR_REQUEST_TOO_LARGE          # nb_r > c
    assert cache.step(np.concatenate([toks, big]), [0, 48, 128]) == O.ERR_REQUEST_TOO_LARGE   # even if an earlier request is fine
    assert cache.step(toks, [0, 32, 16]) == O.ERR_INVALID_ARG
    after = cache.lists()
    for n in ("T1", "T2", "B1", "B2"):
        assert before[n][0].tolist() == after[n][0].tolist()
    assert cache.stats() == st
    # exactly c blocks is allowed
    assert isinstance(cache.step(np.arange(64, dtype=np.int32), [0, 64]), dict)
    with pytest.raises(ValueError):
        O.OracleCache(0)
    with pytest.raises(ValueError):
        O.OracleCache(4, 15)
    with pytest.raises(ValueError):
        O.OracleCache(4, 16, 7)


def test_empty_and_short_requests():
    cache = O.OracleCache(8)
    out = cache.step(np.arange(40, dtype=np.int32), [0, 0, 15, 15, 40])    # empty, <B, empty, 25 tokens -> 1 block
    assert out["blk_off"].tolist() == [0, 0, 0, 0, 1]
    assert out["prefix_len"].tolist() == [0, 0, 0, 0]
    assert out["n_access"] == 1
    out = cache.step(np.zeros(0, np.int32), [0])
    assert out["n_access"] == 0
    st = cache.stats()
    assert st["requests"] == 4 and st["steps"] == 2 and st["tokens_seen"] == 40 and st["tokens_hashed"] == 16


def test_lru_hit_rate_matches_che_approximation():
    """Statistical sanity: LRU block hit rate of single-block Zipf traffic vs Che's approximation (~1 point)."""
    rng = np.random.default_rng(40)
    n_items, c, s = 2000, 200, 0.9
    p = W.zipf_probabilities(n_items, s)
    trace = rng.choice(n_items, size=60000, p=p) + 2
    cache = O.OracleCache(c, 16, O.POLICY_LRU)
    hits = 0
    for s0 in range(0, len(trace), 500):
        out = cache.step_keys([[int(k)] for k in trace[s0:s0 + 500]])
        if s0 >= 10000:
            hits += int((out["cls"] == O.HIT_T1).sum())
    measured = hits / (len(trace) - 10000)
    lo, hi = 0.0, 1e7
    for _ in range(200):   # characteristic time T: sum_i (1 - exp(-p_i T)) = c
        mid = (lo + hi) / 2
        if (1 - np.exp(-p * mid)).sum() < c:
            lo = mid
        else:
            hi = mid
    che = float((p * (1 - np.exp(-p * lo))).sum())
    assert abs(measured - che) < 0.015, (measured, che)


def test_scan_resistance_config4_shape():
    """one-shot traffic clears T1 but T2 survives -> ARC keeps the hot set, LRU is flushed."""
    rates = {}
    for policy in (O.POLICY_ARC, O.POLICY_LRU):
        rng = np.random.default_rng(50)
        c = 256
        cache = O.OracleCache(c, 16, policy)
        hot = [rng.integers(0, 32000, size=16 * 8, dtype=np.int32) for _ in range(16)]   # 128 hot blocks
        hits = acc = 0
        for step in range(120):
            reqs = []
            for _ in range(8):
                if rng.random() < 0.3:
                    reqs.append(rng.integers(0, 32000, size=16 * 64, dtype=np.int32))      # scan (<< c, as in D4: 1,024 of 65,536)
                else:
                    reqs.append(hot[int(rng.integers(0, 16))])
            tokens, offsets = W.pack_requests(reqs)
            out = cache.step(tokens, offsets)
            if step >= 20:
                hot_mask = np.repeat(np.diff(out["blk_off"]) == 8, np.diff(out["blk_off"]))
                hits += int(np.isin(out["cls"], HITS)[hot_mask].sum())
                acc += int(hot_mask.sum())
        rates[policy] = hits / acc
    assert rates[O.POLICY_ARC] > rates[O.POLICY_LRU] + 0.3, rates


def test_dbl_never_moves_p_and_equals_arc_without_resident_pressure():
    """DBL: p stays at c // 2 whatever is accessed; on a working set that fits the cache
    (no eviction ever) DBL, ARC and LRU agree on classes and block IDs."""
    rng = np.random.default_rng(77)
    c = 16
    dbl = O.OracleCache(c, 16, O.POLICY_DBL)
    for _ in range(300):
        out = dbl.step_keys([[int(k) for k in rng.integers(2, 60, size=int(rng.integers(1, 5)))]])
        assert set(out["p_after"].tolist()) <= {c // 2}
    assert dbl.stats()["p"] == c // 2
    a, d = O.OracleCache(c, 16, O.POLICY_ARC), O.OracleCache(c, 16, O.POLICY_DBL)
    for _ in range(200):
        req = [[int(k) for k in rng.integers(2, 2 + c, size=int(rng.integers(1, 4)))]]
        oa, od = a.step_keys(req), d.step_keys(req)
        for k in ("cls", "block_id", "evicted_id", "prefix_len"):
            assert np.array_equal(oa[k], od[k]), k


def test_windowed_zipf_generator_shape_and_shift():
    """NEXT-2 workload: 6 windows x 512 requests, deterministic, popularity reshuffled per window."""
    from paper_2606_21238_b200 import workloads as W

    tr = W.make_windowed_zipf(2048, seed=3, n_docs=50, mean_doc_tokens=1200.0)
    assert tr.info.n_requests == 3072 and len(tr.choice) == 3072
    tr2 = W.make_windowed_zipf(2048, seed=3, n_docs=50, mean_doc_tokens=1200.0)
    assert np.array_equal(tr.choice, tr2.choice) and W.trace_digest(tr, max_steps=40) == W.trace_digest(tr2, max_steps=40)
    tops = [int(np.bincount(tr.choice[w * 512:(w + 1) * 512], minlength=50).argmax()) for w in range(6)]
    assert len(set(tops)) >= 3                                   # the hot document changes between windows
    for w in range(6):                                           # inside a window the head of the Zipf law dominates
        cnt = np.sort(np.bincount(tr.choice[w * 512:(w + 1) * 512], minlength=50))[::-1]
        assert cnt[0] > 3 * cnt[9]
    # ARC tracks the shifts at least as well as LRU on this workload (oracle, small cache)
    rates = {}
    for pol in (O.POLICY_ARC, O.POLICY_LRU):
        oc = O.OracleCache(1024, 16, pol)
        for tok, off in W.make_windowed_zipf(1024, seed=3, n_docs=50, mean_doc_tokens=1200.0).steps():
            oc.step(tok, off, unpack=False)
        st = oc.stats()
        rates[pol] = (st["hit_t1"] + st["hit_t2"]) / st["accesses"]
    assert rates[O.POLICY_ARC] >= rates[O.POLICY_LRU] - 0.01, rates


def _keys(names, n):
    return [n.key(x) for x in names]


@pytest.mark.parametrize("impl", ["bf", "cpp"])
def test_step_wide_pins_hand_trace_G(impl):
    """NEXT-3, step-wide pin scope: c = 4, ARC.  Steps [X0..X3], [X0..X3], [Y0][Z0].  In the third step
    Z0's REPLACE prefers T1 (t1 = 1 > p = 0) whose only entry Y0 was brought in by an earlier request of the SAME step:
    under step-wide pins it is still pinned and the victim comes from T2 (X2); under the default request scope Y0 itself
    is evicted.  Derived by hand from R5/R7."""
    from helpers import KeyNames

    def make(scope):
        cch = BF.BruteForceCache(4) if impl == "bf" else O.OracleCache(4)
        if impl == "bf":
            cch.pin_scope = scope
        else:
            cch.set_pin_scope(scope)
        return cch

    for scope in (0, 1):
        n = KeyNames()
        cch = make(scope)
        X = _keys(["X0", "X1", "X2", "X3"], n)
        o1 = cch.step_keys([X])
        assert list(o1["block_id"]) == [3, 2, 1, 0] and list(o1["cls"]) == [0, 0, 0, 0]      # tail first: X3 gets ID 0
        o2 = cch.step_keys([X])
        assert list(o2["cls"]) == [1, 1, 1, 1] and list(o2["prefix_len"]) == [64]
        o3 = cch.step_keys([_keys(["Y0"], n), _keys(["Z0"], n)])
        assert list(o3["cls"]) == [0, 0]
        L = cch.lists()
        name = lambda lst: n.names(lst if impl == "bf" else lst[0])
        if scope == 1:
            assert list(o3["block_id"]) == [0, 1] and list(o3["evicted_id"]) == [0, 1]      # X3 then X2 leave T2
            assert name(L["T1"]) == ["Y0", "Z0"] and name(L["T2"]) == ["X1", "X0"] and name(L["B2"]) == ["X3", "X2"] and name(L["B1"]) == []
        else:
            assert list(o3["block_id"]) == [0, 0] and list(o3["evicted_id"]) == [0, 0]      # X3, then Y0 itself
            assert name(L["T1"]) == ["Z0"] and name(L["T2"]) == ["X2", "X1", "X0"] and name(L["B2"]) == ["X3"] and name(L["B1"]) == ["Y0"]
        # admission rule of the step scope: a step may pin at most c blocks; refused without a state change
        big = [_keys(["P0", "P1", "P2"], n), _keys(["Q0", "Q1"], n)]
        before = cch.lists()
        r = cch.step_keys(big)
        if scope == 1:
            assert r == O.ERR_REQUEST_TOO_LARGE
            after = cch.lists()
            assert all(list(np.asarray(before[k] if impl == "bf" else before[k][0])) == list(np.asarray(after[k] if impl == "bf" else after[k][0])) for k in ("T1", "T2", "B1", "B2"))
        else:
            assert isinstance(r, dict)


@pytest.mark.parametrize("policy", [0, 1, 2])
def test_step_wide_pins_differential_and_invariants(policy):
    rng = np.random.default_rng(300 + policy)
    for c in (2, 3, 5, 8):
        bf, cpp = BF.BruteForceCache(c, 16, policy), O.OracleCache(c, 16, policy)
        bf.pin_scope = 1
        cpp.set_pin_scope(1)
        for _ in range(300):
            reqs, left = [], c
            while left > 0 and rng.random() < 0.8:
                nb = int(rng.integers(1, min(left, 3) + 1))
                base = int(rng.integers(0, 4))
                reqs.append([1000 + 10 * base + i for i in range(nb)])       # shared prefixes
                left -= nb
            a, b = bf.step_keys(reqs), cpp.step_keys(reqs)
            for k in ("cls", "block_id", "evicted_id", "p_after", "prefix_len", "alloc_ids", "evict_ids"):
                assert list(a[k]) == b[k].tolist(), (c, policy, k)
            L = cpp.lists()
            check_invariants(L, c, policy_lru=(policy == 1))


# ---------------------------------------------------------------------------------------------------------------------
# NEXT-3, held pins with explicit release

def _make_held(impl, c, policy=0):
    cch = BF.BruteForceCache(c, 16, policy) if impl == "bf" else O.OracleCache(c, 16, policy)
    if impl == "bf":
        cch.pin_scope = 2
    else:
        cch.set_pin_scope(2)
    return cch


def _unheld(cch, impl, n):
    """names of the unheld entries of every list, LRU -> MRU"""
    L = cch.lists()
    if impl == "bf":
        return {k: n.names([x for x in L[k] if cch.holds.get(x, 0) == 0]) for k in ("T1", "T2", "B1", "B2")}
    return {k: n.names(L[k][0]) for k in ("T1", "T2", "B1", "B2")}


@pytest.mark.parametrize("impl", ["bf", "cpp"])
def test_held_pins_hand_trace_H(impl):
    """c = 4, ARC, pin scope 2.  Worked by hand from R5/R7 and the release rule of DESIGN.md §3.4: a block with holds is
    never a victim; a block re-enters at the MRU end of its list when its last hold is released, in the order of the
    release call; a step is refused when holds outstanding + its accesses exceed c."""
    from helpers import KeyNames

    n = KeyNames()
    cch = _make_held(impl, 4)
    A, B, Cq = _keys(["A0", "A1"], n), _keys(["B0", "B1"], n), _keys(["C0", "C1"], n)
    o = cch.step_keys([A])
    assert list(o["block_id"]) == [1, 0] and list(o["cls"]) == [0, 0]
    o = cch.step_keys([B])
    assert list(o["block_id"]) == [3, 2] and cch.hold_units() == 4
    assert cch.step_keys([_keys(["C0"], n)]) == O.ERR_REQUEST_TOO_LARGE          # 4 holds outstanding + 1 > c
    assert _unheld(cch, impl, n) == dict(T1=[], T2=[], B1=[], B2=[])
    assert cch.release([1, 0]) == 0 and cch.hold_units() == 2                    # A0 first, then A1
    assert _unheld(cch, impl, n)["T1"] == ["A0", "A1"]
    # T1 holds everything (t1 = c, no ghosts): case 4A-else evicts T1's first unheld entry without a ghost: A0, then A1
    o = cch.step_keys([Cq])
    assert list(o["cls"]) == [0, 0] and list(o["block_id"]) == [0, 1] and list(o["evicted_id"]) == [0, 1]
    assert cch.release([3, 2]) == 0 and cch.release([0, 1]) == 0 and cch.hold_units() == 0
    assert _unheld(cch, impl, n) == dict(T1=["B0", "B1", "C0", "C1"], T2=[], B1=[], B2=[])
    o = cch.step_keys([B])
    assert list(o["cls"]) == [1, 1] and list(o["prefix_len"]) == [32]
    assert _unheld(cch, impl, n) == dict(T1=["C0", "C1"], T2=[], B1=[], B2=[])   # B0, B1 are in T2 but held
    assert cch.release([3, 2]) == 0
    assert _unheld(cch, impl, n)["T2"] == ["B0", "B1"]
    o = cch.step_keys([_keys(["D0"], n)])                                        # REPLACE: t1 = 2 > p = 0 -> T1's LRU entry C0
    assert list(o["cls"]) == [0] and list(o["block_id"]) == [0] and list(o["evicted_id"]) == [0]
    assert _unheld(cch, impl, n) == dict(T1=["C1"], T2=["B0", "B1"], B1=["C0"], B2=[])
    assert cch.release([0]) == 0
    o = cch.step_keys([_keys(["B0"], n), _keys(["B0"], n)])                      # two requests hold the same block
    assert list(o["cls"]) == [2, 2] and list(o["prefix_len"]) == [16, 16] and cch.hold_units() == 2
    assert cch.release([3]) == 0 and cch.hold_units() == 1                       # one hold left: B0 stays out of reach
    assert _unheld(cch, impl, n)["T2"] == ["B1"]
    o = cch.step_keys([_keys(["E0", "E1"], n)])
    # E1: n = 5 >= c -> REPLACE takes C1 (ID 1) from T1;  E0: t1 + b1 = c -> drop B1's LRU ghost C0, REPLACE takes D0 (ID 0)
    assert list(o["cls"]) == [0, 0] and list(o["block_id"]) == [0, 1] and list(o["evicted_id"]) == [0, 1]
    assert _unheld(cch, impl, n) == dict(T1=[], T2=["B1"], B1=["C1", "D0"], B2=[])
    assert cch.release([3]) == 0
    assert _unheld(cch, impl, n)["T2"] == ["B1", "B0"]
    assert cch.release([3]) == O.ERR_INVALID_ARG                                 # nothing left to release: refused, no change
    assert cch.release([0, 1]) == 0 and cch.hold_units() == 0
    assert _unheld(cch, impl, n) == dict(T1=["E0", "E1"], T2=["B1", "B0"], B1=["C1", "D0"], B2=[])
    st = cch.stats if impl == "bf" else cch.stats()
    assert st["evict_t1"] == 5 and st["drop_b1"] == 1 and st["hit_t1"] == 2 and st["hit_t2"] == 2


@pytest.mark.parametrize("policy", [0, 1, 2])
def test_held_pins_released_in_access_order_equal_request_scope(policy):
    """If every request is released right after its own batch-1 step, tail block first (the access order R2), the held
    scope is the default scope: same outputs, same lists.  Pins the release rule to the already pinned R4 semantics."""
    rng = np.random.default_rng(410 + policy)
    for c in (3, 6, 16):
        ref, held = O.OracleCache(c, 16, policy), O.OracleCache(c, 16, policy)
        held.set_pin_scope(2)
        for _ in range(400):
            nb = int(rng.integers(1, min(c, 5) + 1))
            base = int(rng.integers(0, 6))
            req = [[5000 + 100 * base + i for i in range(nb)]]
            a, b = ref.step_keys(req), held.step_keys(req)
            for k in ("cls", "block_id", "evicted_id", "p_after", "prefix_len", "alloc_ids", "evict_ids"):
                assert a[k].tolist() == b[k].tolist(), (c, policy, k)
            assert held.release(b["block_id"][::-1]) == 0
            La, Lb = ref.lists(), held.lists()
            for k in ("T1", "T2", "B1", "B2"):
                assert La[k][0].tolist() == Lb[k][0].tolist() and La[k][1].tolist() == Lb[k][1].tolist(), (c, policy, k)


@pytest.mark.parametrize("policy", [0, 1, 2])
def test_held_pins_differential_and_invariants(policy):
    """Brute force against the C++ oracle under random steps and random releases (whole requests, in random order, some
    sharing blocks so that hold counts exceed one); held blocks are resident and never evicted."""
    rng = np.random.default_rng(500 + policy)
    for c in (3, 5, 9):
        bf, cpp = BF.BruteForceCache(c, 16, policy), O.OracleCache(c, 16, policy)
        bf.pin_scope = 2
        cpp.set_pin_scope(2)
        live = []                     # block-ID arrays of the requests not yet released
        for it in range(400):
            if live and (rng.random() < 0.5 or cpp.hold_units() > c - 2):
                k = int(rng.integers(0, len(live)))
                ids = live.pop(k)
                ids = ids[rng.permutation(len(ids))]
                if len(live) and rng.random() < 0.3:      # two requests in one call
                    ids = np.concatenate([ids, live.pop(int(rng.integers(0, len(live))))])
                assert bf.release(ids.tolist()) == 0 and cpp.release(ids) == 0
            else:
                reqs, left = [], c - cpp.hold_units()
                while left > 0 and rng.random() < 0.7:
                    nb = int(rng.integers(1, min(left, 3) + 1))
                    base = int(rng.integers(0, 4))
                    reqs.append([1000 + 10 * base + i for i in range(nb)])
                    left -= nb
                held_before = {x: h for x, h in bf.holds.items()}
                a, b = bf.step_keys(reqs), cpp.step_keys(reqs)
                for k in ("cls", "block_id", "evicted_id", "p_after", "prefix_len", "alloc_ids", "evict_ids"):
                    assert list(a[k]) == b[k].tolist(), (c, policy, k)
                off = b["blk_off"]
                for r in range(len(reqs)):
                    live.append(b["block_id"][off[r]:off[r + 1]].copy())
                resident = set(bf.T1) | set(bf.T2)
                assert set(held_before) <= resident, "a held block was evicted"
            assert bf.hold_units() == cpp.hold_units() == sum(len(x) for x in live)
            Lb, Lc = bf.lists(), cpp.lists()
            for k in ("T1", "T2", "B1", "B2"):
                assert [x for x in Lb[k] if bf.holds.get(x, 0) == 0] == Lc[k][0].tolist(), (c, policy, k, it)
            sc = cpp.stats()
            assert (len(bf.T1), len(bf.T2), len(bf.B1), len(bf.B2), bf.p) == (sc["t1"], sc["t2"], sc["b1"], sc["b2"], sc["p"])
        # over-releasing and unknown IDs are refused without a change
        before = cpp.lists()
        assert cpp.release(np.array([c + 5], np.int32)) == O.ERR_INVALID_ARG
        if live:
            twice = np.concatenate([live[0], live[0], live[0], live[0]])
            if cpp.release(twice) == O.ERR_INVALID_ARG:
                after = cpp.lists()
                assert all(before[k][0].tolist() == after[k][0].tolist() for k in ("T1", "T2", "B1", "B2"))
