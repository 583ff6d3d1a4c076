"""Hand-worked traces A-E (tests/golden/) replayed on both oracle implementations."""
import pytest

from helpers import KeyNames, parse_trace
from oracle import oracle as O
from oracle import oracle_bruteforce as BF


def _replay(trace_file, c, policy, impl, compare_lists=True, lru_classes=False):
    reqs = parse_trace(trace_file)
    names = KeyNames()
    cache = BF.BruteForceCache(c, 16, policy) if impl == "bf" else O.OracleCache(c, 16, policy)
    for r in reqs:
        keys = [names.key(k) for k in r["keys"]]
        out = cache.step_keys([keys])
        nb = len(keys)
        # fixture lines are in ACCESS order = block nb-1 first
        for j, acc in enumerate(r["accesses"]):
            i = nb - 1 - j
            assert r["keys"][i] == acc["key"]
            want_cls = acc["cls"]
            if lru_classes and want_cls == 2:
                want_cls = 1
            assert int(out["cls"][i]) == want_cls, (trace_file, acc)
            assert int(out["block_id"][i]) == acc["id"], (trace_file, acc)
            assert int(out["evicted_id"][i]) == acc["evicted"], (trace_file, acc)
            if policy in (0, 2):
                assert int(out["p_after"][i]) == acc["p"], (trace_file, acc)
        if r["prefix_len"] is not None:
            assert int(out["prefix_len"][0]) == r["prefix_len"]
        # the fixture gives the lists after every access; after the request's LAST access they must match
        if compare_lists and policy in (0, 2):
            L = cache.lists()
            got = [names.names(L[n] if impl == "bf" else L[n][0]) for n in ("T1", "T2", "B1", "B2")]
            assert got == r["accesses"][-1]["lists"], (trace_file, r["accesses"][-1])
            assert L["p"] == r["accesses"][-1]["p"]
        # alloc / evict lists in access order
        want_alloc = [a["id"] for a in r["accesses"] if a["cls"] not in (1, 2)]
        want_evict = [a["evicted"] for a in r["accesses"] if a["evicted"] >= 0]
        assert list(map(int, out["alloc_ids"])) == want_alloc
        assert list(map(int, out["evict_ids"])) == want_evict
    return cache


@pytest.mark.parametrize("impl", ["bf", "cpp"])
def test_trace_A(impl):
    _replay("trace_A.txt", 4, 0, impl)


@pytest.mark.parametrize("impl", ["bf", "cpp"])
@pytest.mark.parametrize("policy", [0, 1])
def test_trace_B(impl, policy):
    _replay("trace_B.txt", 4, policy, impl)


@pytest.mark.parametrize("impl", ["bf", "cpp"])
def test_trace_C(impl):
    _replay("trace_C.txt", 4, 0, impl)


@pytest.mark.parametrize("impl", ["bf", "cpp"])
def test_trace_D_and_E(impl):
    _replay("trace_DE.txt", 2, 0, impl)
    _replay("trace_DE.txt", 2, 1, impl, lru_classes=True)


@pytest.mark.parametrize("impl", ["bf", "cpp"])
def test_trace_F_dbl(impl):
    """DBL = ARC's lists and REPLACE with p frozen at c // 2."""
    _replay("trace_F.txt", 4, 2, impl)


def test_trace_F_intermediate_lists():
    reqs = parse_trace("trace_F.txt")
    names = KeyNames()
    for impl in ("bf", "cpp"):
        cache = BF.BruteForceCache(4, 16, 2) if impl == "bf" else O.OracleCache(4, 16, 2)
        for r in reqs:
            cache.step_keys([[names.key(r["keys"][0])]])
            L = cache.lists()
            got = [names.names(L[n] if impl == "bf" else L[n][0]) for n in ("T1", "T2", "B1", "B2")]
            assert got == r["accesses"][0]["lists"], r
            assert L["p"] == 2


def test_trace_A_intermediate_lists_bruteforce():
    """Trace A gives the lists after every single access; single-block requests let us check each line."""
    reqs = parse_trace("trace_A.txt")
    names = KeyNames()
    for impl in ("bf", "cpp"):
        cache = BF.BruteForceCache(4) if impl == "bf" else O.OracleCache(4)
        for r in reqs:
            cache.step_keys([[names.key(r["keys"][0])]])
            L = cache.lists()
            got = [names.names(L[n] if impl == "bf" else L[n][0]) for n in ("T1", "T2", "B1", "B2")]
            assert got == r["accesses"][0]["lists"]


def test_paper_b2_ghost_flow():
    """'A request for a KV block that appears in B2 is a miss ... ARC puts this KV block to the
    frequency cache T2, evicts the LRU block from T1. The combination of T1 and T2 is of fixed size.'"""
    cache = O.OracleCache(4)
    n = KeyNames()
    for ch in "a b c a d e b f g a d".split():
        cache.step_keys([[n.key(ch)]])
    before = cache.lists()
    assert n.key("b") in before["B2"][0].tolist()
    lru_of_t1 = int(before["T1"][0][0])
    out = cache.step_keys([[n.key("b")]])
    after = cache.lists()
    assert int(out["cls"][0]) == O.GHOST_B2                       # a miss (not a hit class)
    assert int(after["T2"][0][-1]) == n.key("b")                  # goes to T2 (MRU end)
    assert lru_of_t1 not in after["T1"][0].tolist()               # LRU of T1 evicted ...
    assert int(after["B1"][0][-1]) == lru_of_t1                   # ... into B1
    assert len(after["T1"][0]) + len(after["T2"][0]) == 4         # fixed combined size
