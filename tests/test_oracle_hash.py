"""Pins of the oracle's hash (H1-H6): survey vectors, closed form of the chain, bijectivity of the
per-word term, agreement of the two independent oracle implementations."""
import numpy as np
import pytest

from helpers import GOLDEN
from oracle import oracle as O
from oracle import oracle_bruteforce as BF

MASK = (1 << 64) - 1


def _vectors():
    rows = []
    for line in (GOLDEN / "hash_vectors.txt").read_text().splitlines():
        if line.strip() and not line.startswith("#"):
            rows.append([f.strip() for f in line.split(";")])
    return rows


def test_survey_vectors_both_oracles():
    for row in _vectors():
        if row[0] == "mix":
            z, want = int(row[1], 16), int(row[2], 16)
            assert BF.mix(z) == want
            want_key = want + 2 if want < 2 else want   # H5 reserved values
            assert O.key_from_state(z) == want_key
        elif row[0] == "kpow":
            assert pow(BF.K, int(row[1]), 1 << 64) == int(row[2], 16)
        else:
            toks = eval(row[1])
            want_keys = [int(x, 16) for x in row[3].split()]
            assert BF.block_keys(toks) == want_keys, row[0]
            keys, blk_off = O.hash_blocks(np.array(toks, np.int32), [0, len(toks)])
            assert keys.tolist() == want_keys, row[0]
            assert blk_off.tolist() == [0, len(want_keys)]
            if row[2] != "-":
                assert BF.content_hash(toks[:16]) == int(row[2], 16)
                assert O.content_hash(toks[:16]) == int(row[2], 16)


def test_reserved_key_rule():
    assert O.key_from_state(0) == 2                      # mix(0) = 0 -> key 2
    # mix is a bijection; invert it to find the state whose mix is 1 and check it maps to 3
    def unxorshift(z, s):
        r = z
        for _ in range(64 // s + 1):
            r = z ^ (r >> s)
        return r & MASK
    inv = lambda c: pow(c, -1, 1 << 64)
    z = unxorshift(1, 31)
    z = (z * inv(BF.C2)) & MASK
    z = unxorshift(z, 27)
    z = (z * inv(BF.C1)) & MASK
    z = unxorshift(z, 30)
    assert BF.mix(z) == 1
    assert O.key_from_state(z) == 3
    assert O.key_from_state(BF.S0) == BF.mix(BF.S0)


def test_chain_closed_form():
    """H4: s_i = K^(i+1) S0 + sum_{j<=i} K^(i-j) g_j, evaluated with Python pow, not with the loop."""
    rng = np.random.default_rng(1)
    toks = rng.integers(-2**31, 2**31, size=16 * 37 + 5, dtype=np.int64).astype(np.int32)
    keys, _ = O.hash_blocks(toks, [0, len(toks)])
    g = [O.content_hash(toks[16 * j:16 * j + 16]) for j in range(37)]
    for i in (0, 1, 2, 17, 36):
        s = pow(BF.K, i + 1, 1 << 64) * BF.S0
        for j in range(i + 1):
            s += pow(BF.K, i - j, 1 << 64) * g[j]
        assert int(keys[i]) == O.key_from_state(s & MASK)


def test_content_hash_definition_written_out():
    """H3 for one block, written as a single big-integer expression."""
    t = [5, 9, 2**31 - 1, -7, 0, 0, 123456, 42, 1, 2, 3, 4, 5, 6, 7, 8]
    u = [x & 0xFFFFFFFF for x in t]
    g = 0
    for k in range(8):
        e = (((u[2 * k] | (u[2 * k + 1] << 32)) + (k + 1) * 0x9E3779B97F4A7C15) * 0xBF58476D1CE4E5B9) % 2**64
        g = (g + (e ^ (e >> 32))) % 2**64
    assert O.content_hash(t) == g == BF.content_hash(t)


def test_single_word_difference_never_collides():
    """Each term of H3 is a bijection of w_k (odd multiplier, invertible fold), so two blocks that differ
    in exactly one word have different g."""
    rng = np.random.default_rng(2)
    base = rng.integers(0, 128000, size=16, dtype=np.int32)
    g0 = O.content_hash(base)
    seen = {g0}
    for trial in range(4000):
        b = base.copy()
        k = int(rng.integers(0, 8))
        b[2 * k] = rng.integers(0, 128000)
        b[2 * k + 1] = rng.integers(0, 128000)
        if (b == base).all():
            continue
        assert O.content_hash(b) != g0
    # position salt: permuting two different words changes g
    b = base.copy()
    b[[0, 1, 2, 3]] = base[[2, 3, 0, 1]]
    assert O.content_hash(b) != g0


def test_cpp_vs_bruteforce_random_requests():
    rng = np.random.default_rng(3)
    lens = [0, 1, 15, 16, 17, 31, 32, 33, 160, 1000, 7, 16 * 64 + 3]
    reqs = [rng.integers(-5, 200000, size=n).astype(np.int32) for n in lens]
    toks = np.concatenate(reqs)
    offs = np.concatenate([[0], np.cumsum(lens)])
    keys, blk_off = O.hash_blocks(toks, offs)
    want = [k for r in reqs for k in BF.block_keys(r.tolist())]
    assert keys.tolist() == want
    assert blk_off.tolist() == np.concatenate([[0], np.cumsum([n // 16 for n in lens])]).tolist()
    # a request's keys do not depend on where it sits in the batch (chain restarts at S0)
    k2, _ = O.hash_blocks(reqs[9], [0, len(reqs[9])])
    assert k2.tolist() == keys[blk_off[9]:blk_off[10]].tolist()


def test_prefix_property():
    """Two requests sharing a token prefix share exactly the keys of the shared full blocks."""
    rng = np.random.default_rng(4)
    doc = rng.integers(0, 32000, size=100, dtype=np.int32)   # 6 full blocks + 4 tokens
    a = np.concatenate([doc, rng.integers(0, 32000, size=40, dtype=np.int32)])
    b = np.concatenate([doc, rng.integers(0, 32000, size=40, dtype=np.int32)])
    ka, _ = O.hash_blocks(a, [0, len(a)])
    kb, _ = O.hash_blocks(b, [0, len(b)])
    assert ka[:6].tolist() == kb[:6].tolist()
    assert not set(ka[6:].tolist()) & set(kb[6:].tolist())


def test_hash_errors():
    assert O.lib().oracle_hash_blocks(None, None, 0, 16, None, None) == O.ERR_INVALID_ARG
    offs = np.array([0, 32, 16], np.int64)
    t = np.zeros(32, np.int32)
    assert O.lib().oracle_hash_blocks(O._ptr(t), O._ptr(offs), 2, 16, None, None) == O.ERR_INVALID_ARG
    offs = np.array([0, 32], np.int64)
    assert O.lib().oracle_hash_blocks(O._ptr(t), O._ptr(offs), 1, 15, None, None) == O.ERR_UNSUPPORTED


def test_resumed_chain_split_invariance_and_closed_form():
    """a request may continue a sequence at a block boundary from the H4 state returned for its earlier
    blocks.  (1) Splitting a prompt at ANY block boundary and resuming gives the keys of the unsplit prompt, and the
    same final state; tokens after the last full block never enter the state.  (2) The returned state is the closed form
    s K^n + sum_j K^(n-1-j) g_j in Python big integers.  Both oracle implementations."""
    rng = np.random.default_rng(77)
    for _ in range(60):
        nb = int(rng.integers(1, 40))
        tail = int(rng.integers(0, 16))
        tok = rng.integers(-2 ** 31, 2 ** 31, size=16 * nb + tail).astype(np.int32)
        off = np.array([0, len(tok)], np.int64)
        whole_keys, _ = O.hash_blocks(tok, off)
        oc = O.OracleCache(64)
        whole = oc.step(tok, off)
        g = [BF.content_hash(tok[16 * i:16 * i + 16].tolist()) for i in range(nb)]
        s = BF.S0
        for gi in g:
            s = (s * BF.K + gi) & MASK
        assert int(whole["chain_state"][0]) == s == (BF.S0 * pow(BF.K, nb, 1 << 64) + sum(pow(BF.K, nb - 1 - j, 1 << 64) * g[j] for j in range(nb))) & MASK
        cut = int(rng.integers(0, nb + 1))
        part_tail = int(rng.integers(0, 16)) if cut < nb else 0
        a = tok[:16 * cut + part_tail]                       # may end inside block `cut`: those tokens are not hashed yet
        b = tok[16 * cut:]                                   # the continuation starts again at the block boundary
        oa, ob = O.OracleCache(64), O.OracleCache(64)
        ra = oa.step(a, np.array([0, len(a)], np.int64))
        rb = ob.step(b, np.array([0, len(b)], np.int64), chain_in=ra["chain_state"])
        assert int(rb["chain_state"][0]) == s
        ka, _ = O.hash_blocks(a, np.array([0, len(a)], np.int64))
        kb_bf, sb_bf = BF.block_keys(b.tolist(), 16, int(ra["chain_state"][0]), True)
        assert sb_bf == s and BF.block_keys(a.tolist(), 16, BF.S0, True)[1] == int(ra["chain_state"][0])
        assert np.array_equal(np.concatenate([ka, np.array(kb_bf, np.uint64)]), whole_keys)
        # the C++ oracle's resumed keys, seen through the cache: after the whole prompt was served by `oc`, the
        # continuation's blocks are all hits there iff the keys are the same
        rc = oc.step(b, np.array([0, len(b)], np.int64), chain_in=ra["chain_state"])
        assert (rc["cls"] != 0).all() and rc["prefix_len"][0] == 16 * (nb - cut)


@pytest.mark.parametrize("policy", [0, 1, 2])
def test_resumed_requests_differential(policy):
    """Brute force against the C++ oracle on decode-shaped traffic: sequences grow by one or two blocks per step from
    their stored chain state while new prompts arrive; outputs and states agree."""
    rng = np.random.default_rng(80 + policy)
    for c in (4, 9):
        bf, cpp = BF.BruteForceCache(c, 16, policy), O.OracleCache(c, 16, policy)
        seqs = []                                            # (chain state, blocks so far)
        for _ in range(120):
            reqs, chain = [], []
            for i in range(len(seqs)):
                if rng.random() < 0.6:
                    reqs.append(rng.integers(0, 3, size=16 * int(rng.integers(1, 3)) + int(rng.integers(0, 16))).astype(np.int32))
                    chain.append(seqs[i])
                else:
                    reqs.append(np.zeros(0, np.int32))       # not scheduled this step
                    chain.append(seqs[i])
            n_old = len(reqs)
            if len(seqs) < 3 and rng.random() < 0.5:
                reqs.append(rng.integers(0, 3, size=16 * int(rng.integers(1, min(c, 3) + 1))).astype(np.int32))
                chain.append(BF.S0)
            off = np.zeros(len(reqs) + 1, np.int64)
            off[1:] = np.cumsum([len(r) for r in reqs])
            tok = np.concatenate(reqs) if reqs else np.zeros(0, np.int32)
            a = bf.step(tok.tolist(), off.tolist(), chain_in=chain)
            b = cpp.step(tok, off, chain_in=np.array(chain, np.uint64))
            for k in ("cls", "block_id", "evicted_id", "p_after", "prefix_len"):
                assert list(a[k]) == b[k].tolist(), (c, policy, k)
            assert [int(x) for x in a["chain_state"]] == [int(x) for x in b["chain_state"]]
            seqs = [int(x) for x in b["chain_state"]]
            if len(seqs) == 3 and rng.random() < 0.3:
                seqs.pop(int(rng.integers(0, 3)))            # a sequence finishes
