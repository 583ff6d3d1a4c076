"""Brute-force reference of the prefix-KV lookup + ARC update.  TEST INFRASTRUCTURE ONLY.

Only `tests/`, `__graft_entry__.smoke()` and `bench.py`'s cpu_baseline / `--impl reference`
legs may import anything under `oracle/`.  Nothing here is shared with the CUDA path.

This file is the *slowest and plainest* statement of the method: four Python lists and a
set of pinned keys; sizes are recomputed with `len`, membership is searched with `in`,
every integer is a Python big integer reduced mod 2**64 by hand.  It exists to pin
`arc_oracle.cpp` (differential test on tiny caches, SURVEY.md §8(c) pin 3) and is itself
pinned by the hand-worked traces A-E (tests/golden/), the invariants I1-I12 and the LRU
stack-distance closed form.

What it follows
---------------
* Structure: L1 = T1 + B1 (seen once), L2 = T2 + B2 (seen at least twice); T1, T2 hold
  KV blocks in memory, B1, B2 hold only metadata of evicted blocks; the combined size of
  T1 and T2 is fixed.
* Ghost-hit flow: a request for a block in B2 is a miss, the block is regenerated, put in
  T2, and the LRU block of T1 is evicted; hits in B1 mean "invest more space in T1"
  (PAPER.md:60).
* Eviction is at KV-block level, blocks of e.g. 16 tokens.
* LRU baseline = naive vLLM eviction.
* The case analysis itself is deferred by the paper to Megiddo & Modha, FAST'03
  (PAPER.md:60, :183); it is restated as rules R1-R12 in SURVEY.md §8(c) / DESIGN.md §3 and
  followed here rule by rule.  Block-level details the paper leaves open (hash H1-H6,
  tail-first order R2, per-request pins R4, integer p R6, block IDs R8) are the readings
  listed in DESIGN.md §4.

Parity pins for every function here: see DESIGN.md §5.  None is "parity unpinned".
"""

MASK = (1 << 64) - 1

# ---- hash H1-H6 (fixed by this build, the paper names no hash) -------------
M = 0x9E3779B97F4A7C15
C1 = 0xBF58476D1CE4E5B9
C2 = 0x94D049BB133111EB
K = 0xD1342543DE82EF95
S0 = 0x243F6A8885A308D3


def mix(z):
    """H5 finaliser."""
    z &= MASK
    z ^= z >> 30
    z = (z * C1) & MASK
    z ^= z >> 27
    z = (z * C2) & MASK
    z ^= z >> 31
    return z


def fold(e):
    return (e ^ (e >> 32)) & MASK


def content_hash(block_tokens):
    """H2 + H3: g = sum_k fold((w_k + (k+1) M) C1), w_k = t[2k] | t[2k+1] << 32 (tokens as uint32)."""
    assert len(block_tokens) % 2 == 0
    g = 0
    for k in range(len(block_tokens) // 2):
        lo = int(block_tokens[2 * k]) & 0xFFFFFFFF  # H1: int32 reinterpreted as uint32
        hi = int(block_tokens[2 * k + 1]) & 0xFFFFFFFF
        w = lo | (hi << 32)
        e = ((w + (k + 1) * M) * C1) & MASK
        g = (g + fold(e)) & MASK
    return g


def block_keys(tokens, block_size=16, s=S0, return_state=False):
    """H4-H6: keys of the full blocks of one request, block 0 first.  s: the chain state before block 0 (S0 for a prompt,
    or the state returned for the sequence's earlier blocks: a request that continues at a block boundary)."""
    keys = []
    for i in range(len(tokens) // block_size):  # H6: only full blocks
        g = content_hash(tokens[i * block_size:(i + 1) * block_size])
        s = (s * K + g) & MASK  # H4
        key = mix(s)
        if key < 2:  # H5: 0 and 1 are reserved
            key += 2
        keys.append(key)
    return (keys, s) if return_state else keys


# ---- classes / codes (numbers fixed by the C ABI contract) ----------------
MISS, HIT_T1, HIT_T2, GHOST_B1, GHOST_B2 = 0, 1, 2, 3, 4
POLICY_ARC, POLICY_LRU, POLICY_DBL = 0, 1, 2   # DBL: ARC's lists with p frozen at c // 2
OK, ERR_INVALID_ARG, ERR_UNSUPPORTED, ERR_REQUEST_TOO_LARGE = 0, -1, -2, -3


class BruteForceCache:
    """Lists are Python lists written LRU -> MRU (index 0 is the LRU end)."""

    def __init__(self, capacity_blocks, block_size=16, policy=POLICY_ARC):
        assert capacity_blocks >= 1 and block_size % 2 == 0
        self.c, self.B, self.policy = capacity_blocks, block_size, policy
        self.T1, self.T2, self.B1, self.B2 = [], [], [], []
        self.p = capacity_blocks // 2 if policy == POLICY_DBL else 0
        self.block_of = {}  # resident key -> block ID (ghosts hold no ID, I8)
        self.next_fresh = 0
        self.pinned = set()
        self.pin_scope = 0  # 0: pins end with their request (R4); 1: with the step (NEXT-3); 2: held (§3.4)
        self.holds = {}  # scope 2: resident key -> accesses not yet released (absent = 0)
        self.stats = dict(steps=0, requests=0, tokens_seen=0, tokens_hashed=0, accesses=0, hit_t1=0, hit_t2=0,
                          ghost_b1=0, ghost_b2=0, miss=0, evict_t1=0, evict_t2=0, drop_b1=0, drop_b2=0,
                          fresh_ids_used=0, prefix_hit_tokens=0)

    # -- R7 -------------------------------------------------------------------------------
    def _first_unpinned(self, lst):
        for x in lst:  # from the LRU end
            if x not in self.pinned and self.holds.get(x, 0) == 0:
                return x
        return None

    def _replace(self, in_b2):
        t1 = len(self.T1)
        prefer_t1 = t1 >= 1 and (t1 > self.p or (in_b2 and t1 == self.p))
        order = [(self.T1, self.B1, "evict_t1"), (self.T2, self.B2, "evict_t2")]
        if not prefer_t1:
            order.reverse()
        for res, ghost, stat in order:
            v = self._first_unpinned(res)
            if v is not None:
                res.remove(v)
                ghost.append(v)  # MRU end of B1 / B2
                self.stats[stat] += 1
                return self.block_of.pop(v)  # the victim loses its block ID, which is returned
        raise AssertionError("no unpinned victim: violates R4 (nb_r <= c)")

    # -- R5 / R10: one access; returns (class, block_id, evicted_id) ----------------------------
    def access(self, x):
        c = self.c
        st = self.stats
        st["accesses"] += 1
        evicted = -1
        if self.policy == POLICY_LRU:  # R10: one list (reported as T1), no ghosts, p = 0
            if x in self.T1:
                st["hit_t1"] += 1
                self.T1.remove(x)
                self.T1.append(x)
                cls = HIT_T1
            else:
                st["miss"] += 1
                cls = MISS
                if len(self.T1) < c:
                    v = self.next_fresh
                    self.next_fresh += 1
                    st["fresh_ids_used"] += 1
                else:
                    victim = self._first_unpinned(self.T1)
                    assert victim is not None
                    self.T1.remove(victim)
                    v = evicted = self.block_of.pop(victim)
                    st["evict_t1"] += 1
                self.T1.append(x)
                self.block_of[x] = v
            self._pin(x)
            return cls, self.block_of[x], evicted

        t1, t2, b1, b2 = len(self.T1), len(self.T2), len(self.B1), len(self.B2)  # read before any change
        if x in self.T1 or x in self.T2:  # case 1
            if x in self.T1:
                cls = HIT_T1
                st["hit_t1"] += 1
                self.T1.remove(x)
            else:
                cls = HIT_T2
                st["hit_t2"] += 1
                self.T2.remove(x)
            self.T2.append(x)
        elif x in self.B1:  # case 2
            cls = GHOST_B1
            st["ghost_b1"] += 1
            delta = max(1, b2 // b1)
            if self.policy != POLICY_DBL:  # DBL: no adaptation
                self.p = min(c, self.p + delta)
            v = evicted = self._replace(False)
            self.B1.remove(x)
            self.T2.append(x)
            self.block_of[x] = v
        elif x in self.B2:  # case 3
            cls = GHOST_B2
            st["ghost_b2"] += 1
            delta = max(1, b1 // b2)
            if self.policy != POLICY_DBL:
                self.p = max(0, self.p - delta)
            v = evicted = self._replace(True)
            self.B2.remove(x)
            self.T2.append(x)
            self.block_of[x] = v
        else:  # case 4
            cls = MISS
            st["miss"] += 1
            if t1 + b1 == c:  # (A)
                if t1 < c:
                    self.B1.pop(0)
                    st["drop_b1"] += 1
                    v = evicted = self._replace(False)
                else:  # B1 empty, T1 holds everything: evict without making a ghost
                    victim = self._first_unpinned(self.T1)
                    assert victim is not None
                    self.T1.remove(victim)
                    v = evicted = self.block_of.pop(victim)
                    st["evict_t1"] += 1
            else:  # (B)
                n = t1 + t2 + b1 + b2
                if n >= c:
                    if n == 2 * c:
                        self.B2.pop(0)
                        st["drop_b2"] += 1
                    v = evicted = self._replace(False)
                else:
                    v = self.next_fresh
                    self.next_fresh += 1
                    st["fresh_ids_used"] += 1
            self.T1.append(x)
            self.block_of[x] = v
        self._pin(x)  # R4
        return cls, self.block_of[x], evicted

    def _pin(self, x):
        if self.pin_scope == 2:
            self.holds[x] = self.holds.get(x, 0) + 1  # held until released: one hold per access
        else:
            self.pinned.add(x)

    # -- scope 2: one hold back per listed block ID, in order; at zero the block goes to the MRU end
    def release(self, block_ids):
        key_of = {b: x for x, b in self.block_of.items()}
        left = dict(self.holds)
        for b in block_ids:  # check everything first: a bad ID fails the call with no change
            x = key_of.get(int(b))
            if x is None or left.get(x, 0) == 0:
                return ERR_INVALID_ARG
            left[x] -= 1
        for b in block_ids:
            x = key_of[int(b)]
            self.holds[x] -= 1
            if self.holds[x] == 0:
                del self.holds[x]
                lst = self.T1 if x in self.T1 else self.T2
                lst.remove(x)
                lst.append(x)
        return 0

    def hold_units(self):
        return sum(self.holds.values())

    # -- R2, R3, R4, R9: one step over lists of keys (block 0 first inside each request) ----------
    def step_keys(self, requests_keys):
        """requests_keys: list of lists of keys.  Returns a dict of per-step outputs (8(b))."""
        for keys in requests_keys:
            if len(keys) > self.c:
                return ERR_REQUEST_TOO_LARGE  # R11: no state change
        if self.pin_scope == 1 and sum(len(k) for k in requests_keys) > self.c:
            return ERR_REQUEST_TOO_LARGE  # step-wide pins: the step may pin at most c blocks (admission rule)
        if self.pin_scope == 2 and self.hold_units() + sum(len(k) for k in requests_keys) > self.c:
            return ERR_REQUEST_TOO_LARGE  # held: holds outstanding plus the step's accesses may not exceed c
        out = dict(prefix_len=[], blk_off=[0], cls=[], block_id=[], evicted_id=[], p_after=[], alloc_ids=[], evict_ids=[])
        for keys in requests_keys:  # R2: requests in ascending index
            nb = len(keys)
            cls = [0] * nb
            bid = [0] * nb
            evi = [0] * nb
            paf = [0] * nb
            for i in range(nb - 1, -1, -1):  # R2: tail first, block 0 last
                cls[i], bid[i], evi[i] = self.access(keys[i])
                paf[i] = self.p
                if cls[i] not in (HIT_T1, HIT_T2):
                    out["alloc_ids"].append(bid[i])
                if evi[i] >= 0:
                    out["evict_ids"].append(evi[i])
            if self.pin_scope == 0:
                self.pinned.clear()  # R4: all pins of the request drop together
            lead = 0
            while lead < nb and cls[lead] in (HIT_T1, HIT_T2):  # R9
                lead += 1
            out["prefix_len"].append(lead * self.B)
            self.stats["prefix_hit_tokens"] += lead * self.B
            out["blk_off"].append(out["blk_off"][-1] + nb)
            out["cls"] += cls
            out["block_id"] += bid
            out["evicted_id"] += evi
            out["p_after"] += paf
        self.pinned.clear()  # step-wide scope: all pins of the step drop together
        self.stats["steps"] += 1
        self.stats["requests"] += len(requests_keys)
        return out

    def step(self, tokens, offsets, chain_in=None):
        """Same on token IDs: tokens is a flat sequence, offsets has n_req+1 entries; chain_in[r] = the chain state request
        r continues from (None: new prompts).  The outputs then carry chain_state[r], the state after r's last full block."""
        n_req = len(offsets) - 1
        for r in range(n_req):
            if offsets[r + 1] < offsets[r] or offsets[0] < 0:
                return ERR_INVALID_ARG
        pairs = [block_keys(tokens[offsets[r]:offsets[r + 1]], self.B, S0 if chain_in is None else int(chain_in[r]), True)
                 for r in range(n_req)]
        reqs = [k for k, _ in pairs]
        out = self.step_keys(reqs)
        if isinstance(out, dict):
            out["chain_state"] = [st for _, st in pairs]
            self.stats["tokens_seen"] += int(offsets[n_req] - offsets[0])
            self.stats["tokens_hashed"] += self.B * sum(len(k) for k in reqs)
        return out

    def lists(self):
        return dict(T1=list(self.T1), T2=list(self.T2), B1=list(self.B1), B2=list(self.B2), p=self.p)
