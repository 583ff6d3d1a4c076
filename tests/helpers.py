"""Shared test helpers (fixture parsing, invariant checks).  No method arithmetic: the invariant
checker only inspects list dumps; it never decides an access."""
from pathlib import Path

import numpy as np

CLASS = {"MISS": 0, "HIT_T1": 1, "HIT_T2": 2, "GHOST_B1": 3, "GHOST_B2": 4}
GOLDEN = Path(__file__).resolve().parent / "golden"


def parse_trace(name):
    """-> list of requests; each request = dict(keys=[names block0 first] or None, prefix_len, accesses=[...])
    where an access = dict(key, cls, id, evicted, p, lists=[T1,T2,B1,B2] as lists of names)."""
    reqs = []
    for line in (GOLDEN / name).read_text().splitlines():
        line = line.strip()
        if not line or line.startswith("#"):
            continue
        if line.startswith("req "):
            keys, plen = line[4:].split("->")
            reqs.append(dict(keys=keys.split(), prefix_len=int(plen), accesses=[]))
            continue
        head, *lists = line.split("|")
        key, cls, bid, evi, p = head.split()
        acc = dict(key=key, cls=CLASS[cls], id=int(bid), evicted=-1 if evi == "-" else int(evi), p=int(p),
                   lists=[l.split() for l in lists])
        if not reqs or (reqs[-1]["keys"] is None):
            reqs.append(dict(keys=None, prefix_len=None, accesses=[acc]))  # one block per request
        else:
            reqs[-1]["accesses"].append(acc)
    for r in reqs:
        if r["keys"] is None:
            r["keys"] = [r["accesses"][0]["key"]]
    return reqs


class KeyNames:
    """Stable mapping letter <-> 64-bit key (>= 2) for key-level traces."""

    def __init__(self):
        self.fwd, self.rev = {}, {}

    def key(self, name):
        if name not in self.fwd:
            k = 1000 + 7 * len(self.fwd)
            self.fwd[name] = k
            self.rev[k] = name
        return self.fwd[name]

    def names(self, keys):
        return [self.rev[int(k)] for k in keys]


def check_invariants(lists, c, policy_lru=False, pinned=()):
    """I1-I9 of SURVEY.md §8(c) on a dump {T1,T2,B1,B2: (keys, blocks), p, next_fresh}."""
    T1, T2, B1, B2 = (lists[n] for n in ("T1", "T2", "B1", "B2"))
    t1, t2, b1, b2 = (len(x[0]) for x in (T1, T2, B1, B2))
    p, nf = lists["p"], lists["next_fresh"]
    assert t1 + t2 <= c, "I1"
    assert t1 + b1 <= c, "I2"
    assert t1 + t2 + b1 + b2 <= 2 * c, "I3"
    assert 0 <= p <= c, "I4"
    allk = np.concatenate([T1[0], T2[0], B1[0], B2[0]])
    assert len(np.unique(allk)) == len(allk), "I5 lists disjoint, keys unique"
    res_ids = np.concatenate([T1[1], T2[1]])
    assert sorted(res_ids.tolist()) == list(range(nf)), "I6 resident IDs are exactly 0..next_fresh-1"
    assert nf <= c
    if t1 + t2 < c:
        assert b1 == 0 and b2 == 0, "I7 no ghosts before the cache is full"
        assert nf == t1 + t2
    assert all(b == -1 for b in np.concatenate([B1[1], B2[1]]).tolist()), "I8 ghosts hold no ID"
    resident = set(np.concatenate([T1[0], T2[0]]).tolist())
    assert set(pinned) <= resident, "I9 pinned are resident"
    if policy_lru:
        assert t2 == 0 and b1 == 0 and b2 == 0 and p == 0
