"""Randomised soak of the whole path on the GPU against the oracle: random cache sizes, policies, pin scopes (with
releases under held pins), K3 machines and request mixes drawn from a persistent prefix tree (shared prefixes between
consecutive requests, long and short requests, empty and duplicate requests).  Every output of every step, the
counters and the four lists.  A time budget per configuration keeps the file at about half a minute."""
import sys
import time
from pathlib import Path

import numpy as np
import pytest

if str(Path(__file__).resolve().parent.parent) not in sys.path:      # also runnable as a script (the long soak, see main)
    sys.path.insert(0, str(Path(__file__).resolve().parent.parent))

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

from oracle import oracle as O
from paper_2606_21238_b200 import workloads as W


@pytest.fixture(scope="module")
def A():
    if not torch.cuda.is_available():
        pytest.fail("-m gpu tests need a CUDA device")
    from paper_2606_21238_b200 import arc as A_

    A_.load_library()
    return A_


KEYS = ("prefix_len", "blk_off", "cls", "block_id", "evicted_id", "p_after", "alloc_ids", "evict_ids", "chain_state")
STAT = ("accesses", "hit_t1", "hit_t2", "ghost_b1", "ghost_b2", "miss", "evict_t1", "evict_t2", "drop_b1", "drop_b2", "t1", "t2", "b1", "b2", "p")

def tree_request(rng, table, nb):
    depth, br, B = table.shape
    path = rng.integers(0, br, size=nb)
    if rng.random() < 0.6:
        path[: min(nb, int(rng.integers(1, 40)))] = 0
    toks = [table[min(l, depth - 1), int(b)] for l, b in enumerate(path)]
    toks.append(rng.integers(0, 1000, size=int(rng.integers(0, 16)), dtype=np.int32))
    return np.concatenate(toks).astype(np.int32)

def run(A, seed, budget_s):
    rng = np.random.default_rng(seed)
    c = int(rng.choice([40, 300, 2000, 9000]))
    policy = int(rng.integers(0, 3)); scope = int(rng.choice([0, 0, 1, 2])); machine = int(rng.choice([0, 3, 3, 3, 2, 4, 4, 5]))
    depth = int(rng.integers(3, 40)); br = int(rng.choice([2, 3]))
    table = rng.integers(0, 1000, size=(depth, br, 16), dtype=np.int32)
    gc, oc = A.ArcCache(c, 16, policy), O.OracleCache(c, 16, policy)
    gc.set_machine(machine); gc.set_pin_scope(scope); oc.set_pin_scope(scope)
    live = []; t0 = time.time(); steps = 0
    while time.time() - t0 < budget_s:
        if scope == 2 and live and (rng.random() < 0.4 or oc.hold_units() > c * 0.7):
            ids = live.pop(int(rng.integers(0, len(live))))
            gc.release(ids); assert oc.release(ids) == 0
            continue
        budget = c if scope == 0 else (c if scope == 1 else c - oc.hold_units())
        reqs = []; left = budget if scope else 10 ** 9
        nreq = int(rng.integers(1, 40))
        for _ in range(nreq):
            mx = min(c, 700, left) if scope else min(c, 700)
            if mx < 1: break
            nb = int(rng.integers(1, mx + 1)) if rng.random() < 0.5 else int(rng.integers(1, min(mx, 30) + 1))
            r = tree_request(rng, table, nb)
            reqs.append(r); left -= len(r) // 16
        if rng.random() < 0.2: reqs.append(np.zeros(0, np.int32))
        if rng.random() < 0.2 and reqs: reqs.append(reqs[0])
        if scope and sum(len(r) // 16 for r in reqs) > budget: reqs = reqs[:1]
        tokens, offsets = W.pack_requests(reqs)
        o = oc.step(tokens, offsets)
        if isinstance(o, int):
            try:
                gc.step(torch.from_numpy(tokens).cuda(), offsets); raise AssertionError("gpu accepted a refused step")
            except A.ArcError as e:
                assert e.code == o
            continue
        g = gc.step(torch.from_numpy(tokens).cuda(), offsets).to_host()
        for k in KEYS:
            if not np.array_equal(g[k], o[k]):
                bad = np.flatnonzero(np.asarray(g[k]) != np.asarray(o[k]))[:5] if len(g[k]) == len(o[k]) else "len"
                raise AssertionError(f"seed {seed} c {c} p {policy} scope {scope} m {machine} step {steps}: {k} differs at {bad}")
        if scope == 2:
            off = o["blk_off"]
            live += [o["block_id"][off[r]:off[r + 1]].copy() for r in range(len(reqs)) if off[r + 1] > off[r]]
        steps += 1
        if steps % 20 == 0:
            gs, os_ = gc.stats(), oc.stats()
            assert all(gs[k] == os_[k] for k in STAT), (seed, steps)
            gl, ol = gc.debug_lists(), oc.lists()
            for n in ("T1", "T2", "B1", "B2"):
                assert np.array_equal(gl[n][0], ol[n][0]) and np.array_equal(gl[n][1], ol[n][1]), (seed, steps, n)
    gs, os_ = gc.stats(), oc.stats()
    assert all(gs[k] == os_[k] for k in STAT), seed
    d = gc.debug_counters()
    gc.close()
    return c, policy, scope, machine, steps, gs["accesses"], d["cut_conflict"], d["win_serial"], d["cut_twin"]



@pytest.mark.parametrize("seed", list(range(12)))
def test_soak_random_configuration(A, seed):
    c, policy, scope, machine, steps, accesses, cuts, serial, twins = run(A, 2000 + seed, 2.5)
    assert steps > 5 and accesses > 0


def main(argv=None):
    """A long soak with a record: python tests/test_gpu_soak.py --minutes 8 --seed0 5000 --out gpurun_out/soak.log
    One line per configuration (seed, cache size, policy, pin scope, K3 machine, steps, accesses, conflict cuts, by-the-book
    accesses, twin cuts); any difference from the oracle raises.  The logs of the round's soaks are in profiles/."""
    import argparse
    import sys
    from pathlib import Path

    sys.path.insert(0, str(Path(__file__).resolve().parent.parent))
    ap = argparse.ArgumentParser()
    ap.add_argument("--minutes", type=float, default=5.0)
    ap.add_argument("--seed0", type=int, default=5000)
    ap.add_argument("--per-config-s", type=float, default=8.0)
    ap.add_argument("--out", default=None)
    a = ap.parse_args(argv)
    from paper_2606_21238_b200 import arc as A_

    A_.load_library()
    log = open(a.out, "w") if a.out else None
    t0, seed, total = time.time(), a.seed0, 0
    head = "# seed c policy pin_scope machine steps accesses conflict_cuts by_the_book twin_cuts"
    print(head)
    if log:
        log.write(head + "\n")
    while time.time() - t0 < 60 * a.minutes:
        r = run(A_, seed, a.per_config_s)
        total += r[5]
        line = f"{seed} " + " ".join(str(x) for x in r)
        print(line, flush=True)
        if log:
            log.write(line + "\n")
            log.flush()
        seed += 1
    tail = f"# {seed - a.seed0} configurations, {total} accesses, {time.time() - t0:.0f} s, no difference from the oracle"
    print(tail)
    if log:
        log.write(tail + "\n")
        log.close()


if __name__ == "__main__":
    main()
