"""Whole-trace parity of the CUDA path against the CPU oracle on BASELINE.json's configs, by per-step digests.

    python tests/full_trace_parity.py --config 5 [--max-steps N] [--policy 0] [--out gpurun_out/full_trace_c5.log]

The trace is streamed once (never materialised); every step goes to the oracle and, through the C ABI, to the GPU; both
sides' outputs are hashed (SHA-256 over cls | block_id | evicted_id | p_after | prefix_len | alloc_ids | evict_ids) and
compared step by step; at the end the counters and the four lists (LRU -> MRU, keys and block IDs) are compared.  The
log keeps one line per 64 steps (a rolling digest over the window, equal on both sides by then) and the summary: steps,
accesses, wall time, hit rates of the whole trace and after the first 10 % of the requests, final and mean t1 / c.
Needs a CUDA device; the oracle is test infrastructure (this file lives under tests/).  profiles/r02_full_trace_parity.md
holds the logs of the runs of configs 4 and 5 (1,954 steps each).
"""
from __future__ import annotations

import argparse
import hashlib
import sys
import time
from pathlib import Path

import numpy as np

ROOT = Path(__file__).resolve().parent.parent
if str(ROOT) not in sys.path:
    sys.path.insert(0, str(ROOT))

KEYS = ("cls", "block_id", "evicted_id", "p_after", "prefix_len", "alloc_ids", "evict_ids")
STAT_KEYS = ("steps", "requests", "tokens_seen", "tokens_hashed", "accesses", "hit_t1", "hit_t2", "ghost_b1", "ghost_b2", "miss", "evict_t1",
             "evict_t2", "drop_b1", "drop_b2", "fresh_ids_used", "prefix_hit_tokens", "t1", "t2", "b1", "b2", "p")


def digest(out) -> bytes:
    h = hashlib.sha256()
    for k in KEYS:
        h.update(np.ascontiguousarray(out[k]).tobytes())
    return h.digest()


def run(config: int, max_steps=None, policy: int = 0, seed: int = 0, log=None, reserve: bool = True):
    import torch

    from oracle import oracle as O
    from paper_2606_21238_b200 import arc as A
    from paper_2606_21238_b200 import workloads as W

    if not torch.cuda.is_available():
        raise SystemExit("needs a CUDA device (no CPU fallback)")
    A.load_library()
    tr = W.make_trace(config, seed=seed)
    c = tr.info.capacity_blocks
    n_total = tr.info.n_steps if max_steps is None else min(max_steps, tr.info.n_steps)
    cut = max(1, int(np.ceil(0.1 * n_total))) - 1
    gc, oc = A.ArcCache(c, 16, policy), O.OracleCache(c, 16, policy)
    if reserve:
        gc.reserve(tr.info.requests_per_step, {1: 400, 2: 30000, 3: 30000, 4: 140000, 5: 420000}[config])
    say = (lambda s: (print(s, flush=True), log.write(s + "\n"), log.flush())) if log else (lambda s: print(s, flush=True))
    say(f"# config {config} ({tr.info.name}) policy {policy} seed {seed}: c = {c}, {tr.info.requests_per_step} requests/step, {n_total} steps")
    t0 = time.time()
    roll_g, roll_o = hashlib.sha256(), hashlib.sha256()
    n_acc = bad = 0
    t1_sum, snap = 0.0, None
    t_gpu = t_cpu = 0.0
    for i, (tokens, offsets) in enumerate(tr.steps(max_steps=max_steps)):
        ta = time.time()
        g = gc.step(torch.from_numpy(tokens).cuda(), offsets).to_host()
        tb = time.time()
        o = oc.step(tokens, offsets)
        tc = time.time()
        t_gpu += tb - ta
        t_cpu += tc - tb
        dg, do = digest(g), digest(o)
        roll_g.update(dg)
        roll_o.update(do)
        n_acc += int(o["n_access"])
        if dg != do:
            bad += 1
            diff = [k for k in KEYS if not np.array_equal(g[k], o[k])]
            say(f"step {i}: DIGESTS DIFFER in {diff}")
            if bad >= 3:
                break
        if i % 16 == 0 or i == cut:
            st = gc.stats()
            t1_sum += st["t1"] / c
            if i == cut:
                snap = st
        if (i + 1) % 64 == 0 or i + 1 == n_total:
            say(f"steps {i + 1 - ((i % 64) + 1):5d}..{i:5d}  accesses so far {n_acc:11d}  rolling gpu {roll_g.hexdigest()[:16]}  oracle {roll_o.hexdigest()[:16]}  "
                f"{'equal' if roll_g.digest() == roll_o.digest() else 'DIFFERENT'}  [{time.time() - t0:6.0f} s]")
    gs, os_ = gc.stats(), oc.stats()
    stats_equal = all(gs[k] == os_[k] for k in STAT_KEYS)
    gl, ol = gc.debug_lists(), oc.lists()
    lists_equal = all(np.array_equal(gl[n][0], ol[n][0]) and np.array_equal(gl[n][1], ol[n][1]) for n in ("T1", "T2", "B1", "B2"))
    dbg = gc.debug_counters()
    acc, hit = gs["accesses"], gs["hit_t1"] + gs["hit_t2"]
    say(f"# done: {i + 1} steps, {n_acc} accesses, {bad} steps with different digests, counters equal: {stats_equal}, lists equal: {lists_equal}")
    say(f"# wall {time.time() - t0:.0f} s (gpu step + copy back {t_gpu:.0f} s, oracle {t_cpu:.0f} s, the rest is trace generation and hashing)")
    say(f"# block hit rate whole trace {hit / max(1, acc):.4f}, prefix-token hit rate {gs['prefix_hit_tokens'] / max(1, gs['tokens_seen']):.4f}")
    if snap:
        a2, h2 = acc - snap["accesses"], hit - snap["hit_t1"] - snap["hit_t2"]
        say(f"# after the first 10 % of the requests: block hit rate {h2 / max(1, a2):.4f}, prefix-token hit rate "
            f"{(gs['prefix_hit_tokens'] - snap['prefix_hit_tokens']) / max(1, gs['tokens_seen'] - snap['tokens_seen']):.4f}")
    say(f"# t1/c final {gs['t1'] / c:.4f}, mean (every 16th step) {t1_sum / max(1, (i // 16) + 1):.4f}; p/c final {gs['p'] / c:.4f}; "
        f"t1 {gs['t1']} t2 {gs['t2']} b1 {gs['b1']} b2 {gs['b2']}")
    say(f"# K3 windows: all-hit {dbg['win_hit']}, general {dbg['win_general']}, by-the-book accesses {dbg['win_serial']}, conflict cuts {dbg['cut_conflict']}, twin cuts {dbg['cut_twin']}")
    gc.close()
    oc.close()
    return bad == 0 and stats_equal and lists_equal and roll_g.digest() == roll_o.digest()


def main(argv=None):
    ap = argparse.ArgumentParser(description=__doc__)
    ap.add_argument("--config", type=int, required=True)
    ap.add_argument("--max-steps", type=int, default=None)
    ap.add_argument("--policy", type=int, default=0)
    ap.add_argument("--seed", type=int, default=0)
    ap.add_argument("--out", default=None)
    a = ap.parse_args(argv)
    log = open(a.out, "w") if a.out else None
    ok = run(a.config, a.max_steps, a.policy, a.seed, log)
    if log:
        log.close()
    raise SystemExit(0 if ok else 1)


if __name__ == "__main__":
    main()
