"""Hit-rate / adaptation report on the paper-shaped windowed-Zipf workload.

    python -m paper_2606_21238_b200.report [--cache-tokens 30000 100000 200000 300000] [--seed 0] [--out report.json]

For every cache size (given in tokens as in the paper; blocks = tokens / 16) and every policy
(ARC, LRU, DBL) the 3,072-request trace (6 windows x 512, Zipf 1.0, popularity reshuffled per window) is
run through the CUDA library one request per step (the paper's batch size 1) and the report gives: block hit rate and
prefix-token hit rate over the whole trace and after the first window (warm-up split), and the
T1 ratio t1 / c after every request (the quantity of PAPER.md:141-149, Fig. 7).  Needs a CUDA device.
"""
from __future__ import annotations

import argparse
import json
import sys

import numpy as np


def run(cache_tokens, seed=0, policies=(0, 1, 2), requests_per_step=1, sample_every=16):
    import torch

    from . import arc as A
    from . import workloads as W

    names = {0: "ARC", 1: "LRU", 2: "DBL"}
    out = {"workload": "windowed Zipf: 6 windows x 512 requests, s = 1.0, 381 synthetic documents of about 5k tokens", "seed": seed, "runs": []}
    for tokens in cache_tokens:
        c = max(1, int(tokens) // 16)
        for pol in policies:
            tr = W.make_windowed_zipf(c, seed=seed, requests_per_step=requests_per_step)
            cache = A.ArcCache(c, 16, pol)
            warm = None
            t1_ratio, p_ratio = [], []
            for i, (tok, off) in enumerate(tr.steps()):
                if int((np.diff(off) // 16).max(initial=0)) > c:
                    continue                                   # a document larger than the cache cannot be pinned (R4): skipped
                cache.step(torch.from_numpy(tok).cuda(), off)
                if (i + 1) * requests_per_step == tr.window:
                    warm = cache.stats()
                if i % sample_every == 0:
                    st = cache.stats()
                    t1_ratio.append(round(st["t1"] / c, 4))
                    p_ratio.append(round(st["p"] / c, 4))
            st = cache.stats()
            acc, hit = st["accesses"], st["hit_t1"] + st["hit_t2"]
            rec = {"cache_tokens": int(tokens), "capacity_blocks": c, "policy": names[pol], "requests": st["requests"],
                   "block_hit_rate": hit / max(1, acc), "prefix_token_hit_rate": st["prefix_hit_tokens"] / max(1, st["tokens_seen"]),
                   "t1_ratio_every_%d_requests" % (sample_every * requests_per_step): t1_ratio,
                   "p_over_c": p_ratio, "t1_ratio_median": float(np.median(t1_ratio)) if t1_ratio else None}
            if warm is not None:
                a2, h2 = acc - warm["accesses"], hit - warm["hit_t1"] - warm["hit_t2"]
                rec["block_hit_rate_after_first_window"] = h2 / max(1, a2)
            out["runs"].append(rec)
            cache.close()
    return out


def main(argv=None):
    ap = argparse.ArgumentParser(description=__doc__)
    ap.add_argument("--cache-tokens", type=int, nargs="+", default=[30000, 100000, 200000, 300000])
    ap.add_argument("--seed", type=int, default=0)
    ap.add_argument("--out", default=None)
    a = ap.parse_args(argv)
    rep = run(a.cache_tokens, a.seed)
    text = json.dumps(rep)
    if a.out:
        with open(a.out, "w") as f:
            f.write(text)
    for r in rep["runs"]:
        print(f"{r['cache_tokens']:>8} tokens  {r['policy']:3}  block hit {100 * r['block_hit_rate']:6.2f} %  prefix-token hit {100 * r['prefix_token_hit_rate']:6.2f} %  "
              f"after window 1 {100 * r.get('block_hit_rate_after_first_window', 0):6.2f} %  median t1/c {r['t1_ratio_median']}", file=sys.stderr)
    if not a.out:
        print(text)


if __name__ == "__main__":
    main()
