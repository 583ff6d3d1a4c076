#!/usr/bin/env python
"""bench.py - the driver's benchmark contract for the arc_step hot path.

One "step" = one arc_step (K1 chained block hashing, K2 directory probe + reserve, K3 ARC state
machine, K4 finalize) over one scheduler batch of a seeded synthetic trace.  Default workload:
BASELINE.json configs[1] (document-QA shaped: c = 8,192 blocks x 16 tokens, 64 requests per step).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config 2] [--impl ours|reference]

Prints ONE JSON line (rank 0).  Keys beyond the base contract:
  value            block accesses/s, steps enqueued back to back on one stream, tokens resident in HBM
  tokens_hashed_per_s, requests_per_s   the same timed region in the metric's other units
  e2e              the same metric through arc_step_host (pinned HOST tokens in, results out, per step)
  roofline         K1 (the HBM-bound kernel) through arc_hash_blocks on >= 1 GiB of D5-shaped requests
  kernels          per-kernel device time of the timed steps (CUDA events between the kernels, separate pass)
  hit_rate         ARC vs LRU on the same steps
  cpu_baseline     the CPU oracle, as it stands, one thread, on the same steps
Multi-GPU (--gpus N under torchrun): replicas only: every rank runs its own cache on its
own seeded trace, no data-path collective; value = sum of accesses / max over ranks of the device time.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time
from pathlib import Path

import numpy as np

ROOT = Path(__file__).resolve().parent
if str(ROOT) not in sys.path:
    sys.path.insert(0, str(ROOT))

METRIC = "arc_block_accesses_per_s"
UNIT = "accesses/s"
ALGO_BYTES_PER_BLOCK = 72          # K1: 64 B of tokens read + 8 B key written


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=600)
    ap.add_argument("--warmup", type=int, default=30)
    ap.add_argument("--config", type=int, default=2, help="BASELINE.json configs index + 1 (default 2 = doc-QA)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--seed", type=int, default=0)
    ap.add_argument("--bulk-gib", type=float, default=1.0, help="size of the K1 roofline run in GiB of tokens")
    ap.add_argument("--no-extras", action="store_true", help="skip the breakdown / roofline / hit-rate / cpu legs")
    ap.add_argument("--only-k1", action="store_true", help="run only the K1 bulk roofline leg (for ncu captures of the hashing kernel)")
    return ap.parse_args()


def peaks():
    p = ROOT / "MEASURED_PEAKS.json"
    if p.exists():
        try:
            return float(json.loads(p.read_text())["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md)"


def build_steps(config: int, n_steps: int, seed: int):
    """The first n_steps steps of the config's trace: list of (tokens int32, offsets int64)."""
    from paper_2606_21238_b200 import workloads as W

    tr = W.make_trace(config, seed=seed)
    steps = list(tr.steps(max_steps=n_steps))
    if len(steps) < n_steps:
        raise SystemExit(f"config {config} has only {len(steps)} steps; lower --steps/--warmup")
    return tr.info, steps


def step_counts(steps, B=16):
    acc = [int((np.diff(o) // B).sum()) for _, o in steps]
    tok = [int(o[-1] - o[0]) for _, o in steps]
    req = [len(o) - 1 for _, o in steps]
    return acc, tok, req


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 200 ms while the timed region runs."""

    Q = "clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown," \
        "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap"

    def __init__(self, index: int):
        self.index, self.rows, self._stop, self._t = index, [], threading.Event(), None

    def _run(self):
        while not self._stop.is_set():
            try:
                out = subprocess.run(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}", "--format=csv,noheader,nounits"],
                                     capture_output=True, text=True, timeout=5).stdout.strip()
                if out:
                    self.rows.append([x.strip() for x in out.splitlines()[0].split(",")])
            except Exception:
                pass
            self._stop.wait(0.05)

    def __enter__(self):
        self._t = threading.Thread(target=self._run, daemon=True)
        self._t.start()
        return self

    def __exit__(self, *a):
        self._stop.set()
        self._t.join(timeout=6)

    def summary(self):
        if not self.rows:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["unsampled"]}
        sm = sorted(float(r[0]) for r in self.rows if r[0].replace(".", "").isdigit())
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [n for i, n in enumerate(names) if any(len(r) > 3 + i and r[3 + i].lower().startswith("active") for r in self.rows)]
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": float(self.rows[0][1]) if self.rows[0][1].replace(".", "").isdigit() else None,
                "power_w_max": max((float(r[2]) for r in self.rows if r[2].replace(".", "").isdigit()), default=None),
                "samples": len(self.rows), "reasons": reasons}


# ------------------------------------------------------------------------------------------ our arm

def stage_on_device(torch, steps):
    """All steps' tokens in ONE device buffer (pinned host copy kept for the e2e leg); per-step base offsets."""
    total = sum(len(t) for t, _ in steps)
    host = torch.empty(total + 4, dtype=torch.int32).pin_memory()
    bases, pos = [], 0
    hv = host.numpy()
    for t, _ in steps:
        bases.append(pos)
        hv[pos:pos + len(t)] = t
        pos += len(t)
    dev = host.cuda(non_blocking=False)
    return host, dev, bases


def run_device_resident(torch, A, info, steps, dev, bases, warmup, policy, stream, profile=False):
    """Replays steps on a fresh handle; returns (handle, elapsed_ms of the timed steps, per-kernel sums)."""
    cache = A.ArcCache(info.capacity_blocks, info.block_size, policy)
    acc, _, req = step_counts(steps)
    cache.reserve(max(req), max(acc))
    sp = int(stream.cuda_stream)
    base_ptr = dev.data_ptr()
    for i in range(warmup):
        rc = cache.step_raw(base_ptr + 4 * bases[i], steps[i][1], sp)
        assert rc == 0, rc
    sums = {}
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    if profile:
        cache.set_profiling(True)
    stream.synchronize()
    launches0 = cache.launch_count()
    ev0.record(stream)
    for i in range(warmup, len(steps)):
        rc = cache.step_raw(base_ptr + 4 * bases[i], steps[i][1], sp)
        assert rc == 0, rc
        if profile:
            for k, v in cache.last_kernel_times().items():
                sums[k] = sums.get(k, 0.0) + v
    ev1.record(stream)
    stream.synchronize()
    cache.stats()      # raises on a device-side directory error
    return cache, ev0.elapsed_time(ev1), sums, cache.launch_count() - launches0


def run_e2e(torch, A, info, steps, host, bases, warmup, stream):
    """arc_step_host: pinned HOST tokens -> device inside the call, results back to pinned host, per step."""
    cache = A.ArcCache(info.capacity_blocks, info.block_size, A.POLICY_ARC)
    acc, _, req = step_counts(steps)
    cache.reserve(max(req), max(acc))
    hv = host.numpy()
    views = [hv[bases[i]:bases[i] + len(steps[i][0])] for i in range(len(steps))]
    d2h = h2d = 0
    for i in range(warmup):
        cache.step_host(views[i], steps[i][1], stream)
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    stream.synchronize()
    t0 = time.perf_counter()
    ev0.record(stream)
    for i in range(warmup, len(steps)):
        r = cache.step_host(views[i], steps[i][1], stream)
        d2h += r["d2h_bytes"]   # one packed copy: prefix_len | counts | alloc_ids | evict_ids, as the library counts it
        h2d += r["h2d_bytes"]   # tokens + offsets and block offsets
    ev1.record(stream)
    stream.synchronize()
    wall_ms = (time.perf_counter() - t0) * 1e3
    cache.close()
    return max(wall_ms, ev0.elapsed_time(ev1)), d2h, h2d


def k1_bulk_roofline(torch, A, gib, stream, seed):
    """arc_hash_blocks over >= gib GiB of D5-shaped requests (lognormal(mean 8000, sigma 0.5) clipped to
    [1000, 32768] tokens, vocab 128,000): far larger than the 126 MB L2, so every launch streams from HBM."""
    n_tok = int(gib * (1 << 30) / 4)
    rng = np.random.Generator(np.random.PCG64(np.random.SeedSequence(seed + 77)))
    mu = np.log(8000.0) - 0.125
    lens = np.clip(np.rint(rng.lognormal(mu, 0.5, size=int(n_tok / 6000) + 64)), 1000, 32768).astype(np.int64)
    offs = np.concatenate([[0], np.cumsum(lens)])
    offs = offs[:np.searchsorted(offs, n_tok, side="right")]
    g = torch.Generator(device="cuda")
    g.manual_seed(seed + 78)
    tokens = torch.randint(0, 128000, (int(offs[-1]),), dtype=torch.int32, device="cuda", generator=g)
    n_blocks = int((np.diff(offs) // 16).sum())
    out = torch.empty(n_blocks, dtype=torch.int64, device="cuda")

    def timed(fn, reps=10, warm=10):
        for _ in range(warm):
            fn()
        evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(reps)]
        stream.synchronize()
        for a, b in evs:
            a.record(stream)
            fn()
            b.record(stream)
        stream.synchronize()
        ms = sorted(a.elapsed_time(b) for a, b in evs)
        return float(np.mean(ms)), ms[0]

    # through the API: host offsets in, the call copies them (its own copy stream) and launches
    api_mean, api_best = timed(lambda: A.hash_blocks(tokens, offs, 16, out=out, stream=stream))
    keys_api = out.clone()
    # the kernel alone: offsets and block offsets already on the device
    d_off = torch.from_numpy(offs).cuda()
    blk = np.zeros(len(offs), np.int64)
    blk[1:] = np.cumsum(np.diff(offs) // 16)
    d_blk = torch.from_numpy(blk).cuda()
    ticket = torch.zeros(2, dtype=torch.int32, device="cuda")
    out.zero_()
    ker_mean, ker_best = timed(lambda: A.hash_blocks_device(tokens, d_off, d_blk, len(offs) - 1, out, ticket, stream=stream))
    same = bool(torch.equal(out, keys_api))
    return dict(blocks=n_blocks, requests=len(offs) - 1, api_ms=api_mean, api_best_ms=api_best, kernel_ms=ker_mean, kernel_best_ms=ker_best,
                same_keys=same)


def k2_probe_bench(torch, A, stream, seed, n_keys=1 << 24):
    """K2 alone on a directory far larger than L2: capacity 16 M blocks (2 GiB table), 16 M distinct random keys inserted,
    then looked up again in a different random order (every probe is one random 128-B bucket read from HBM)."""
    cache = A.ArcCache(n_keys, 16, A.POLICY_ARC)
    g = torch.Generator(device="cuda")
    g.manual_seed(seed + 91)
    keys = torch.randint(2, 2 ** 62, (n_keys,), dtype=torch.int64, device="cuda", generator=g)
    nodes = torch.empty(n_keys, dtype=torch.int32, device="cuda")
    cache.reserve(1, n_keys)
    cache.debug_probe(keys, nodes, stream)                      # inserts
    stream.synchronize()
    first = nodes.clone()
    perm = torch.randperm(n_keys, device="cuda", generator=g)
    keys2 = keys[perm].contiguous()
    for _ in range(2):
        cache.debug_probe(keys2, nodes, stream)
    evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(5)]
    stream.synchronize()
    for a, b in evs:
        a.record(stream)
        cache.debug_probe(keys2, nodes, stream)
        b.record(stream)
    stream.synchronize()
    ok = bool(torch.equal(nodes, first[perm]))                  # every key found again, at the node it was given
    ms = float(np.mean([a.elapsed_time(b) for a, b in evs]))
    cache.close()
    return n_keys, ms, ok


def serving_loop_leg(torch, A, info, steps, stream, seed, n_steps=240, new_per_step=8, decode_steps=2):
    """NEXT-3 measured: continuous batching under held pins.  Every step admits `new_per_step` prompts of
    the configured trace, every sequence admitted in the last `decode_steps` steps grows by one block of generated tokens
    from its stored chain state (arc_step_resume), and the sequences admitted `decode_steps` steps ago finish: all their
    holds go back in one arc_release.  Timed on the device; the same loop is then replayed on the CPU oracle and the
    counters compared."""
    from oracle import oracle as O

    S0 = 0x243F6A8885A308D3
    rng = np.random.Generator(np.random.PCG64(np.random.SeedSequence(seed + 99)))
    prompts = []
    for tok, off in steps:
        prompts += [tok[off[r]:off[r + 1]] for r in range(len(off) - 1)]
    need = n_steps * new_per_step
    prompts = [p[:len(p) // 16 * 16] for p in prompts[:need]]           # whole blocks: decode continues at a block boundary
    n_steps = len(prompts) // new_per_step
    gen = rng.integers(0, 128000, size=(n_steps, decode_steps * new_per_step, 16)).astype(np.int32)
    plan = []                                                            # per step: (tokens, offsets, n_new, n_dec)
    held = []                                                            # holds of the cohorts still running, oldest first
    for i in range(n_steps):
        new = prompts[i * new_per_step:(i + 1) * new_per_step]
        n_dec = new_per_step * min(i, decode_steps)
        # admission (the scheduler's job): holds outstanding + this step's blocks <= c; the longest prompts are cut until it fits
        budget = info.capacity_blocks - sum(held) - n_dec
        while sum(len(p) for p in new) // 16 > budget:
            k = max(range(len(new)), key=lambda j: len(new[j]))
            new[k] = new[k][:len(new[k]) // 32 * 16]
        held = [h + new_per_step for h in held] + [sum(len(p) for p in new) // 16]
        if len(held) > decode_steps:
            held.pop(0)
        reqs = new + [gen[i, d] for d in range(n_dec)]
        off = np.zeros(len(reqs) + 1, np.int64)
        off[1:] = np.cumsum([len(r) for r in reqs])
        plan.append((np.concatenate(reqs), off, len(new), n_dec))
    dev_tok = [torch.from_numpy(t).cuda() for t, _, _, _ in plan]
    s0_new = torch.full((new_per_step,), S0, dtype=torch.int64, device="cuda")                 # S0 < 2^63: same bit pattern

    def run(cache, on_gpu):
        """One pass of the loop; returns (accesses, ids released)."""
        hist = []                # per step: (block ids of each of its sequences so far, their chain states)
        n_acc = n_rel = 0
        for i, (tok, off, n_new, n_dec) in enumerate(plan):
            # decode requests are ordered oldest cohort first: cohort i-decode_steps .. i-1, new_per_step sequences each
            cohorts = hist[-min(i, decode_steps):] if i else []
            if on_gpu:
                chain = torch.cat([s0_new] + [c["state"] for c in cohorts])
                r = cache.step(dev_tok[i], off, stream, chain_in=chain)
                ids, st, bo = r.block_id.clone(), r.chain_state.clone(), off // 16
            else:
                chain = np.concatenate([np.full(n_new, S0, np.uint64)] + [c["state"] for c in cohorts])
                r = cache.step(tok, off, chain_in=chain)
                ids, st, bo = r["block_id"], r["chain_state"], off // 16
            n_acc += int(bo[-1])
            for k, c in enumerate(cohorts):                               # each running sequence took one more block
                a = int(bo[n_new + k * new_per_step])
                c["ids"].append(ids[a:a + new_per_step])
                c["state"] = st[n_new + k * new_per_step:n_new + (k + 1) * new_per_step]
            hist.append(dict(ids=[ids[:int(bo[n_new])]], state=st[:n_new]))
            if len(hist) > decode_steps:                                  # the oldest cohort finishes
                done = hist.pop(0)
                rel = (torch.cat if on_gpu else np.concatenate)(done["ids"])
                cache.release(rel)
                n_rel += int(rel.shape[0])
        for done in hist:                                                 # the pass ends with nothing held
            rel = (torch.cat if on_gpu else np.concatenate)(done["ids"])
            cache.release(rel)
            n_rel += int(rel.shape[0])
        return n_acc, n_rel

    cache = A.ArcCache(info.capacity_blocks, info.block_size, A.POLICY_ARC)
    cache.set_pin_scope(A.PIN_HELD)
    cache.reserve(new_per_step * (decode_steps + 1), max(int(o[-1]) // 16 for _, o, _, _ in plan))
    run(cache, True)                                                      # warm-up pass: buffers sized, cache in steady state
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    stream.synchronize()
    ev0.record(stream)
    n_acc, n_rel = run(cache, True)
    ev1.record(stream)
    stream.synchronize()
    ms = ev0.elapsed_time(ev1)
    st = cache.stats()
    cache.close()
    oc = O.OracleCache(info.capacity_blocks, info.block_size, 0)
    oc.set_pin_scope(2)
    run(oc, False)
    t0 = time.perf_counter()
    run(oc, False)
    cpu_s = time.perf_counter() - t0
    so = oc.stats()
    same = all(st[k] == so[k] for k in ("accesses", "hit_t1", "hit_t2", "ghost_b1", "ghost_b2", "miss", "evict_t1", "evict_t2", "p", "t1", "t2", "b1", "b2"))
    return {"what": f"held pins + arc_step_resume + arc_release: {new_per_step} prompts admitted per step, each sequence decodes {decode_steps} blocks "
                    f"(one per step) and then releases everything it holds; c={info.capacity_blocks}",
            "steps": n_steps, "accesses_per_step": n_acc / n_steps, "released_ids_per_step": n_rel / n_steps,
            "ms_per_step": ms / n_steps, "accesses_per_s": n_acc / (ms * 1e-3),
            "includes": "binding work per step (chain-state gather, clone of block_id for the later release) and one release launch",
            "hit_rate_blocks": (st["hit_t1"] + st["hit_t2"]) / max(1, st["accesses"]),
            "cpu_oracle_accesses_per_s": n_acc / cpu_s, "parity_spot_check": same}


def cpu_oracle_leg(info, steps, policy=0):
    """The oracle as it stands (g++ -O2, std::list + unordered_map, one thread) over the same steps."""
    from oracle import oracle as O

    oc = O.OracleCache(info.capacity_blocks, info.block_size, policy)
    t0 = time.perf_counter()
    n = 0
    for tokens, offsets in steps:
        n += oc.step(tokens, offsets, unpack=False)
    dt = time.perf_counter() - t0
    tm, st = oc.timing(), oc.stats()
    oc.close()
    return n, dt, tm, st


def hit_rates(st):
    a = max(1, st["accesses"])
    return {"block_hit_rate": (st["hit_t1"] + st["hit_t2"]) / a, "prefix_token_hit_rate": st["prefix_hit_tokens"] / max(1, st["tokens_seen"])}


def run_ours(args):
    import torch
    import torch.distributed as dist

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the hot path has no CPU fallback (use --impl reference for the oracle)")
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    from paper_2606_21238_b200 import arc as A
    from paper_2606_21238_b200 import parallel as P

    A.load_library()
    if args.only_k1:
        peak, peak_src = peaks()
        k1 = k1_bulk_roofline(torch, A, args.bulk_gib, torch.cuda.current_stream(), args.seed)
        gb = ALGO_BYTES_PER_BLOCK * k1["blocks"] / 1e9
        k1.update(kernel="K1 chained block hashing", api_GBps=gb / (k1["api_ms"] * 1e-3), kernel_GBps=gb / (k1["kernel_ms"] * 1e-3), peak=peak,
                  frac=gb / (k1["api_ms"] * 1e-3) / peak, frac_kernel=gb / (k1["kernel_ms"] * 1e-3) / peak, peak_source=peak_src)
        print(json.dumps(k1))
        return
    W_, K = args.warmup, args.steps
    info, steps = build_steps(args.config, W_ + K, P.replica_seed(args.seed, rank))
    acc, tok, req = step_counts(steps)
    n_acc, n_tok, n_req = sum(acc[W_:]), sum(tok[W_:]), sum(req[W_:])
    host, dev, bases = stage_on_device(torch, steps)
    stream = torch.cuda.current_stream()

    # ---- timed region: K steps enqueued back to back, tokens resident in HBM --------------------------
    P.barrier(dist if world > 1 else None)
    torch.cuda.synchronize()
    with ClockSampler(local) as clk:
        cache, ms, _, launches = run_device_resident(torch, A, info, steps, dev, bases, W_, A.POLICY_ARC, stream)
    torch.cuda.synchronize()
    P.barrier(dist if world > 1 else None)
    st_arc = cache.stats()
    cache.close()
    ms_max, tot_acc, tot_tok, tot_req = P.reduce_timing(dist if world > 1 else None, torch, ms, n_acc, n_tok, n_req)

    # ---- e2e: the same steps through arc_step_host (H2D + D2H inside) ----------------------------------
    e2e_ms, d2h, h2d_total = run_e2e(torch, A, info, steps, host, bases, W_, stream)
    e2e_ms_max, _, _, _ = P.reduce_timing(dist if world > 1 else None, torch, e2e_ms, n_acc, n_tok, n_req)
    h2d = h2d_total / K

    line = {
        "metric": METRIC, "value": tot_acc / (ms_max * 1e-3), "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W_,
        "ms_per_step": ms_max / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "u64 hash / i32 directory", "data": "synthetic",
        "config": {"workload": f"BASELINE.json configs[{args.config - 1}] ({info.name}): c={info.capacity_blocks} blocks x {info.block_size} tokens, "
                               f"{info.requests_per_step} requests/step, steps {W_}..{W_ + K - 1} of the seeded trace",
                   "accesses_per_step": n_acc / K, "tokens_per_step": n_tok / K, "policy": "ARC",
                   "parallelism": "replicas only" if world > 1 else "single GPU",
                   "l2": f"inputs larger than L2: every step reads its own slice of a {4 * sum(tok) / 1e6:.0f} MB token window staged in HBM; "
                         "the directory is deliberately L2-resident"},
        "tokens_hashed_per_s": 16 * tot_acc / (ms_max * 1e-3), "tokens_seen_per_s": tot_tok / (ms_max * 1e-3),
        "requests_per_s": tot_req / (ms_max * 1e-3),
        "e2e": {"value": tot_acc / (e2e_ms_max * 1e-3), "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h / K,
                "ms_per_step": e2e_ms_max / K, "api": "arc_step_host (synchronous, pinned host tokens)"},
        "gpu_launches": launches,
        "clocks": clk.summary(),
    }

    if rank == 0 and not args.no_extras:
        peak, peak_src = peaks()
        # per-kernel breakdown: a separate pass with CUDA events between the kernels (it syncs every step)
        c2, _, sums, _ = run_device_resident(torch, A, info, steps, dev, bases, W_, A.POLICY_ARC, stream, profile=True)
        line["k3_debug"] = c2.debug_counters()
        c2.close()
        tot = max(sums.get("total_ms", 0.0), 1e-9)
        line["kernels"] = {k: {"ms_per_step": v / K, "share": v / tot} for k, v in sums.items() if k != "total_ms"}
        line["kernels"]["total_ms_per_step"] = tot / K
        line["k3_ns_per_access"] = 1e6 * sums.get("machine_ms", 0.0) / max(1, n_acc)
        line["dominant_kernel"] = {"kernel": "K3 ARC machine (arc_machine_wide_kernel, one CTA)", "share_of_step": sums.get("machine_ms", 0.0) / tot,
                                   "bound": "latency: dependent instructions of one serial state machine (DESIGN.md 7.3); neither HBM nor tensor nor ALU throughput",
                                   "ns_per_access": 1e6 * sums.get("machine_ms", 0.0) / max(1, n_acc),
                                   "ncu": "profiles/r01e_held_resume_roll.md: about 43 warp instructions per access over 8 warps (38-52 on steps 15-17), 19 % issue-active per scheduler",
                                   "issue_roofline": {"bound": "alu", "what": "warp-instruction issue of the ONE SM the machine runs on (4 schedulers x 1 instruction per clock)",
                                                      "achieved": 43.0 * n_acc / max(sums.get("machine_ms", 0.0) * 1e-3, 1e-12), "unit": "warp instructions/s",
                                                      "peak": 4 * 1.965e9, "frac": 43.0 * n_acc / max(sums.get("machine_ms", 0.0) * 1e-3, 1e-12) / (4 * 1.965e9),
                                                      "instructions_per_access": "43, from the ncu capture named above (smsp__inst_executed.sum / accesses of that step)"}}
        k1_insitu = ALGO_BYTES_PER_BLOCK * n_acc / max(sums.get("hash_ms", 0.0) * 1e-3, 1e-12) / 1e9
        # K1 roofline: bulk run through arc_hash_blocks
        nb, nreq_b, mean_ms, best_ms = k1_bulk_roofline(torch, A, args.bulk_gib, stream, args.seed)
        achieved = ALGO_BYTES_PER_BLOCK * nb / (mean_ms * 1e-3) / 1e9
        line["roofline"] = {"kernel": "K1 chained block hashing (arc_hash_blocks)", "bound": "hbm", "achieved": achieved, "peak": peak,
                            "unit": "GB/s", "frac": achieved / peak, "frac_of_nominal_8000": achieved / 8000.0, "peak_source": peak_src,
                            "traffic": 1.168e9 if abs(args.bulk_gib - 1.0) < 1e-9 else None,
                            "traffic_source": "dram__bytes_read.sum + dram__bytes_write.sum of one ncu --set full capture of this launch (profiles/r01e_held_resume_roll.md: 1.0855 GB + 82.3 MB)",
                            "algorithmic_bytes_per_launch": ALGO_BYTES_PER_BLOCK * nb, "ms_per_launch": mean_ms,
                            "best_ms": best_ms, "tokens_per_s": 16 * nb / (mean_ms * 1e-3),
                            "workload": f"{nreq_b} D5-shaped requests, {nb} blocks, {64 * nb / 2**30:.2f} GiB of tokens (>> 126 MB L2)",
                            "in_situ_GBps": k1_insitu}
        # K2 alone, table >> L2
        nk, k2_ms, k2_ok = k2_probe_bench(torch, A, stream, args.seed)
        line["probe"] = {"kernel": "K2 probe_reserve + resolve (arc_debug_probe)", "keys": nk, "ms_per_launch": k2_ms, "keys_per_s": nk / (k2_ms * 1e-3),
                         "found_all": k2_ok, "table": "capacity 16 M blocks: 2 GiB table of 16-B slots in 128-B buckets, load 0.125",
                         "algorithmic_GBps": 28 * nk / (k2_ms * 1e-3) / 1e9, "sector_level_GBps": 140 * nk / (k2_ms * 1e-3) / 1e9,
                         "frac_of_measured_hbm_sector_level": 140 * nk / (k2_ms * 1e-3) / 1e9 / peak,
                         "bytes_model": "algorithmic 28 B/key (8 B key + 16 B slot + 4 B node id); sector level 140 B/key (8 + one 128-B bucket + 4)",
                         "in_situ_us_per_step": 1e3 * sums.get("probe_ms", 0.0) / K}
        # ARC vs LRU on the same steps
        c3, _, _, _ = run_device_resident(torch, A, info, steps, dev, bases, W_, A.POLICY_LRU, stream)
        st_lru = c3.stats()
        c3.close()
        c4, _, _, _ = run_device_resident(torch, A, info, steps, dev, bases, W_, A.POLICY_DBL, stream)
        st_dbl = c4.stats()
        c4.close()
        ha, hl = hit_rates(st_arc), hit_rates(st_lru)
        line["hit_rate"] = {"arc": ha, "lru": hl, "dbl": hit_rates(st_dbl),
                            "arc_minus_lru_points": {k: 100 * (ha[k] - hl[k]) for k in ha},
                            "scope": f"all {W_ + K} steps from an empty cache",
                            "paper_context": "+10.8% hit rate / -12.6% TTFT (doc QA), +2.1% / -2.0% (conversation): Qwen3-14B, vLLM, 1x H100 PCIe 80 GB (PAPER.md:7, :86, :111, :117)"}
        line["state"] = {k: st_arc[k] for k in ("t1", "t2", "b1", "b2", "p")}
        # NEXT-3 measured: a continuous-batching loop under held pins (only where a batch fits the cache)
        if args.config == 2:
            line["serving_loop"] = serving_loop_leg(torch, A, info, steps, stream, args.seed)
        # the CPU oracle on the same steps, on this box's host cores
        n_o, dt, tm, st_o = cpu_oracle_leg(info, steps)
        line["cpu_baseline"] = {"value": n_o / dt, "unit": UNIT, "cores": 1, "kind": "oracle",
                                "sample": f"the same {W_ + K} steps (warm-up included), {n_o} accesses, {dt:.2f} s: hashing {tm['hash_seconds']:.2f} s + ARC {tm['arc_seconds']:.2f} s",
                                "host_cpus": os.cpu_count()}
        line["parity_spot_check"] = all(st_o[k] == st_arc[k] for k in ("accesses", "hit_t1", "hit_t2", "ghost_b1", "ghost_b2", "miss", "p", "t1", "t2", "b1", "b2"))
    if rank == 0:
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


# ------------------------------------------------------------------------------------ reference arm

def run_reference(args):
    """The tier's reference arm = the CPU oracle as it stands, on this box's host cores (rank 0 only)."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    info, steps = build_steps(args.config, args.warmup + args.steps, args.seed)
    from oracle import oracle as O

    oc = O.OracleCache(info.capacity_blocks, info.block_size, O.POLICY_ARC)
    for tokens, offsets in steps[:args.warmup]:
        oc.step(tokens, offsets, unpack=False)
    acc, tok, req = step_counts(steps[args.warmup:])
    t0 = time.perf_counter()
    for tokens, offsets in steps[args.warmup:]:
        oc.step(tokens, offsets, unpack=False)
    dt = time.perf_counter() - t0
    v = sum(acc) / dt
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": 1e3 * dt / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "u64 hash / i32 directory", "data": "synthetic",
        "config": {"workload": f"BASELINE.json configs[{args.config - 1}] ({info.name}): c={info.capacity_blocks} blocks x {info.block_size} tokens, "
                               f"{info.requests_per_step} requests/step, steps {args.warmup}..{args.warmup + args.steps - 1} of the seeded trace",
                   "policy": "ARC"},
        "tokens_hashed_per_s": 16 * v, "requests_per_s": sum(req) / dt,
        "cpu_baseline": {"value": v, "unit": UNIT, "cores": 1, "kind": "oracle",
                         "sample": f"every timed step is one whole step of the workload ({sum(acc)} accesses in {dt:.2f} s)"},
        "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }))


if __name__ == "__main__":
    a = parse_args()
    run_reference(a) if a.impl == "reference" else run_ours(a)
