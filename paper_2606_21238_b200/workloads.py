"""Seeded synthetic request traces shaped like the paper's workloads.

This module only *generates inputs* (token IDs and CSR offsets).  It holds none of
the method's arithmetic (no hashing, no cache logic) and is the one module that
both the CPU oracle's tests and the CUDA path's tests / bench import.

The paper measures on QuALITY / WikiQA document QA (a long shared
document followed by a short unique question, documents drawn by Zipf popularity)
and on the Qwen-Bailian conversation trace (growing dialogue history,
~2.3k input tokens).  Those datasets are not available; the generators below take
their *shape* and follow BASELINE.json `configs` as pinned in SURVEY.md §8(d) D1-D5.

Conventions: numpy Generator(PCG64); one SeedSequence child per
purpose; token dtype int32; bounded Zipf  P(rank k) ∝ k^(-s), k = 1..n, rank k <->
item k-1, no reshuffling.  A trace is produced one step at a time:
`for tokens, offsets in trace.steps(): ...` where request r of the step is
`tokens[offsets[r]:offsets[r+1]]`.
"""
from __future__ import annotations

import hashlib
from dataclasses import dataclass
from typing import Iterator, List, Optional, Tuple

import numpy as np

Step = Tuple[np.ndarray, np.ndarray]  # (tokens int32[total], offsets int64[n_req+1])


def _children(seed: int, n: int):
    """n independent SeedSequence children of `seed`, one per purpose."""
    return np.random.SeedSequence(seed).spawn(n)


def _gen(seed_seq) -> np.random.Generator:
    """A fresh generator at the start of its stream (so a trace can be replayed)."""
    return np.random.Generator(np.random.PCG64(seed_seq))


def zipf_probabilities(n_items: int, s: float) -> np.ndarray:
    ranks = np.arange(1, n_items + 1, dtype=np.float64)
    w = ranks ** (-float(s))
    return w / w.sum()


def _pack(requests: List[np.ndarray]) -> Step:
    """CSR-pack a list of int32 arrays."""
    n = len(requests)
    offsets = np.zeros(n + 1, dtype=np.int64)
    if n:
        offsets[1:] = np.cumsum([len(r) for r in requests], dtype=np.int64)
        tokens = np.concatenate(requests).astype(np.int32, copy=False) if offsets[-1] else np.zeros(0, np.int32)
    else:
        tokens = np.zeros(0, np.int32)
    return np.ascontiguousarray(tokens), offsets


@dataclass
class TraceInfo:
    name: str
    capacity_blocks: int
    block_size: int
    requests_per_step: int
    n_requests: int

    @property
    def n_steps(self) -> int:
        return -(-self.n_requests // self.requests_per_step)


class Trace:
    """Base: subclasses implement `_request_stream()` yielding one int32 array per request."""

    info: TraceInfo

    def _request_stream(self) -> Iterator[np.ndarray]:
        raise NotImplementedError

    def requests(self, max_requests: Optional[int] = None) -> Iterator[np.ndarray]:
        for i, r in enumerate(self._request_stream()):
            if max_requests is not None and i >= max_requests:
                return
            yield r

    def steps(self, max_steps: Optional[int] = None, requests_per_step: Optional[int] = None) -> Iterator[Step]:
        rps = requests_per_step or self.info.requests_per_step
        batch: List[np.ndarray] = []
        n_steps = 0
        for r in self._request_stream():
            batch.append(r)
            if len(batch) == rps:
                yield _pack(batch)
                batch = []
                n_steps += 1
                if max_steps is not None and n_steps >= max_steps:
                    return
        if batch:
            yield _pack(batch)


# ----------------------------------------------------------------------------- doc QA


class DocQATrace(Trace):
    """Whole document (Zipf popularity) ++ fresh unique question suffix (D1, D2; doc half of D4, D5)."""

    def __init__(self, info: TraceInfo, *, n_docs: int, vocab: int, zipf_s: float, doc_len, q_len: Tuple[int, int], seed: int):
        self.info = info
        ss_corpus, ss_pop, ss_suffix = _children(seed, 3)
        rng_corpus, rng_pop = _gen(ss_corpus), _gen(ss_pop)
        lengths = doc_len(rng_corpus, n_docs)
        self.docs = [rng_corpus.integers(0, vocab, size=int(n), dtype=np.int32) for n in lengths]
        self.choice = rng_pop.choice(n_docs, size=info.n_requests, p=zipf_probabilities(n_docs, zipf_s))
        self.ss_suffix = ss_suffix
        self.vocab = vocab
        self.q_len = q_len

    def _request_stream(self):
        # question lengths / tokens are drawn in request order from one stream
        rng = _gen(self.ss_suffix)
        lo, hi = self.q_len
        for d in self.choice:
            n_q = int(rng.integers(lo, hi + 1))
            q = rng.integers(0, self.vocab, size=n_q, dtype=np.int32)
            yield np.concatenate([self.docs[int(d)], q])


def _uniform_len(lo: int, hi: int):
    return lambda rng, n: rng.integers(lo, hi + 1, size=n)


def _lognormal_len(mean: float, sigma: float, lo: int, hi: int):
    mu = np.log(mean) - sigma * sigma / 2.0  # "mean" read as the expectation
    return lambda rng, n: np.clip(np.rint(rng.lognormal(mu, sigma, size=n)), lo, hi).astype(np.int64)


# ----------------------------------------------------------------------- conversation


class ConversationTrace(Trace):
    """Multi-turn sessions; each turn's prompt = whole prior conversation ++ new user turn (D3)."""

    def __init__(self, info: TraceInfo, *, n_sessions: int, vocab: int, seed: int, mean_gap: float = 1.0,
                 mean_think: float = 100.0, mean_turns: float = 5.0, max_turns: int = 20,
                 user_len: Tuple[int, int] = (20, 300), reply_len: Tuple[int, int] = (50, 500),
                 max_requests: Optional[int] = None):
        ss_arrivals, ss_tokens = _children(seed, 2)
        rng_arrivals = _gen(ss_arrivals)
        starts = np.cumsum(rng_arrivals.exponential(mean_gap, size=n_sessions))
        turns = np.minimum(rng_arrivals.geometric(1.0 / mean_turns, size=n_sessions), max_turns)
        sess = np.repeat(np.arange(n_sessions), turns)
        first = np.concatenate([[0], np.cumsum(turns)[:-1]])
        turn_idx = np.arange(len(sess)) - np.repeat(first, turns)
        think = rng_arrivals.exponential(mean_think, size=len(sess))
        think[turn_idx == 0] = 0.0
        # time of turn j = session start + sum of think times of turns 1..j
        csum = np.cumsum(think)
        base = np.repeat(csum[first], turns)
        t = np.repeat(starts, turns) + (csum - base)
        order = np.lexsort((turn_idx, sess, t))  # by time, ties: session, turn
        if max_requests is not None:
            order = order[:max_requests]
        self.ev_sess = sess[order]
        self.ev_turn = turn_idx[order]
        self.n_turns = turns
        self.ss_tokens = ss_tokens
        self.vocab, self.user_len, self.reply_len = vocab, user_len, reply_len
        info.n_requests = len(order)
        self.info = info

    def _request_stream(self):
        rng = _gen(self.ss_tokens)
        hist = {}
        for s, j in zip(self.ev_sess.tolist(), self.ev_turn.tolist()):
            user = rng.integers(0, self.vocab, size=int(rng.integers(self.user_len[0], self.user_len[1] + 1)), dtype=np.int32)
            reply = rng.integers(0, self.vocab, size=int(rng.integers(self.reply_len[0], self.reply_len[1] + 1)), dtype=np.int32)
            prev = hist.get(s)
            prompt = user if prev is None else np.concatenate([prev, user])
            yield prompt
            if j + 1 < int(self.n_turns[s]):
                hist[s] = np.concatenate([prompt, reply])  # reply appended *after* the request
            else:
                hist.pop(s, None)


# ------------------------------------------------------------------------------ mixes


class ScanMixTrace(Trace):
    """D4: 70 % doc-QA hot set, 30 % one-shot 16,384-token scans."""

    def __init__(self, info: TraceInfo, *, seed: int, scan_prob: float = 0.3, scan_len: int = 16384,
                 n_docs: int = 500, zipf_s: float = 1.1, vocab: int = 32000):
        self.info = info
        ss_mix, ss_scan = _children(seed, 2)
        self.is_scan = _gen(ss_mix).random(info.n_requests) < scan_prob
        self.ss_scan = ss_scan
        self.scan_len, self.vocab = scan_len, vocab
        n_hot = int((~self.is_scan).sum())
        self.hot = DocQATrace(TraceInfo("hot", info.capacity_blocks, info.block_size, info.requests_per_step, n_hot),
                              n_docs=n_docs, vocab=vocab, zipf_s=zipf_s, doc_len=_uniform_len(64, 448),
                              q_len=(16, 64), seed=seed + 1)

    def _request_stream(self):
        rng = _gen(self.ss_scan)
        hot = self.hot._request_stream()
        for scan in self.is_scan.tolist():
            if scan:
                yield rng.integers(0, self.vocab, size=self.scan_len, dtype=np.int32)
            else:
                yield next(hot)


class InterleaveTrace(Trace):
    """D5: two request streams interleaved by a seeded mask with exact counts, each keeping its order."""

    def __init__(self, info: TraceInfo, a: Trace, b: Trace, n_a: int, n_b: int, seed: int):
        (ss_mix,) = _children(seed, 1)
        self.take_a = _gen(ss_mix).permutation(n_a + n_b) < n_a
        self.a, self.b = a, b
        info.n_requests = n_a + n_b
        self.info = info

    def _request_stream(self):
        sa, sb = self.a._request_stream(), self.b._request_stream()
        for t in self.take_a.tolist():
            yield next(sa) if t else next(sb)


class WindowedZipfTrace(Trace):
    """The paper's own workload shape: `n_windows` windows of `window` requests; inside a window documents
    are drawn Zipf(s); the rank -> document assignment is reshuffled for every window (popularity shifts).  Whole document
    ++ fresh question, one request per step by default (the paper runs batch size 1).  Documents are
    synthetic (lognormal lengths, uniform tokens); the QuALITY / WikiQA texts are not available and not imitated."""

    def __init__(self, info: TraceInfo, *, n_docs: int, vocab: int, zipf_s: float, doc_len, q_len: Tuple[int, int],
                 window: int, n_windows: int, seed: int):
        info.n_requests = window * n_windows
        self.info = info
        ss_corpus, ss_pop, ss_suffix, ss_perm = _children(seed, 4)
        rng_corpus, rng_pop, rng_perm = _gen(ss_corpus), _gen(ss_pop), _gen(ss_perm)
        lengths = doc_len(rng_corpus, n_docs)
        self.docs = [rng_corpus.integers(0, vocab, size=int(n), dtype=np.int32) for n in lengths]
        p = zipf_probabilities(n_docs, zipf_s)
        choice = []
        self.window_perms = []
        for _ in range(n_windows):
            perm = rng_perm.permutation(n_docs)            # rank k -> document perm[k], redrawn per window
            self.window_perms.append(perm)
            choice.append(perm[rng_pop.choice(n_docs, size=window, p=p)])
        self.choice = np.concatenate(choice)
        self.window = window
        self.ss_suffix, self.vocab, self.q_len = ss_suffix, vocab, q_len

    def _request_stream(self):
        rng = _gen(self.ss_suffix)
        lo, hi = self.q_len
        for d in self.choice:
            q = rng.integers(0, self.vocab, size=int(rng.integers(lo, hi + 1)), dtype=np.int32)
            yield np.concatenate([self.docs[int(d)], q])


def make_windowed_zipf(capacity_blocks: int, seed: int = 0, *, n_docs: int = 381, mean_doc_tokens: float = 5000.0,
                       window: int = 512, n_windows: int = 6, zipf_s: float = 1.0, requests_per_step: int = 1) -> WindowedZipfTrace:
    """3,072 requests = 6 windows x 512, Zipf exponent 1.0, items reshuffled per window
    (PAPER.md:99); 381 documents of about 5k tokens (the counts PAPER.md:97 quotes for its document set)."""
    info = TraceInfo("windowed-zipf", capacity_blocks, 16, requests_per_step, 0)
    return WindowedZipfTrace(info, n_docs=n_docs, vocab=128000, zipf_s=zipf_s,
                             doc_len=_lognormal_len(mean_doc_tokens, 0.5, 1000, 16000), q_len=(16, 64),
                             window=window, n_windows=n_windows, seed=seed)


# ---------------------------------------------------------------------------- configs

CONFIG_NAMES = {1: "tiny-docqa", 2: "docqa", 3: "conversation", 4: "scan-hotset", 5: "scale-stress"}


def make_trace(config: int, seed: int = 0, *, scale: float = 1.0) -> Trace:
    """BASELINE.json configs[config-1] as pinned in SURVEY.md §8(d).

    `scale` < 1 shrinks only the *number of requests / sessions* (for bounded tests and
    bench windows); cache size, corpus and per-request shapes are unchanged.
    """
    def n(x):
        return max(1, int(round(x * scale)))

    if config == 1:
        info = TraceInfo(CONFIG_NAMES[1], 64, 16, 8, n(2000))
        return DocQATrace(info, n_docs=20, vocab=32000, zipf_s=1.0, doc_len=_uniform_len(64, 448), q_len=(16, 64), seed=seed)
    if config == 2:
        info = TraceInfo(CONFIG_NAMES[2], 8192, 16, 64, n(50000))
        return DocQATrace(info, n_docs=200, vocab=128000, zipf_s=0.8, doc_len=_lognormal_len(4000, 0.5, 1000, 16000),
                          q_len=(32, 128), seed=seed)
    if config == 3:
        info = TraceInfo(CONFIG_NAMES[3], 32768, 16, 128, 0)
        return ConversationTrace(info, n_sessions=n(40000), vocab=128000, seed=seed)
    if config == 4:
        info = TraceInfo(CONFIG_NAMES[4], 65536, 16, 256, n(500000))
        return ScanMixTrace(info, seed=seed)
    if config == 5:
        n_each = n(1000000)
        info = TraceInfo(CONFIG_NAMES[5], 1048576, 16, 1024, 0)
        docs = DocQATrace(TraceInfo("d5-docs", info.capacity_blocks, 16, 1024, n_each), n_docs=5000, vocab=128000,
                          zipf_s=0.9, doc_len=_lognormal_len(8000, 0.5, 1000, 32768), q_len=(32, 128), seed=seed + 11)
        conv = ConversationTrace(TraceInfo("d5-conv", info.capacity_blocks, 16, 1024, 0),
                                 n_sessions=max(8, int(n_each * 0.21)), vocab=128000, seed=seed + 12, max_requests=n_each)
        n_conv = conv.info.n_requests
        return InterleaveTrace(info, docs, conv, n_each, n_conv, seed=seed + 13)
    raise ValueError(f"unknown config {config}")


def trace_digest(trace: Trace, max_steps: Optional[int] = None) -> str:
    """SHA-256 over the offsets and tokens of every step (reproducibility check)."""
    h = hashlib.sha256()
    for tokens, offsets in trace.steps(max_steps):
        h.update(offsets.tobytes())
        h.update(tokens.tobytes())
    return h.hexdigest()


# ----------------------------------------------------------------- small test inputs


def prefix_tree_requests(rng: np.random.Generator, *, n_requests: int, block_size: int, branching: int, depth: int,
                         max_blocks: int, tail_tokens: bool = True) -> List[np.ndarray]:
    """Tiny-cache differential inputs: requests are root-to-node paths in a small token-block tree,
    so that chained keys are shared between requests (SURVEY §8(c) pin 3)."""
    # each tree edge is one block of `block_size` tokens determined by (depth level, branch)
    table = rng.integers(0, 1000, size=(depth, branching, block_size), dtype=np.int32)
    out = []
    for _ in range(n_requests):
        nb = int(rng.integers(1, max_blocks + 1))
        path = rng.integers(0, branching, size=nb)
        toks = [table[min(lvl, depth - 1), int(b)] for lvl, b in enumerate(path)]
        if tail_tokens:
            toks.append(rng.integers(0, 1000, size=int(rng.integers(0, block_size)), dtype=np.int32))
        out.append(np.concatenate(toks).astype(np.int32))
    return out


def pack_requests(requests: List[np.ndarray]) -> Step:
    return _pack(list(requests))
