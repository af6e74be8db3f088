"""ORACLE (test infrastructure, not product): the whole prefix-cached prefill path on the CPU, request by
request, composed of oracle/ordering.py, oracle/blocks.py and oracle/attention.py.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this.
Shares no code with paper_2606_19667_b200/; inputs come from tracegen (seeded generators only).

Per request (SURVEY.md §3 build call stack):
   O = order(D); observe(O); tokens = docs[O] ‖ query; (table, c) = lookup(tokens);
   append RoPE'd K / V of the suffix to the pool; attention of the suffix rows over prefix + suffix; release.
Admission "sequential": release right after each request.  Admission "waves": requests are admitted until
the pool reports NoSpace, the wave is prefilled, released, and admission resumes (SURVEY.md §8(d) cfg 4/5).
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

import tracegen
from .attention import PagedPool, attention_suffix, attention_full
from .blocks import BlockManager, NoSpace, chain_hashes, matched_docs
from .ordering import KnowledgeTree
from .strategies import RecencyOrder, order_exhaustive, order_sorted


@dataclass
class RequestResult:
    r: int
    order: list
    depth: int
    tokens: np.ndarray
    table: list
    n_cached: int
    wave: int
    out: np.ndarray | None = None       # fp64 [s, Hq, D]


@dataclass
class RunResult:
    requests: list = field(default_factory=list)
    evictions: int = 0
    waves: int = 0


def attention_flops(Hq, D, n, c):
    """algorithmic FLOPs of one request: 4*Hq*D*[n(n+1)/2 - c(c+1)/2]."""
    return 4 * Hq * D * (n * (n + 1) // 2 - c * (c + 1) // 2)


def run_trace(trace, strategy: str = "greedy", compute: bool = True, requests=None, sample_rows=None):
    """strategy: 'greedy' (Algorithm 1) | 'retrieval' (identity, the comparison arm PAPER.md:155) | 'sorted' | 'recency' |
    'exhaustive' (the arms of Table 4, oracle/strategies.py) | 'greedy_feedback' (Algorithm 1 + stale marking from the
    engine's actual match) | 'greedy_resident' (Algorithm 1 confirmed by peeks on the real index,
    PAPER.md:314) — the NEXT-1 arms of oracle/ordering.py.
    compute=False does the host path only (order / lookup / tables).
    """
    cfg = trace.cfg
    tree = KnowledgeTree(cfg.H)
    recency = RecencyOrder()
    bm = BlockManager(cfg.NB, eager_register=True)
    pool = PagedPool(cfg.NB, cfg.Hkv, cfg.D) if compute else None
    res = RunResult()
    todo = list(range(cfg.n_req)) if requests is None else list(requests)
    wave_open, wave = [], 0

    def prefill(rr, req_id):
        if compute:
            rows = tracegen.prompt_qkv(trace, rr.r, rr.order, rr.n_cached)
            q, k, v = (tracegen.bf16_bits_to_f64(x) for x in tracegen.split_qkv(cfg, rows))
            rr.out = attention_suffix(pool, rr.table, rr.n_cached, q, k, v, cfg.theta)

    def close_wave():
        nonlocal wave
        for rr, req_id in wave_open:
            prefill(rr, req_id)
        for rr, req_id in wave_open:
            bm.release(req_id)
        wave_open.clear()
        wave += 1

    i = 0
    while i < len(todo):
        r = todo[i]
        D = trace.retrieval[r]
        if strategy in ("greedy", "greedy_feedback"):
            O, depth = tree.order(D)
        elif strategy == "greedy_resident":
            O, depth = tree.order_resident(D, lambda docs: bm.resident_prefix(tracegen.doc_prefix_tokens(trace, docs)))
        elif strategy == "retrieval":
            O, depth = list(D), tree.ell(D)
        elif strategy == "sorted":
            O = order_sorted(D)
            depth = tree.ell(O)
        elif strategy == "recency":
            O = recency.order(D)
            depth = tree.ell(O)
        elif strategy == "exhaustive":
            O, _ = order_exhaustive(list(D), lambda o: 16 * bm.match(tracegen.assemble_prompt(trace, r, o)))
            depth = tree.ell(O)
        else:
            raise ValueError(strategy)
        tokens = tracegen.assemble_prompt(trace, r, O)
        try:
            req_id, table, c = bm.lookup(tokens)
        except NoSpace:
            if not wave_open:
                raise
            close_wave()
            continue                        # retry the same request in the next wave (order() is pure)
        if strategy in ("greedy_feedback", "greedy_resident"):
            tree.feedback(O, depth, matched_docs(tracegen.doc_segment_ends(trace, O), c, len(tokens)))
        tree.observe(O)
        recency.observe(O)
        rr = RequestResult(r, O, depth, tokens, table, c, wave)
        res.requests.append(rr)
        wave_open.append((rr, req_id))
        if cfg.admission == "sequential":
            close_wave()
        i += 1
    if wave_open:
        close_wave()
    res.evictions = bm.evictions
    res.waves = wave
    return res


def full_recompute(trace, rr: RequestResult) -> np.ndarray:
    """full(n) of the same ordered prompt, no cache: the invariant 'prefix-cached == full recompute'."""
    cfg = trace.cfg
    rows = tracegen.prompt_qkv(trace, rr.r, rr.order, 0)
    q, k, v = (tracegen.bf16_bits_to_f64(x) for x in tracegen.split_qkv(cfg, rows))
    return attention_full(q, k, v, cfg.theta)
