"""Trace driver: runs a synthetic RAG trace (tracegen) through the C-ABI path, request by request / wave by wave.

Orchestration only — every step of the path (ordering, hashing, block management, RoPE + scatter, attention) is a
cw_* call into libcacheweaver.so.  Per request:
    O = cw_order(D); tokens = docs[O] ‖ query; (table, c) = cw_lookup(tokens); cw_observe(O)
then per wave ONE cw_append_kv + ONE cw_prefill_attn over all suffixes, then cw_release.
Admission "sequential": a wave is one request.  Admission "waves": requests are admitted until cw_lookup reports
CW_ERR_NO_SPACE, the wave is prefilled and released, and admission resumes.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

import tracegen
from .binding import BLOCK_SIZE, Context, NoSpace


@dataclass
class RequestRecord:
    r: int
    order: list
    depth: int
    tokens: np.ndarray
    table: np.ndarray
    n_cached: int
    wave: int
    out: np.ndarray | None = None        # bf16 bits, uint16 [s, Hq, D]


@dataclass
class Wave:
    items: list                          # (r, order, n_cached)
    cu: np.ndarray                       # int32 [B+1]
    nc: np.ndarray                       # int32 [B]
    tables: np.ndarray                   # int32 [B, max_blocks]
    recs: list = field(default_factory=list)
    reqs: np.ndarray | None = None       # int64 [B] request handles, valid until the wave is released

    @property
    def B(self):
        return len(self.nc)

    @property
    def T(self):
        return int(self.cu[-1])

    @property
    def max_blocks(self):
        return int(self.tables.shape[1])

    @property
    def max_q(self):
        return int(np.diff(self.cu).max())

    @property
    def max_kv(self):
        return int((self.nc + np.diff(self.cu)).max())


def make_context(cfg: tracegen.Config, device=None, max_position=None) -> Context:
    return Context(cfg.NB, cfg.Hq, cfg.Hkv, cfg.D, cfg.H, rope_theta=cfg.theta,
                   max_position=max_position or cfg.n, eager_register=True, device=device)


def attention_flops(Hq, D, n, c):
    """algorithmic FLOPs of one request: 4*Hq*D*[n(n+1)/2 - c(c+1)/2] (unmasked pairs; QK^T + PV)."""
    return 4 * Hq * D * (n * (n + 1) // 2 - c * (c + 1) // 2)


def append_bytes(cfg: tracegen.Config, T):
    """algorithmic bytes of cw_append_kv for T suffix tokens: q in + q' out + k,v in + pool out + 4 B descriptor."""
    return T * (2 * cfg.Hq * cfg.D * 2 + 2 * 2 * cfg.Hkv * cfg.D * 2 + 4)


class TraceRunner:
    def __init__(self, trace: tracegen.Trace, strategy: str = "greedy", device=None, ctx: Context | None = None):
        self.trace, self.cfg, self.strategy, self.device = trace, trace.cfg, strategy, device
        self.ctx = ctx or make_context(trace.cfg, device)
        self.waves: list[Wave] = []
        self.records: list[RequestRecord] = []

    # ---- host path -----------------------------------------------------------------------------------------
    def _admit(self, r):
        D = self.trace.retrieval[r]
        if self.strategy in ("greedy", "greedy_feedback"):
            O, depth = self.ctx.cw_order(D)
        elif self.strategy == "retrieval":
            O, depth = list(D), self.ctx.cw_predict(D)
        elif self.cfg.layout != "plain":
            raise ValueError("the token-based arms of cw_order_arm assemble docs ‖ query; use greedy / retrieval / "
                             "greedy_feedback with the literal prompt layout")
        else:                                              # sorted | recency | exhaustive | greedy_resident (cw_order_arm)
            O, depth = self.ctx.cw_order_arm(self.strategy, D, self.trace.doc_tokens, self.trace.query_tokens[r])
        tokens = tracegen.assemble_prompt(self.trace, r, O)
        req, table, c = self.ctx.cw_lookup(tokens)        # raises NoSpace with state unchanged
        if self.strategy in ("greedy_feedback", "greedy_resident"):
            self.ctx.cw_feedback_tokens(O, depth, tracegen.doc_segment_ends(self.trace, O), c, len(tokens))
        self.ctx.cw_observe(O)
        return req, RequestRecord(r, O, depth, tokens, table, c, len(self.waves))

    def run(self, compute: bool = True, keep_outputs: bool = True, requests=None, on_wave=None):
        """Runs the whole trace.  compute=False: host path only (orders, block tables, hit counts)."""
        cfg = self.cfg
        todo = list(range(cfg.n_req)) if requests is None else list(requests)
        open_wave, i = [], 0

        def close_wave():
            recs = [rec for _, rec in open_wave]
            tables = np.zeros((len(recs), max(len(rec.table) for rec in recs)), dtype=np.int32)
            for b, rec in enumerate(recs):
                tables[b, : len(rec.table)] = rec.table
            s = np.array([len(rec.tokens) - rec.n_cached for rec in recs], dtype=np.int64)
            cu = np.zeros(len(recs) + 1, dtype=np.int32)
            cu[1:] = np.cumsum(s)
            wave = Wave([(rec.r, rec.order, rec.n_cached) for rec in recs], cu,
                        np.array([rec.n_cached for rec in recs], dtype=np.int32), tables, recs,
                        np.array([req for req, _ in open_wave], dtype=np.int64))
            if compute:
                self.prefill_wave(wave, keep_outputs)
            if on_wave is not None:
                on_wave(wave)
            for req, _ in open_wave:
                self.ctx.cw_release(req)
            self.waves.append(wave)
            self.records.extend(recs)
            open_wave.clear()

        while i < len(todo):
            try:
                req, rec = self._admit(todo[i])
            except NoSpace:
                if not open_wave:
                    raise
                close_wave()
                continue
            open_wave.append((req, rec))
            if cfg.admission == "sequential":
                close_wave()
            i += 1
        if open_wave:
            close_wave()
        return self.records

    # ---- device path ---------------------------------------------------------------------------------------
    def wave_inputs(self, wave: Wave):
        """seeded bf16 activations of the wave's suffix rows -> device tensors q [T,Hq,D], k, v [T,Hkv,D]."""
        import torch
        cfg = self.cfg
        rows = tracegen.batch_suffix_qkv(self.trace, wave.items)
        q, k, v = tracegen.split_qkv(cfg, rows)
        return tuple(torch.from_numpy(x.view(np.int16)).view(torch.bfloat16).to(self.device, non_blocking=False)
                     for x in (q, k, v))

    def wave_descriptors(self, wave: Wave):
        import torch
        d_cu = torch.from_numpy(wave.cu).to(self.device)
        d_nc = torch.from_numpy(wave.nc).to(self.device)
        d_tables = torch.from_numpy(wave.tables).to(self.device)
        d_work = torch.empty(self.ctx.cw_attn_work_ints(wave.B, wave.T), dtype=torch.int32, device=self.device)
        return d_cu, d_nc, d_tables, d_work

    def prefill_wave(self, wave: Wave, keep_outputs: bool = True):
        import torch
        q, k, v = self.wave_inputs(wave)
        d_cu, d_nc, d_tables, d_work = self.wave_descriptors(wave)
        q_roped, out = torch.empty_like(q), torch.empty_like(q)
        self.ctx.cw_append_kv(q, k, v, q_roped, d_cu, d_nc, d_tables, wave.max_blocks, wave.B, wave.T)
        s = np.diff(wave.cu)
        self.ctx.cw_prefill_attn(q_roped, out, d_cu, d_nc, d_tables, wave.max_blocks, wave.B, wave.T,
                                 int(s.max()), int((wave.nc + s).max()), d_work)
        torch.cuda.synchronize()
        if int(d_work[1]) != 0:
            raise RuntimeError("cw_prefill_attn rejected a request descriptor on the device")
        if keep_outputs:
            o = out.view(torch.int16).cpu().numpy().view(np.uint16)
            for b, rec in enumerate(wave.recs):
                rec.out = o[wave.cu[b]: wave.cu[b + 1]]
        return q_roped, out


def admit_waves(ctx: Context, trace: tracegen.Trace, strategy: str = "greedy", requests=None, on_wave=None,
                force_waves: bool = True):
    """Whole-trace admission through cw_admit_batch (one C call per wave) + cw_release_batch.
    Admission "waves" (or force_waves): as many requests as fit are admitted, the wave is handed to on_wave (which
    launches the kernels), released, and admission resumes.  Admission "sequential": one request per wave.
    Returns the list of Wave objects (recs hold order / depth / table / n_cached, tokens omitted)."""
    cfg = trace.cfg
    todo = list(range(cfg.n_req)) if requests is None else list(requests)
    doc_ids = np.asarray([trace.retrieval[r] for r in todo], dtype=np.int64).reshape(len(todo), cfg.k)
    queries = np.ascontiguousarray(trace.query_tokens[todo])
    waves, i = [], 0
    step = None if (force_waves or cfg.admission == "waves") else 1
    while i < len(todo):
        j = len(todo) if step is None else min(len(todo), i + step)
        a = ctx.cw_admit_batch(doc_ids[i:j], strategy, trace.doc_tokens, queries[i:j], cfg.blocks_per_req)
        m = a["admitted"]
        if m == 0:
            raise NoSpace(-2, "a single request does not fit the pool")
        recs = [RequestRecord(todo[i + b], a["orders"][b].tolist(), int(a["pred"][b]), None,
                              a["tables"][b, : cfg.blocks_per_req].copy(), int(a["n_cached"][b]), len(waves))
                for b in range(m)]
        wave = Wave([(rec.r, rec.order, rec.n_cached) for rec in recs], a["cu"][: m + 1].copy(), a["n_cached"][:m].copy(),
                    a["tables"][:m].copy(), recs, a["reqs"][:m].copy())
        if on_wave is not None:
            on_wave(wave)
        ctx.cw_release_batch(a["reqs"][:m])
        waves.append(wave)
        i += m
    return waves
