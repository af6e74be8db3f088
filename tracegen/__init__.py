"""Seeded synthetic inputs for the prefix-cached prefill path (shared by the oracle and the CUDA path).

This module holds NO arithmetic of the method: no ordering, hashing, block management, RoPE or attention.
It only draws the synthetic RAG traces of SURVEY.md §8(d) (document pools, retrieval lists, queries) and
the bf16 Q/K/V activations, and concatenates prompt pieces.  Both `oracle/` and the tests/bench of the CUDA
path import it; neither imports the other.

The traces stand in for the paper's controlled synthetic bursty corpus (§4 "Workload":
topical regions, ~200-token passages, top-k 5, adjacent-query overlap) and its sweeps (Table 5 top-k,
Figure 4 overlap, Table 11 concurrency); the authors' generator and traces are not available.

Q/K/V are *keyed by the document prefix*: the activation chunk for document O[j] of a request is drawn from
a generator seeded by (config seed, O[0..j]); query chunks by (config seed, request index).  Identical
document prefix => identical pre-RoPE Q/K/V, different prefix => different values, as in a real
transformer, so a false cache hit cannot pass the "prefix-cached == full recompute" parity check.
"""
from __future__ import annotations

from concurrent.futures import ThreadPoolExecutor
from dataclasses import dataclass, field

import numpy as np

BLOCK_SIZE = 16  # PAPER.md:39 "the token block size is 16 tokens"

# Paper-literal prompt layout ("a fixed instruction, then the ordered evidence blocks
# under [Document r: id] headers, then the query"; App. A).  There is no tokenizer here, so the template's
# fixed strings are stood in for by reserved token ids outside the corpus vocabulary [0, 32000):
#   instruction  INSTR_LEN seeded corpus-vocabulary tokens, the same for every request of a trace (~30 words in App. A)
#   header(r, d) "[", "Document", rank r, ":", doc id d, "]", newline          -> HEADER_LEN tokens; contains the RANK
#   separator    blank line after the document text                             -> SEP_LEN token
#   query        "Question", ":", <query tokens>, newline, "Answer", ":"        -> QHEAD_LEN + q_len + QTAIL_LEN tokens
INSTR_LEN, HEADER_LEN, SEP_LEN, QHEAD_LEN, QTAIL_LEN = 30, 7, 1, 2, 3
T_LBRACKET, T_DOCUMENT, T_COLON, T_RBRACKET, T_NEWLINE, T_BLANKLINE, T_QUESTION, T_ANSWER = range(32000, 32008)
T_RANK0, T_DOCID0 = 32100, 33000


@dataclass(frozen=True)
class Config:
    name: str
    seed: int
    n_docs: int          # pool size (per cluster for mode "zipf")
    doc_len: int
    n_req: int
    k: int               # top-k
    n_shared: int        # docs shared with the previous request (mode "overlap")
    q_len: int           # query tokens
    Hq: int
    Hkv: int
    D: int
    NB: int              # KV pool blocks
    H: int               # recency window (floor(NB / ceil(n/16)))
    theta: float
    mode: str = "overlap"    # "overlap" | "zipf"
    n_clusters: int = 1
    zipf_s: float = 1.1
    admission: str = "sequential"   # "sequential" | "waves"
    layout: str = "plain"    # "plain": docs ‖ query (north_star) | "literal": the paper's template (App. A), see segments()
    doc_jitter: int = 0      # layout "literal": document lengths are drawn from U[doc_len - jitter, doc_len + jitter]

    @property
    def n(self) -> int:
        """prompt length in tokens; for the literal layout (ragged documents) the largest possible one."""
        if self.layout == "literal":
            return INSTR_LEN + self.k * (HEADER_LEN + self.doc_len + self.doc_jitter + SEP_LEN) + QHEAD_LEN + self.q_len + QTAIL_LEN
        return self.k * self.doc_len + self.q_len

    @property
    def blocks_per_req(self) -> int:
        return -(-self.n // BLOCK_SIZE)

    @property
    def width(self) -> int:
        """elements per token of the packed [q | k | v] activation row."""
        return (self.Hq + 2 * self.Hkv) * self.D


def n_shared_for(overlap_pct: int, k: int) -> int:
    """n_shared = floor(overlap*k + 0.5)."""
    return int(np.floor(overlap_pct / 100.0 * k + 0.5))


CONFIGS = {
    # BASELINE.json configs[0..4]
    1: Config("cfg1-tiny", 0, 10, 64, 4, 3, 2, 32, 2, 1, 64, 64, 4, 1e4),
    2: Config("cfg2-llama3-8b", 0, 200, 256, 64, 5, 3, 48, 32, 8, 128, 8192, 98, 5e5),
    4: Config("cfg4-qwen2.5-7b-concurrent", 0, 50, 512, 256, 10, 0, 64, 28, 4, 128, 32768, 101, 1e6,
              mode="zipf", n_clusters=8, admission="waves"),
    5: Config("cfg5-70b-long", 0, 400, 512, 32, 20, 10, 64, 64, 8, 128, 16384, 25, 5e5, admission="waves"),
}


def config3(k: int, overlap_pct: int, n_req: int = 128) -> Config:
    """Overlap/top-k sweep cell at the 8B shapes (BASELINE.json configs[2]); inherits cfg 2."""
    n = k * 256 + 48
    nb = 8192
    return Config(f"cfg3-k{k}-ov{overlap_pct}", 1000 * k + overlap_pct, 200, 256, n_req, k,
                  n_shared_for(overlap_pct, k), 48, 32, 8, 128, nb, nb // (-(-n // BLOCK_SIZE)), 5e5)


@dataclass
class Trace:
    cfg: Config
    doc_tokens: np.ndarray              # int32 [total_docs, doc_len] (layout "literal": padded to the longest document)
    retrieval: list                     # n_req lists of int64 doc ids, in retrieval rank
    query_tokens: np.ndarray            # int32 [n_req, q_len]
    doc_lens: np.ndarray | None = None  # int32 [total_docs], layout "literal" only
    instr_tokens: np.ndarray | None = None   # int32 [INSTR_LEN], layout "literal" only
    _chunks: dict = field(default_factory=dict, repr=False)


def make_trace(cfg: Config) -> Trace:
    """Everything derived in a fixed order from one PCG64 generator seeded with cfg.seed."""
    rng = np.random.default_rng(cfg.seed)
    total_docs = cfg.n_docs * cfg.n_clusters
    doc_tokens = rng.integers(0, 32000, size=(total_docs, cfg.doc_len + (cfg.doc_jitter if cfg.layout == "literal" else 0)),
                              dtype=np.int32)
    retrieval = []
    if cfg.mode == "overlap":
        prev = None
        for _ in range(cfg.n_req):
            if prev is None:
                docs = rng.choice(total_docs, size=cfg.k, replace=False)
            else:
                shared = rng.choice(prev, size=cfg.n_shared, replace=False)
                rest = np.setdiff1d(np.arange(total_docs), prev)
                fresh = rng.choice(rest, size=cfg.k - cfg.n_shared, replace=False)
                docs = np.concatenate([shared, fresh])
                rng.shuffle(docs)
            prev = docs.copy()
            retrieval.append([int(d) for d in docs])
    elif cfg.mode == "zipf":
        w = np.arange(1, cfg.n_docs + 1, dtype=np.float64) ** (-cfg.zipf_s)
        w /= w.sum()
        for _ in range(cfg.n_req):
            c = int(rng.integers(0, cfg.n_clusters))
            docs = rng.choice(cfg.n_docs, size=cfg.k, replace=False, p=w)   # draw order = retrieval order
            retrieval.append([int(c * cfg.n_docs + d) for d in docs])
    else:
        raise ValueError(cfg.mode)
    query_tokens = rng.integers(0, 32000, size=(cfg.n_req, cfg.q_len), dtype=np.int32)
    if cfg.layout == "literal":      # drawn last, so the plain-layout traces of the same seed are unchanged
        doc_lens = rng.integers(cfg.doc_len - cfg.doc_jitter, cfg.doc_len + cfg.doc_jitter + 1, size=total_docs).astype(np.int32)
        instr = rng.integers(0, 32000, size=INSTR_LEN, dtype=np.int32)
        return Trace(cfg, doc_tokens, retrieval, query_tokens, doc_lens, instr)
    return Trace(cfg, doc_tokens, retrieval, query_tokens)


def jaccard(a, b) -> float:
    """|A∩B|/|A∪B| between two retrieved sets — a trace statistic, not part of the method."""
    a, b = set(a), set(b)
    return len(a & b) / len(a | b)


def segments(trace: Trace, r, order):
    """The prompt of request r under `order` as a list of (key, tokens) segments; the key names what the segment's
    activations depend on (the document PREFIX for evidence blocks), r = None leaves the query segment out.
      plain   : [doc O[0]] … [doc O[k-1]] [query]                                  (north_star: docs then query)
      literal : [instruction] [header(1, O[0]) doc O[0] blank line] … [Question: query \n Answer:]   (App. A)"""
    cfg = trace.cfg
    i32 = lambda xs: np.asarray(xs, dtype=np.int32)
    segs = []
    if cfg.layout == "literal":
        segs.append(((2,), trace.instr_tokens))
        for j, d in enumerate(order):
            d = int(d)
            hdr = i32([T_LBRACKET, T_DOCUMENT, T_RANK0 + j + 1, T_COLON, T_DOCID0 + d, T_RBRACKET, T_NEWLINE])
            segs.append(((0, *[int(x) for x in order[: j + 1]]),
                         np.concatenate([hdr, trace.doc_tokens[d, : trace.doc_lens[d]], i32([T_BLANKLINE])])))
        if r is not None:
            segs.append(((1, int(r)), np.concatenate([i32([T_QUESTION, T_COLON]), trace.query_tokens[r],
                                                      i32([T_NEWLINE, T_ANSWER, T_COLON])])))
    else:
        for j, d in enumerate(order):
            segs.append(((0, *[int(x) for x in order[: j + 1]]), trace.doc_tokens[int(d)]))
        if r is not None:
            segs.append(((1, int(r)), trace.query_tokens[r]))
    return segs


def assemble_prompt(trace: Trace, r: int, order) -> np.ndarray:
    """a3: the prompt tokens of request r with its documents in `order` (see segments())."""
    return np.ascontiguousarray(np.concatenate([t for _, t in segments(trace, r, order)]), dtype=np.int32)


def doc_prefix_tokens(trace: Trace, docs) -> np.ndarray:
    """tokens of the prompt prefix that ends with the leading documents `docs` (no query): what a residency peek looks up."""
    parts = [t for _, t in segments(trace, None, docs)]
    if not parts:
        return np.zeros(0, dtype=np.int32)
    return np.ascontiguousarray(np.concatenate(parts), dtype=np.int32)


def doc_segment_ends(trace: Trace, order) -> list:
    """prompt position just past the segment of each document of `order` (cumulative segment lengths: prompt structure
    only — what counts as a matched document is decided by the oracle and by the library, each on its own)."""
    pos, ends = 0, []
    for key, t in segments(trace, None, order):
        pos += len(t)
        if key[0] == 0:
            ends.append(pos)
    return ends


def f32_to_bf16_bits(x: np.ndarray) -> np.ndarray:
    """float32 -> bf16 bit pattern (uint16), round-to-nearest-even.  Input conversion only."""
    u = np.ascontiguousarray(x, dtype=np.float32).view(np.uint32)
    return ((u + np.uint32(0x7FFF) + ((u >> np.uint32(16)) & np.uint32(1))) >> np.uint32(16)).astype(np.uint16)


def bf16_bits_to_f64(b: np.ndarray) -> np.ndarray:
    """bf16 bit pattern (uint16) -> float64, exact."""
    return (np.ascontiguousarray(b, dtype=np.uint16).astype(np.uint32) << np.uint32(16)).view(np.float32).astype(np.float64)


def _chunk(seed: int, key: tuple, length: int, width: int) -> np.ndarray:
    g = np.random.Generator(np.random.PCG64(np.random.SeedSequence([seed, *key])))
    return f32_to_bf16_bits(g.standard_normal((length, width), dtype=np.float32))


def qkv_chunk_keys(trace: Trace, r: int, order):
    """(key, length) of each activation chunk of request r's prompt under `order` (one chunk per prompt segment)."""
    if trace.cfg.layout == "plain":          # no token arrays needed: fixed lengths
        cfg = trace.cfg
        keys = [((0, *[int(d) for d in order[: j + 1]]), cfg.doc_len) for j in range(len(order))]
        keys.append(((1, int(r)), cfg.q_len))
        return keys
    return [(key, len(t)) for key, t in segments(trace, r, order)]


def prompt_qkv(trace: Trace, r: int, order, start: int = 0, cache: bool = False) -> np.ndarray:
    """bf16 bits, uint16 [n - start, (Hq+2Hkv)*D]: packed rows [q heads | k heads | v heads] for prompt
    positions start..n-1 of request r under `order`.  N(0,1) rounded to bf16 (BASELINE.json configs)."""
    cfg = trace.cfg
    out, pos = [], 0
    for key, length in qkv_chunk_keys(trace, r, order):
        if pos + length > start:
            if cache and key in trace._chunks:
                c = trace._chunks[key]
            else:
                c = _chunk(cfg.seed, key, length, cfg.width)
                if cache:
                    trace._chunks[key] = c
            out.append(c[max(0, start - pos):])
        pos += length
    return np.concatenate(out, axis=0)


def batch_suffix_qkv(trace: Trace, items, threads: int = 8) -> np.ndarray:
    """items: list of (r, order, n_cached).  Returns the concatenated suffix rows (uint16 [T, width])."""
    with ThreadPoolExecutor(max_workers=threads) as ex:
        parts = list(ex.map(lambda it: prompt_qkv(trace, it[0], it[1], it[2]), items))
    return np.concatenate(parts, axis=0)


def split_qkv(cfg: Config, rows: np.ndarray):
    """packed rows -> (q [T,Hq,D], k [T,Hkv,D], v [T,Hkv,D]) contiguous copies (uint16 bf16 bits)."""
    T = rows.shape[0]
    a, b = cfg.Hq * cfg.D, (cfg.Hq + cfg.Hkv) * cfg.D
    q = np.ascontiguousarray(rows[:, :a]).reshape(T, cfg.Hq, cfg.D)
    k = np.ascontiguousarray(rows[:, a:b]).reshape(T, cfg.Hkv, cfg.D)
    v = np.ascontiguousarray(rows[:, b:]).reshape(T, cfg.Hkv, cfg.D)
    return q, k, v
