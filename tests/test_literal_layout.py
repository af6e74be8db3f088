"""NEXT-3: the paper-literal prompt layout — "a fixed instruction, then the ordered evidence blocks under
[Document r: id] headers, then the query" (App. A), ~200-token passages that
are not multiples of the 16-token block.  tracegen.segments builds it from reserved header tokens (no tokenizer here).

Pins that do not re-type the code under test: the three properties the paper states for this layout (shared instruction;
evidence before the query; the rank r inside the header), turned into matched-block counts that are
worked out by hand from the segment lengths."""
import dataclasses

import numpy as np
import pytest

import tracegen
from oracle.blocks import BlockManager, matched_docs
from oracle.pipeline import run_trace
from paper_2606_19667_b200.engine import TraceRunner


def literal_config(**kw):
    d = dict(name="literal-small", seed=11, n_docs=12, doc_len=200, doc_jitter=20, n_req=24, k=4, n_shared=3, q_len=24,
             NB=600, H=8, layout="literal")
    d.update(kw)
    return dataclasses.replace(tracegen.CONFIGS[1], **d)


def test_layout_structure():
    trace = tracegen.make_trace(literal_config())
    O = trace.retrieval[0]
    segs = tracegen.segments(trace, 0, O)
    assert [k[0] for k, _ in segs] == [2, 0, 0, 0, 0, 1]
    assert len(segs[0][1]) == tracegen.INSTR_LEN and np.array_equal(segs[0][1], tracegen.segments(trace, 5, trace.retrieval[5])[0][1])
    for j, (key, t) in enumerate(segs[1:-1]):
        d = O[j]
        assert key == (0, *O[: j + 1]) and len(t) == 7 + trace.doc_lens[d] + 1
        assert t[2] == tracegen.T_RANK0 + j + 1 and t[4] == tracegen.T_DOCID0 + d          # rank and id sit in the header
        assert 180 <= trace.doc_lens[d] <= 220
    q = segs[-1][1]
    assert len(q) == 2 + 24 + 3 and q[0] == tracegen.T_QUESTION and q[-2] == tracegen.T_ANSWER
    n = sum(len(t) for _, t in segs)
    assert n == len(tracegen.assemble_prompt(trace, 0, O)) <= trace.cfg.n
    assert any(trace.doc_lens % 16 != 0)


def test_divergence_points_by_hand():
    """request 1 served with order [A, B, C, D].  Hand-worked matches of a second prompt (peek):
      same order, other query        -> everything up to the block holding the query's first differing token
      [A, B, D, C]                   -> instruction + blocks of A and B + the part of header 3 before the doc id ('[', 'Document', rank 3, ':')
      [B, A, C, D] (A at rank 2)     -> the instruction and the first 4 header tokens only: 34 tokens -> 2 blocks
    """
    trace = tracegen.make_trace(literal_config())
    A, B, C, D = trace.retrieval[0]
    bm = BlockManager(600)
    req, _, _ = bm.lookup(tracegen.assemble_prompt(trace, 0, [A, B, C, D]))
    L = lambda d: 7 + int(trace.doc_lens[d]) + 1
    evid = 30 + L(A) + L(B) + L(C) + L(D)
    assert bm.match(tracegen.assemble_prompt(trace, 1, [A, B, C, D])) == (evid + 2) // 16     # 'Question', ':' are shared too
    assert bm.match(tracegen.assemble_prompt(trace, 1, [A, B, D, C])) == (30 + L(A) + L(B) + 4) // 16
    assert bm.match(tracegen.assemble_prompt(trace, 1, [B, A, C, D])) == 34 // 16 == 2
    # the aligned plain layout has no header: the same swap of the last two documents keeps both leading documents whole
    plain = tracegen.make_trace(dataclasses.replace(literal_config(), layout="plain", doc_len=208, doc_jitter=0))
    A, B, C, D = plain.retrieval[0]
    bm2 = BlockManager(600)
    bm2.lookup(tracegen.assemble_prompt(plain, 0, [A, B, C, D]))
    assert bm2.match(tracegen.assemble_prompt(plain, 1, [A, B, D, C])) == 2 * 13
    assert bm2.match(tracegen.assemble_prompt(plain, 1, [B, A, C, D])) == 0


@pytest.mark.parametrize("strategy", ["retrieval", "greedy", "greedy_feedback"])
def test_library_matches_oracle_on_the_literal_layout(strategy):
    trace = tracegen.make_trace(literal_config())
    ref = run_trace(trace, strategy, compute=False)
    recs = TraceRunner(trace, strategy, device=None).run(compute=False)
    for a, o in zip(recs, ref.requests):
        assert (a.order, a.depth, a.n_cached, a.table.tolist()) == (o.order, o.depth, o.n_cached, list(o.table)), a.r
        assert np.array_equal(a.tokens, o.tokens)
    if strategy == "greedy":
        hits = sum(o.n_cached for o in ref.requests)
        base = sum(o.n_cached for o in run_trace(trace, "retrieval", compute=False).requests)
        assert hits > base >= 16 * (len(ref.requests) - 1)        # the instruction block is always reused; greedy adds to it


def test_feedback_does_not_punish_the_lost_partial_block():
    """With unaligned documents the block a document shares with the next header is never matched; a document counts as
    matched when all its FULL blocks are (oracle.blocks.matched_docs), so the feedback arm marks nothing stale without eviction
    and orders exactly like plain greedy."""
    trace = tracegen.make_trace(literal_config())
    a = run_trace(trace, "greedy", compute=False)
    b = run_trace(trace, "greedy_feedback", compute=False)
    assert [r.order for r in a.requests] == [r.order for r in b.requests]
    assert all(r.depth == matched_docs(tracegen.doc_segment_ends(trace, r.order), r.n_cached, len(r.tokens)) for r in a.requests)


@pytest.mark.gpu
def test_literal_layout_trace_on_the_gpu():
    """the whole path on the literal layout (ragged prompts: 1.0-1.1k tokens, suffix lengths that are not multiples of 16
    from the second wave on): orders / tables bit-exact, every output row within the north_star tolerance."""
    torch = pytest.importorskip("torch")
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device (there is no CPU fallback)")
    trace = tracegen.make_trace(literal_config(n_req=8, Hq=4, Hkv=2, D=128, theta=5e5))
    ref = run_trace(trace, "greedy")
    recs = TraceRunner(trace, "greedy", device="cuda:0").run()
    worst = 0.0
    for a, o in zip(recs, ref.requests):
        assert (a.order, a.depth, a.n_cached, a.table.tolist()) == (o.order, o.depth, o.n_cached, list(o.table))
        got = tracegen.bf16_bits_to_f64(a.out).reshape(o.out.shape)
        d = got - o.out
        assert np.abs(d).max() <= 2e-2 and np.linalg.norm(d) / np.linalg.norm(o.out) <= 1e-2, a.r
        worst = max(worst, float(np.abs(d).max()))
    assert sum(a.n_cached for a in recs) > 0
