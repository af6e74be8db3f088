"""Pins for the NEXT-1 part of the oracle (oracle/ordering.py: stale epochs, feedback, residency-aware Algorithm 1;
oracle/blocks.py: resident_prefix) — PAPER.md:129-141 (trie over-predicts after eviction; mark stale and stop relying on
it), PAPER.md:314 (use the engine's cache-state signal).  None of these re-types the oracle's own formula: hand-worked
epochs, the hand-worked block-table scenario of SURVEY.md §8(c7) (golden rows req5a_resident / req5a_after_feedback),
and properties against the exhaustive real-hit arm.
"""
import dataclasses

import numpy as np
import pytest

import tracegen
from conftest import golden
from oracle.blocks import BlockManager, matched_docs
from oracle.ordering import KnowledgeTree
from oracle.pipeline import run_trace


def test_stale_epoch_hand_worked():
    """seq 1: [A,B,C]; seq 2: [A,B,E]; then 'prefix A was resident, A,B was not' marks A->B at epoch 2.
    B is unusable, and so is everything below it, until served again; a re-served path is usable again but a sibling
    subtree served before the mark stays unusable (its blocks were released before B's and evicted first)."""
    T = KnowledgeTree(100)
    T.observe(list("ABC"))
    T.observe(list("ABE"))
    assert T.order(list("CBA")) == (list("ABC"), 3)            # no marks: plain Algorithm 1 (B then first child in rank)
    T.mark_stale(list("AB"), 1)
    assert T.ell(list("ABC")) == 1 and T.ell(list("ABE")) == 1
    assert T.order(list("CBA")) == (list("ACB"), 1)            # A, then nothing usable: rest in retrieval rank
    T.observe(list("ABF"))                                      # seq 3 > epoch 2: A, A->B, A->B->F usable again
    assert T.ell(list("ABF")) == 3
    assert T.ell(list("ABC")) == 2 and T.ell(list("ABE")) == 2  # C, E below B were last served at seq 1, 2 <= epoch 2
    assert T.order(list("EBA")) == (list("ABE"), 2)
    T.observe(list("ABE"))                                      # seq 4: that path is back
    assert T.ell(list("ABE")) == 3 and T.ell(list("ABC")) == 2
    assert T.brute_force_dfs(list("ABCE")) == 3 == T.brute_force_permutations(list("ABCE"))[1]


def test_feedback_only_marks_over_prediction():
    T = KnowledgeTree(100)
    T.observe(list("ABC"))
    T.feedback(list("ABC"), 3, 3)
    T.feedback(list("ABC"), 2, 3)                               # under-prediction is not an error of the trie
    assert T.ell(list("ABC")) == 3
    T.feedback(list("ABC"), 3, 0)                               # nothing was resident: the root child goes stale
    assert T.ell(list("ABC")) == 0
    T.mark_stale(list("XYZ"), 1)                                # unknown path: no-op


def _scenario_state():
    """state of the SURVEY.md §8(c7) scenario after req4 (golden rows req1..req4)."""
    g = golden("block_table_scenario.txt")
    rng = np.random.default_rng(123)
    docs = {c: rng.integers(0, 32000, 32, dtype=np.int32) for c in "ABCDEFG"}
    T, bm = KnowledgeTree(8), BlockManager(16, eager_register=True)
    for name in ["req1", "req2", "req3", "req4"]:
        retr = g[name].split("|")[0].split()
        O, _ = T.order(retr)
        T.observe(O)
        req, _, _ = bm.lookup(np.concatenate([docs[d] for d in O] + [rng.integers(0, 32000, 20, dtype=np.int32)]))
        bm.release(req)
    return g, docs, rng, T, bm


def test_scenario_resident_prefixes_after_req4():
    _, docs, _, _, bm = _scenario_state()
    cat = lambda names: np.concatenate([docs[d] for d in names])
    assert bm.resident_prefix(cat("A")) and bm.resident_prefix(cat("AC")) and bm.resident_prefix(cat("ACD"))
    assert bm.resident_prefix(cat("EFG"))
    assert not bm.resident_prefix(cat("AB")) and not bm.resident_prefix(cat("ABC")) and not bm.resident_prefix(cat("C"))
    assert bm.resident_prefix(np.zeros(0, dtype=np.int32)) and bm.resident_prefix(cat("A")[:15])   # no full block: vacuous


def test_scenario_req5a_residency_aware_order():
    g, docs, rng, T, bm = _scenario_state()
    retr, order, depth, m = [x.split() for x in g["req5a_resident"].split("|")]
    O, d = T.order_resident(retr, lambda names: bm.resident_prefix(np.concatenate([docs[x] for x in names])))
    assert (O, d) == (order, int(depth[0]))
    assert bm.match(np.concatenate([docs[x] for x in O] + [rng.integers(0, 32000, 20, dtype=np.int32)])) == int(m[0])
    assert T.ell(list("ABC")) == 1                              # A->B was marked stale by the failed peek


def test_scenario_req5a_feedback_then_greedy():
    g, docs, rng, T, bm = _scenario_state()
    O, pred = T.order(list("BCA"))                              # the plain path over-predicts (golden row req5a)
    assert (O, pred) == (list("ABC"), 3)
    c = 16 * bm.match(np.concatenate([docs[x] for x in O] + [rng.integers(0, 32000, 20, dtype=np.int32)]))
    assert c == 32
    T.feedback(O, pred, c // 32)                                # 32-token documents: 1 document was really cached
    retr, order, depth = [x.split() for x in g["req5a_after_feedback"].split("|")]
    assert T.order(retr) == (order, int(depth[0]))


@pytest.mark.parametrize("seed", range(4))
def test_resident_arm_predicts_exactly_and_never_beats_exhaustive(seed):
    """Small pool with heavy eviction (waves).  greedy_resident: predicted depth == documents really matched, for every
    request (block-aligned documents); per request, with the same cache state, no order matches more blocks than the
    exhaustive real-hit arm; over the trace the plain greedy arm over-predicts at least once (else the test is vacuous)."""
    base = tracegen.CONFIGS[1]
    cfg = dataclasses.replace(base, name=f"evict{seed}", seed=100 + seed, n_docs=8, doc_len=32, n_req=40, k=3, n_shared=2,
                              q_len=20, NB=24, H=12)
    trace = tracegen.make_trace(cfg)
    res = run_trace(trace, "greedy_resident", compute=False)
    for rr in res.requests:
        assert rr.depth == rr.n_cached // cfg.doc_len, (rr.r, rr.order, rr.depth, rr.n_cached)
    plain = run_trace(trace, "greedy", compute=False)
    over = sum(max(0, rr.depth - rr.n_cached // cfg.doc_len) for rr in plain.requests)
    fb = run_trace(trace, "greedy_feedback", compute=False)
    over_fb = sum(max(0, rr.depth - rr.n_cached // cfg.doc_len) for rr in fb.requests)
    assert over > 0 and over_fb <= over
    # same-state comparison with the exhaustive arm: replay the resident arm's state and peek all permutations
    from itertools import permutations
    from oracle.ordering import KnowledgeTree as KT
    T, bm = KT(cfg.H), BlockManager(cfg.NB)
    for r in range(cfg.n_req):
        D = trace.retrieval[r]
        O, _ = T.order_resident(D, lambda docs: bm.resident_prefix(tracegen.doc_prefix_tokens(trace, docs)))
        got = bm.match(tracegen.assemble_prompt(trace, r, O))
        best = max(bm.match(tracegen.assemble_prompt(trace, r, [D[i] for i in p])) for p in permutations(range(cfg.k)))
        assert got <= best
        req, _, c = bm.lookup(tracegen.assemble_prompt(trace, r, O))
        T.feedback(O, T.ell(O), c // cfg.doc_len)
        T.observe(O)
        bm.release(req)


def test_matched_docs_hand_worked_ragged_segments():
    """oracle.blocks.matched_docs on a hand-worked literal-layout prompt: 30 instruction tokens, then per document a
    7-token header, the passage and a blank-line token; passages of 200, 190 and 206 tokens, a 50-token question part:
       doc ends 30+208 = 238, 238+198 = 436, 436+214 = 650; n = 700.
    Full blocks up to each end: 224, 432, 640 tokens.  A lookup that returned n_cached = 224 served document 1 whole
    (its last 14 tokens share a block with header 2 and can never match alone); 432 serves two, 640 all three; one block
    less each time loses the document."""
    ends, n = [238, 436, 650], 700
    assert [matched_docs(ends, c, n) for c in (0, 208, 224, 416, 432, 624, 640, 688)] == [0, 0, 1, 1, 2, 2, 3, 3]
    assert matched_docs([], 64, 100) == 0


def test_matched_docs_does_not_punish_the_lookup_cap():
    """Three block-aligned 32-token documents and NO query: n = 96, and a lookup can return at most 16*floor(95/16) = 80
    cached tokens.  With everything resident (n_cached = 80) all three documents count (the uncapped rule
    said 2, so the feedback arm marked a fully resident leaf stale on every repeat).  With a one-token query (n = 97) the
    cap is 96 and the third document needs n_cached = 96."""
    assert matched_docs([32, 64, 96], 80, 96) == 3
    assert matched_docs([32, 64, 96], 64, 96) == 2
    assert matched_docs([32, 64, 96], 80, 97) == 2
    assert matched_docs([32, 64, 96], 96, 97) == 3


def _all_nodes(tree):
    stack, out = [tree.root], []
    while stack:
        node = stack.pop()
        for c in node.children.values():
            out.append(c)
            stack.append(c)
    return out


def test_repeated_prompt_without_query_is_never_marked_stale():
    """the same 3 documents, no query, served repeatedly through the oracle pipeline with the feedback arm: predicted ==
    actual on every repeat and no node is ever marked stale."""
    bm, tree = BlockManager(24), KnowledgeTree(12)
    rng = np.random.default_rng(0)
    docs = {d: rng.integers(0, 32000, size=32, dtype=np.int32) for d in (5, 6, 7)}
    for rep in range(4):
        O, depth = tree.order([7, 5, 6])
        tokens = np.concatenate([docs[d] for d in O])
        req, table, c = bm.lookup(tokens)
        actual = matched_docs([32, 64, 96], c, len(tokens))
        assert (depth, actual, c) == ((0, 0, 0) if rep == 0 else (3, 3, 80))
        tree.feedback(O, depth, actual)
        tree.observe(O)
        bm.release(req)
        assert all(node.stale_epoch == 0 for node in _all_nodes(tree))
