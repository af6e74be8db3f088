"""Ordering arms of the paper's Table 4: sorted, recency, exhaustive — SURVEY.md §8(f) NEXT-2.
Oracle pins (hand-worked cases, brute force) and bit-exact agreement of cw_order_arm / cw_admit_batch with the oracle."""
import itertools

import numpy as np
import pytest

import tracegen
from oracle.blocks import BlockManager
from oracle.ordering import KnowledgeTree
from oracle.pipeline import run_trace
from oracle.strategies import RecencyOrder, order_exhaustive, order_sorted
from paper_2606_19667_b200 import ARMS, Context, CwError
from paper_2606_19667_b200.engine import TraceRunner, admit_waves, make_context


# ---- oracle pins ------------------------------------------------------------------------------------------
def test_sorted_is_canonical_and_query_independent():
    assert order_sorted([7, 3, 9, 1]) == [1, 3, 7, 9]
    for perm in itertools.permutations([4, 2, 8]):
        assert order_sorted(list(perm)) == [2, 4, 8]            # the same order whatever the retrieval rank


def test_recency_hand_worked():
    r = RecencyOrder()
    assert r.order([5, 3, 9]) == [5, 3, 9]                      # nothing served yet: retrieval rank
    r.observe([1, 2])                                           # seq 1
    r.observe([3, 1])                                           # seq 2: last_served = {1: 2, 2: 1, 3: 2}
    assert r.order([2, 9, 1, 3]) == [1, 3, 2, 9]                # seq 2 (1 then 3, retrieval rank), seq 1, never served
    r.observe([9])                                              # seq 3
    assert r.order([2, 9, 1, 3]) == [9, 1, 3, 2]


def test_exhaustive_first_maximiser_and_brute_force():
    score = {(2, 1, 3): 48, (1, 2, 3): 48, (3, 2, 1): 16}
    O, c = order_exhaustive([1, 2, 3], lambda o: score.get(tuple(o), 0))
    assert (O, c) == ([1, 2, 3], 48)                            # ties: first in lexicographic order of rank indices
    O, c = order_exhaustive([3, 1], lambda o: 0)
    assert (O, c) == ([3, 1], 0)                                # nothing cached: retrieval order


def test_exhaustive_is_the_optimum_of_the_real_block_index():
    """on the same cache state no other permutation matches more blocks; greedy may match fewer (trie over-prediction)."""
    cfg = tracegen.CONFIGS[1]
    trace = tracegen.make_trace(cfg)
    bm, tree = BlockManager(cfg.NB), KnowledgeTree(cfg.H)
    for r in range(cfg.n_req):
        D = trace.retrieval[r]
        peek = lambda o: 16 * bm.match(tracegen.assemble_prompt(trace, r, o))
        O, c = order_exhaustive(list(D), peek)
        assert c == max(peek([D[i] for i in p]) for p in itertools.permutations(range(len(D))))
        assert c >= peek(tree.order(D)[0])
        req, _, _ = bm.lookup(tracegen.assemble_prompt(trace, r, O))
        tree.observe(O)
        bm.release(req)


# ---- library == oracle, bit-exact -------------------------------------------------------------------------
@pytest.mark.parametrize("arm", ["sorted", "recency", "exhaustive"])
@pytest.mark.parametrize("cfg_id,requests", [(1, None), (2, range(24))])
def test_arm_traces_library_equals_oracle(arm, cfg_id, requests):
    cfg = tracegen.CONFIGS[cfg_id]
    trace = tracegen.make_trace(cfg)
    ref = run_trace(trace, arm, compute=False, requests=requests)
    recs = TraceRunner(trace, arm, ctx=make_context(cfg)).run(compute=False, requests=requests)     # per-request calls
    waves = admit_waves(make_context(cfg), trace, arm, requests=requests, force_waves=False)        # cw_admit_batch
    recs2 = [rec for w in waves for rec in w.recs]
    assert len(recs) == len(recs2) == len(ref.requests)
    for a, a2, o in zip(recs, recs2, ref.requests):
        for x in (a, a2):
            assert (x.r, x.order, x.depth, x.n_cached, x.table.tolist()) == (o.r, o.order, o.depth, o.n_cached, list(o.table))


def test_arm_ranking_on_config2():
    """hit blocks over the first 32 requests of config 2: exhaustive >= greedy > sorted, recency, retrieval."""
    trace = tracegen.make_trace(tracegen.CONFIGS[2])
    hit = {}
    for arm in ARMS:
        waves = admit_waves(make_context(trace.cfg), trace, arm, requests=range(32))
        hit[arm] = sum(int(w.nc.sum()) for w in waves) // 16
    assert hit["exhaustive"] >= hit["greedy"] > max(hit["sorted"], hit["recency"], hit["retrieval"])


def test_order_arm_invalid_arguments():
    ctx = Context(16, 2, 1, 64, 4)
    with pytest.raises(CwError):
        ctx.cw_order_arm(9, [1, 2])                                  # unknown arm
    with pytest.raises(CwError):
        ctx.cw_order_arm("sorted", [1, 1])                           # duplicate ids
    with pytest.raises(CwError):
        ctx.cw_order_arm("exhaustive", [0, 1])                       # exhaustive needs the tokens
    docs = np.zeros((4, 16), dtype=np.int32)
    with pytest.raises(CwError):
        ctx.cw_order_arm("exhaustive", list(range(9)), docs, np.zeros(4, np.int32))   # k > 8
    assert ctx.cw_order_arm("sorted", [3, 1, 2]) == ([1, 2, 3], 0)
    assert ctx.cw_order_arm("retrieval", []) == ([], 0)
