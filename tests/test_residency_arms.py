"""NEXT-1 in the library (cw_mark_stale, cw_feedback, CW_ARM_GREEDY_FEEDBACK / CW_ARM_GREEDY_RESIDENT) against the oracle,
bit-exact on orders / predicted depths / block tables / cached tokens; host-only contexts (no GPU needed).
PAPER.md:129-141, :314; the oracle side is pinned in tests/test_oracle_residency.py."""
import dataclasses

import numpy as np
import pytest

import tracegen
from conftest import golden
from oracle.pipeline import run_trace
from paper_2606_19667_b200 import Context
from paper_2606_19667_b200.engine import TraceRunner, admit_waves, make_context


def evicting_config(seed, **kw):
    base = tracegen.CONFIGS[1]
    d = dict(name=f"evict{seed}", seed=100 + seed, n_docs=8, doc_len=32, n_req=40, k=3, n_shared=2, q_len=20, NB=24, H=12)
    d.update(kw)
    return dataclasses.replace(base, **d)


@pytest.mark.parametrize("strategy", ["greedy_feedback", "greedy_resident"])
@pytest.mark.parametrize("seed", range(3))
def test_request_by_request_path_matches_oracle(strategy, seed):
    trace = tracegen.make_trace(evicting_config(seed))
    ref = run_trace(trace, strategy, compute=False)
    recs = TraceRunner(trace, strategy, device=None).run(compute=False)
    assert len(recs) == len(ref.requests)
    for a, o in zip(recs, ref.requests):
        assert (a.order, a.depth, a.n_cached, a.table.tolist()) == (o.order, o.depth, o.n_cached, list(o.table)), a.r


@pytest.mark.parametrize("strategy", ["greedy_feedback", "greedy_resident"])
def test_wave_admission_matches_oracle_and_counts_over_prediction(strategy):
    """cw_admit_batch with the NEXT-1 arms on a wave-admitted trace whose pool is too small (eviction between waves)."""
    cfg = evicting_config(7, n_req=60, NB=40, admission="waves")
    trace = tracegen.make_trace(cfg)
    ref = run_trace(trace, strategy, compute=False)
    ctx = make_context(cfg, None)
    waves = admit_waves(ctx, trace, strategy)
    recs = [rec for w in waves for rec in w.recs]
    for a, o in zip(recs, ref.requests):
        assert (a.order, a.depth, a.n_cached, a.table.tolist(), a.wave) == (o.order, o.depth, o.n_cached, list(o.table), o.wave), a.r
    st = ctx.cw_stats()
    pred = sum(o.depth for o in ref.requests)
    actual = sum(o.n_cached // cfg.doc_len for o in ref.requests)
    over = sum(max(0, o.depth - o.n_cached // cfg.doc_len) for o in ref.requests)
    assert (st["predicted_prefix_docs"], st["actual_prefix_docs"], st["over_predicted_docs"]) == (pred, actual, over)
    if strategy == "greedy_resident":
        assert over == 0
    plain = run_trace(trace, "greedy", compute=False)
    assert sum(max(0, o.depth - o.n_cached // cfg.doc_len) for o in plain.requests) > over


def test_block_table_scenario_rows_through_the_c_abi():
    """golden rows req5a_resident / req5a_after_feedback of the SURVEY.md 8(c7) scenario, through cw_order_arm / cw_feedback."""
    g = golden("block_table_scenario.txt")
    rng = np.random.default_rng(123)
    names = "ABCDEFG"
    doc_tokens = np.stack([rng.integers(0, 32000, 32, dtype=np.int32) for _ in names])
    ids = {c: i for i, c in enumerate(names)}

    def fresh():
        r2 = np.random.default_rng(123)
        [r2.integers(0, 32000, 32, dtype=np.int32) for _ in names]
        ctx = Context(16, 2, 1, 64, 8)
        for name in ["req1", "req2", "req3", "req4"]:
            retr = [ids[c] for c in g[name].split("|")[0].split()]
            O, _ = ctx.cw_order(retr)
            q = r2.integers(0, 32000, 20, dtype=np.int32)
            req, _, _ = ctx.cw_lookup(np.concatenate([doc_tokens[d] for d in O] + [q]))
            ctx.cw_observe(O)
            ctx.cw_release(req)
        return ctx, r2

    ctx, r2 = fresh()
    retr, order, depth, m = [x.split() for x in g["req5a_resident"].split("|")]
    O, d = ctx.cw_order_arm("greedy_resident", [ids[c] for c in retr], doc_tokens)
    assert ([names[i] for i in O], d) == (order, int(depth[0]))
    q = r2.integers(0, 32000, 20, dtype=np.int32)
    assert ctx.cw_lookup(np.concatenate([doc_tokens[i] for i in O] + [q]), peek_only=True) == 16 * int(m[0])
    assert ctx.cw_stats()["stale_marks"] == 1

    ctx, r2 = fresh()
    O, pred = ctx.cw_order([ids[c] for c in "BCA"])
    assert ([names[i] for i in O], pred) == (list("ABC"), 3)
    c = ctx.cw_lookup(np.concatenate([doc_tokens[i] for i in O] + [r2.integers(0, 32000, 20, dtype=np.int32)]), peek_only=True)
    ctx.cw_feedback(O, pred, c // 32)
    retr, order, depth = [x.split() for x in g["req5a_after_feedback"].split("|")]
    O, d = ctx.cw_order([ids[c] for c in retr])
    assert ([names[i] for i in O], d) == (order, int(depth[0]))


def test_matched_docs_through_the_c_abi():
    """cw_matched_docs on the hand-worked ragged prompt and the no-query prompt of tests/test_oracle_residency.py (expected
    values typed here, not taken from the oracle), then against the oracle on random segment ends."""
    from oracle.blocks import matched_docs
    ctx = Context(16, 2, 1, 64, 8)
    ends, n = [238, 436, 650], 700
    assert [ctx.cw_matched_docs(ends, c, n) for c in (0, 208, 224, 416, 432, 624, 640, 688)] == [0, 0, 1, 1, 2, 2, 3, 3]
    assert ctx.cw_matched_docs([32, 64, 96], 80, 96) == 3 and ctx.cw_matched_docs([32, 64, 96], 80, 97) == 2
    rng = np.random.default_rng(3)
    for _ in range(300):
        k = int(rng.integers(0, 7))
        ends = np.cumsum(rng.integers(1, 70, size=k)).tolist()
        n = (ends[-1] if k else 1) + int(rng.integers(0, 40))
        c = 16 * int(rng.integers(0, (n - 1) // 16 + 1))
        assert ctx.cw_matched_docs(ends, c, n) == matched_docs(ends, c, n), (ends, c, n)
    for bad in ([0, 5], [9, 4], [5, 800]):
        with pytest.raises(Exception):
            ctx.cw_matched_docs(bad, 0, 700)


def test_admit_batch_without_query_counts_the_last_document():
    """3 block-aligned documents and q_len = 0, the same request repeated.  The lookup cap (floor((n-1)/16) blocks)
    keeps the last block out of every match; the matched-document count allows for it, so predicted == actual on every
    repeat and the feedback arm marks nothing stale."""
    ctx = Context(24, 2, 1, 64, 12)
    rng = np.random.default_rng(1)
    doc_tokens = rng.integers(0, 32000, size=(8, 32), dtype=np.int32)
    for rep in range(4):
        res = ctx.cw_admit_batch(np.array([[7, 5, 6]], dtype=np.int64), "greedy_feedback", doc_tokens,
                                 np.zeros((1, 0), dtype=np.int32))
        assert int(res["n_cached"][0]) == (0 if rep == 0 else 80)
        ctx.cw_release_batch(res["reqs"])
    st = ctx.cw_stats()
    assert (st["predicted_prefix_docs"], st["actual_prefix_docs"], st["over_predicted_docs"], st["stale_marks"]) == (9, 9, 0, 0)
