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
