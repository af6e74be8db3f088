"""CPU tests of the C-ABI library's host logic (no GPU, no compute kernels):
  * the library loads and exports every symbol include/cacheweaver.h declares
  * cw_order / cw_observe / cw_lookup / cw_release reproduce the paper's worked examples (tests/golden/)
  * bit-exact agreement with the oracle on random op sequences and on the BASELINE.json traces
    (orders, predicted depths, hash chains, block tables, n_cached, free lists, evictions).
The oracle and the library share no code; only tracegen (seeded inputs) is common.
"""
import os
import random
import re

import numpy as np
import pytest

import tracegen
from conftest import ROOT, golden
from oracle.blocks import BlockManager, NoSpace as OracleNoSpace, chain_hashes
from oracle.ordering import KnowledgeTree
from oracle.pipeline import run_trace
from paper_2606_19667_b200 import EXPORTS, Context, CwError, NoSpace, load_library
from paper_2606_19667_b200.engine import TraceRunner, make_context


def host_ctx(NB=16, H=8, eager=True, salt=0):
    return Context(NB, 2, 1, 64, H, eager_register=eager, hash_salt=salt)


def test_library_exports_every_declared_symbol():
    lib = load_library()
    hdr = open(os.path.join(ROOT, "include", "cacheweaver.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = sorted(set(re.findall(r"\b(cw_[a-z_0-9]+)\s*\(", hdr)))
    assert declared, "no declarations parsed"
    for name in declared:
        assert hasattr(lib, name), f"{name} declared in cacheweaver.h but not exported"
    assert sorted(EXPORTS) == declared


def test_figure2_worked_example():
    g = golden("figure2_ordering.txt")
    ids = {n: i + 100 for i, n in enumerate("ABCDEFG")}
    c = host_ctx()
    c.cw_observe([ids[x] for x in g["cached_path"].split()])
    O, depth = c.cw_order([ids[x] for x in g["candidates"].split()])
    assert O == [ids[x] for x in g["expected_order"].split()]
    assert depth == int(g["expected_prefix_docs"])


def test_figure1_alignment():
    g = golden("figure1_alignment.txt")
    names = sorted(set(g["request1_order"].split() + g["request2_retrieval"].split()))
    ids = {n: i for i, n in enumerate(names)}
    c = host_ctx()
    r1 = [ids[x] for x in g["request1_order"].split()]
    r2 = [ids[x] for x in g["request2_retrieval"].split()]
    assert c.cw_order(r1) == (r1, 0)                       # empty trie -> retrieval order
    c.cw_observe(r1)
    assert c.cw_predict(r2) == int(g["retrieval_order_prefix_docs"])
    O, depth = c.cw_order(r2)
    assert depth == int(g["reordered_prefix_docs"]) and O[:4] == r1[:4] and sorted(O) == sorted(r2)


def test_recency_window_hand_worked():
    c = host_ctx(H=2)
    c.cw_observe([1, 2]); c.cw_observe([3]); c.cw_observe([4])
    assert c.cw_order([2, 1]) == ([2, 1], 0)


def test_invalid_arguments():
    c = host_ctx()
    with pytest.raises(CwError):
        c.cw_order([1, 1, 2])
    assert c.cw_order([]) == ([], 0)
    with pytest.raises(CwError):
        c.cw_lookup(np.zeros(0, dtype=np.int32))
    with pytest.raises(CwError):
        c.cw_release(12345)
    with pytest.raises(CwError):
        Context(16, 3, 2, 64, 4)                           # Hq % Hkv != 0
    with pytest.raises(CwError):
        Context(16, 2, 1, 96, 4)                           # head_dim not in {64, 128}
    with pytest.raises(CwError):                            # device call on a host-only context fails loudly
        c._check(c.lib.cw_append_kv(c.h, None, None, None, None, None, None, None, 1, 1, 1, None))


def test_hash_chain_vectors():
    g = golden("fnv1a64_vectors.txt")
    c = host_ctx()
    t = np.arange(32, dtype=np.int32)
    ch = c.cw_hash_chain(t)
    assert [f"{int(x):016x}" for x in ch] == [g["block0_tokens_0_15_parent_0"], g["block1_tokens_16_31_parent_h0"]]
    assert f"{int(c.cw_hash_chain(t[16:])[0]):016x}" == g["block1_tokens_16_31_parent_0"]
    assert f"{int(c.cw_hash_chain(np.zeros(16, dtype=np.int32))[0]):016x}" == g["sixteen_zeros_parent_0"]
    c2 = host_ctx(salt=77)
    rng = np.random.default_rng(3)
    toks = rng.integers(-5, 32000, 100, dtype=np.int32)
    assert [int(x) for x in c2.cw_hash_chain(toks)] == chain_hashes(toks, 77)


def _scenario():
    rng = np.random.default_rng(0)
    docs = {n: rng.integers(0, 32000, 32, dtype=np.int32) for n in "ABCDEFG"}
    return docs, rng


def test_block_table_scenario():
    g = golden("block_table_scenario.txt")
    docs, rng = _scenario()
    ids = {n: i for i, n in enumerate("ABCDEFG")}
    names = {i: n for n, i in ids.items()}
    c = host_ctx(NB=16, H=8)
    prompt = lambda O: np.concatenate([docs[names[d]] for d in O] + [rng.integers(0, 32000, 20, dtype=np.int32)])
    for name in ["req1", "req2", "req3", "req4"]:
        retr, order, depth, m, table, free, evict = [x.split() for x in g[name].split("|")]
        O, d = c.cw_order([ids[x] for x in retr])
        assert ([names[x] for x in O], d) == (order, int(depth[0])), name
        c.cw_observe(O)
        req, tab, nc = c.cw_lookup(prompt(O))
        assert nc == 16 * int(m[0]) and tab.tolist() == [int(x) for x in table], name
        c.cw_release(req)
        assert c.cw_free_list() == [int(x) for x in free], name
        assert c.cw_stats()["evictions"] == int(evict[0]), name
    for name in ["req5a", "req5b"]:
        retr, order, depth, m = [x.split() for x in g[name].split("|")]
        O, d = c.cw_order([ids[x] for x in retr])
        assert ([names[x] for x in O], d) == (order, int(depth[0])), name
        assert c.cw_lookup(prompt(O), peek_only=True) == 16 * int(m[0]), name


def test_no_space_leaves_state_untouched():
    c = host_ctx(NB=4)
    r, tab, nc = c.cw_lookup(np.arange(40, dtype=np.int32))
    before = (c.cw_free_list(), c.cw_stats())
    with pytest.raises(NoSpace):
        c.cw_lookup(np.arange(100, 140, dtype=np.int32))
    assert before == (c.cw_free_list(), c.cw_stats())
    c.cw_release(r)
    assert len(c.cw_free_list()) == 4


@pytest.mark.parametrize("seed", range(12))
def test_random_ops_library_equals_oracle(seed):
    """model-based: the same random op sequence drives the library and the oracle; everything must be bit-equal."""
    rng = random.Random(seed)
    nrng = np.random.default_rng(seed)
    n_docs, H, NB = 7, rng.randint(1, 6), rng.choice([12, 24, 40])
    docs = [nrng.integers(0, 50, 16 * rng.randint(1, 3), dtype=np.int32) for _ in range(n_docs)]
    eager = bool(seed % 2)
    lib = host_ctx(NB=NB, H=H, eager=eager)
    tree, bm = KnowledgeTree(H), BlockManager(NB, eager_register=eager)
    live = []
    for step in range(200):
        if live and (rng.random() < 0.45 or len(live) > 3):
            a, b = live.pop(rng.randrange(len(live)))
            lib.cw_release(a); bm.release(b)
        else:
            D = rng.sample(range(n_docs), rng.randint(1, 4))
            assert lib.cw_order(D) == tuple(tree.order(D))
            assert lib.cw_stats()["order_probes"] == tree.probes
            O = tree.order(D)[0] if rng.random() < 0.7 else D
            assert lib.cw_predict(O) == tree.ell(O)
            toks = np.concatenate([docs[d] for d in O] + [nrng.integers(0, 50, rng.randint(0, 20), dtype=np.int32)])
            assert lib.cw_lookup(toks, peek_only=True) == 16 * bm.match(toks)
            try:
                exp = bm.lookup(toks)
            except OracleNoSpace:
                with pytest.raises(NoSpace):
                    lib.cw_lookup(toks)
            else:
                req, tab, nc = lib.cw_lookup(toks)
                assert (tab.tolist(), nc) == (exp[1], exp[2])
                live.append((req, exp[0]))
                lib.cw_observe(O); tree.observe(O)
        st = lib.cw_stats()
        assert lib.cw_free_list() == bm.free_list()
        assert (st["evictions"], st["hit_blocks"], st["miss_blocks"]) == (bm.evictions, bm.hit_blocks, bm.miss_blocks)
        assert st["seq"] == tree.seq


def _compare_host_trace(cfg, strategy, requests=None):
    trace = tracegen.make_trace(cfg)
    ref = run_trace(trace, strategy, compute=False, requests=requests)
    runner = TraceRunner(trace, strategy, ctx=make_context(cfg))
    recs = runner.run(compute=False, requests=requests)
    assert len(recs) == len(ref.requests)
    for a, b in zip(recs, ref.requests):
        assert (a.r, a.order, a.depth, a.n_cached, a.wave) == (b.r, b.order, b.depth, b.n_cached, b.wave)
        assert a.table.tolist() == b.table
        assert np.array_equal(a.tokens, b.tokens)
    st = runner.ctx.cw_stats()
    assert st["evictions"] == ref.evictions
    assert len(runner.waves) == ref.waves
    # work counters of cw_stats against the plain definitions over the oracle's records
    n = cfg.n
    assert st["prompt_tokens"] == n * len(ref.requests)
    assert st["suffix_tokens"] == sum(n - b.n_cached for b in ref.requests)
    assert st["attn_flops"] == sum(4 * cfg.Hq * cfg.D * sum(p + 1 for p in range(b.n_cached, n)) for b in ref.requests)
    assert st["append_bytes"] == st["suffix_tokens"] * (2 * cfg.Hq * cfg.D * 2 + 2 * 2 * cfg.Hkv * cfg.D * 2 + 4)
    return recs


@pytest.mark.parametrize("strategy", ["greedy", "retrieval"])
def test_trace_cfg1_and_cfg2_host_path_bit_exact(strategy):
    _compare_host_trace(tracegen.CONFIGS[1], strategy)
    recs = _compare_host_trace(tracegen.CONFIGS[2], strategy)
    if strategy == "greedy":
        assert sum(r.n_cached for r in recs) > 0


def test_trace_cfg3_cell_host_path_bit_exact():
    for k, ov in [(3, 30), (10, 90)]:
        _compare_host_trace(tracegen.config3(k, ov, n_req=48), "greedy")


def test_trace_cfg4_cfg5_waves_host_path_bit_exact():
    """concurrent configs: wave boundaries (CW_ERR_NO_SPACE), eviction between waves, trie over-prediction."""
    _compare_host_trace(tracegen.CONFIGS[4], "greedy")
    recs = _compare_host_trace(tracegen.CONFIGS[5], "greedy")
    assert max(r.wave for r in recs) >= 1
    _compare_host_trace(tracegen.CONFIGS[5], "retrieval")


def test_greedy_hits_at_least_retrieval_on_cfg2():
    """the trend the paper claims: greedy order reuses more cached blocks."""
    cfg = tracegen.CONFIGS[2]
    hit = {}
    for s in ("greedy", "retrieval"):
        runner = TraceRunner(tracegen.make_trace(cfg), s, ctx=make_context(cfg))
        hit[s] = sum(r.n_cached for r in runner.run(compute=False))
    assert hit["greedy"] > hit["retrieval"]


@pytest.mark.parametrize("cfg_id,strategy", [(1, "greedy"), (2, "retrieval"), (4, "greedy"), (5, "greedy"), (5, "retrieval")])
def test_admit_batch_equals_per_request_calls_and_oracle(cfg_id, strategy):
    """cw_admit_batch (one C call per wave) == cw_order/cw_lookup/cw_observe per request == the oracle."""
    from paper_2606_19667_b200.engine import admit_waves
    cfg = tracegen.CONFIGS[cfg_id]
    trace = tracegen.make_trace(cfg)
    ref = run_trace(trace, strategy, compute=False)
    ctx = make_context(cfg)
    for _ in range(2):                                   # second pass after cw_reset must reproduce the first
        waves = admit_waves(ctx, trace, strategy, force_waves=False)
        recs = [rec for w in waves for rec in w.recs]
        assert len(waves) == ref.waves and len(recs) == len(ref.requests)
        for a, b in zip(recs, ref.requests):
            assert (a.r, a.order, a.depth, a.n_cached, a.wave) == (b.r, b.order, b.depth, b.n_cached, b.wave)
            assert a.table.tolist() == b.table
        for w in waves:
            assert w.cu[-1] == sum(cfg.n - c for c in w.nc) and w.cu[0] == 0
        assert ctx.cw_stats()["evictions"] == ref.evictions
        ctx.cw_reset()
        st = ctx.cw_stats()
        assert (st["requests"], st["trie_nodes"], st["free_blocks"], st["seq"]) == (0, 0, cfg.NB, 0)
        assert ctx.cw_free_list() == list(range(cfg.NB))


def test_admit_batch_invalid_arguments():
    ctx = host_ctx(NB=64)
    docs = np.zeros((4, 32), dtype=np.int32)
    q = np.zeros((1, 8), dtype=np.int32)
    with pytest.raises(CwError):
        ctx.cw_admit_batch(np.array([[0, 9]]), True, docs, q)          # doc id out of range
    with pytest.raises(CwError):
        ctx.cw_admit_batch(np.array([[1, 1]]), True, docs, q)          # duplicate ids
    with pytest.raises(CwError):
        ctx.cw_admit_batch(np.array([[0, 1]]), True, docs, q, max_blocks=2)   # table too narrow
    a = ctx.cw_admit_batch(np.array([[0, 1]]), True, docs, q)
    assert a["admitted"] == 1 and a["cu"].tolist() == [0, 72]
    with pytest.raises(CwError):
        ctx.cw_release_batch([a["reqs"][0], 12345])


def test_admit_batch_invalid_row_leaves_state_untouched():
    """An invalid row anywhere in the batch (here the LAST one: doc id out of range, then a duplicate) is reported before
    any request is admitted: no block is pinned or registered and the knowledge tree is unchanged."""
    from paper_2606_19667_b200 import Context, CwError
    ctx = Context(64, 2, 1, 64, 4)
    rng = np.random.default_rng(0)
    doc_tokens = rng.integers(0, 32000, size=(10, 32), dtype=np.int32)
    queries = rng.integers(0, 32000, size=(3, 20), dtype=np.int32)
    before = (ctx.cw_stats(), ctx.cw_free_list())
    for bad_row in ([0, 1, 10], [4, 4, 5]):
        ids = np.array([[0, 1, 2], [3, 1, 0], bad_row], dtype=np.int64)
        with pytest.raises(CwError):
            ctx.cw_admit_batch(ids, "greedy", doc_tokens, queries)
        assert (ctx.cw_stats(), ctx.cw_free_list()) == before
    with pytest.raises(CwError):                                   # unknown arm id
        ctx.cw_admit_batch(np.array([[0, 1, 2]], dtype=np.int64), 9, doc_tokens, queries[:1])
    assert (ctx.cw_stats(), ctx.cw_free_list()) == before
    a = ctx.cw_admit_batch(np.array([[0, 1, 2], [3, 1, 0]], dtype=np.int64), "greedy", doc_tokens, queries[:2])
    assert a["admitted"] == 2


@pytest.mark.parametrize("seed", range(4))
def test_extend_matches_oracle_under_random_growth(seed):
    """cw_extend vs oracle BlockManager.extend: several live requests grow in random pieces (with shared prefixes and a pool
    small enough for NO_SPACE), block tables / free lists / hit counts bit-exact, NO_SPACE leaves both sides unchanged."""
    rng = np.random.default_rng(200 + seed)
    NB = 40
    ctx = Context(NB, 2, 1, 64, 4)
    obm = BlockManager(NB)
    base = rng.integers(0, 32000, 96, dtype=np.int32)
    live = []
    for step in range(120):
        op = rng.integers(0, 10)
        if op < 3 and len(live) < 5:
            t = np.concatenate([base[: int(rng.integers(0, 97))], rng.integers(0, 32000, int(rng.integers(1, 40)), dtype=np.int32)])
            try:
                oreq, otable, oc = obm.lookup(t)
            except OracleNoSpace:
                with pytest.raises(NoSpace):
                    ctx.cw_lookup(t)
                continue
            req, table, c = ctx.cw_lookup(t)
            assert (table.tolist(), c) == (otable, oc)
            live.append((req, oreq))
        elif op < 8 and live:
            req, oreq = live[int(rng.integers(0, len(live)))]
            t = rng.integers(0, 32000, int(rng.integers(1, 30)), dtype=np.int32)
            try:
                otable = obm.extend(oreq, t)
            except OracleNoSpace:
                with pytest.raises(NoSpace):
                    ctx.cw_extend(req, t)
                assert ctx.cw_free_list() == obm.free_list()
                continue
            assert ctx.cw_extend(req, t).tolist() == otable
        elif live:
            req, oreq = live.pop(int(rng.integers(0, len(live))))
            ctx.cw_release(req)
            obm.release(oreq)
        assert ctx.cw_free_list() == obm.free_list()
        obm.check_invariants()
    st = ctx.cw_stats()
    assert (st["hit_blocks"], st["miss_blocks"], st["evictions"]) == (obm.hit_blocks, obm.miss_blocks, obm.evictions)


@pytest.mark.parametrize("bits,eager", [(1, True), (3, True), (3, False), (6, True)])
def test_index_key_collisions_never_serve_foreign_blocks(bits, eager):
    """The prefix index keyed by only `bits` bits of the chain hash collides constantly.  Property (cacheweaver.h,
    index_key_bits): a block returned as a hit for position i holds exactly this prompt's tokens [0, 16(i+1)) — checked
    against a test-side record of what every block was allocated for — and the library never reports more cached blocks
    than the oracle, which matches by token-prefix identity; with the full 64-bit key it reports the same."""
    rng = random.Random(bits * 2 + eager)
    nrng = np.random.default_rng(bits)
    NB = 48
    lib = Context(NB, 2, 1, 64, 4, eager_register=eager, index_key_bits=bits)
    full = Context(NB, 2, 1, 64, 4, eager_register=eager)
    docs = [nrng.integers(0, 30, 16 * rng.randint(1, 3), dtype=np.int32) for _ in range(9)]
    content = {}                      # block id -> bytes of the token prefix it was allocated for
    live, fewer = [], 0
    for step in range(400):
        if live and (rng.random() < 0.5 or len(live) > 2):
            for h, x in zip((lib, full), live.pop(rng.randrange(len(live)))[:2]):
                h.cw_release(x)
            continue
        O = rng.sample(range(len(docs)), rng.randint(1, 3))
        toks = np.concatenate([docs[d] for d in O] + [nrng.integers(0, 30, rng.randint(1, 20), dtype=np.int32)])
        raw = toks.astype("<i4").tobytes()
        try:
            req, tab, nc = lib.cw_lookup(toks)
        except NoSpace:
            continue
        rf, tf, ncf = full.cw_lookup(toks)
        live.append((req, rf))
        for i, b in enumerate(tab.tolist()):
            pre = raw[: 64 * (i + 1)]
            if i < nc // 16:
                assert content.get(b) == pre, f"step {step}: hit block {b} at position {i} holds another prefix"
            else:
                content[b] = pre if 16 * (i + 1) <= len(toks) else None      # partial last block: never matched
        assert nc <= ncf
        fewer += nc < ncf
    assert fewer > 0, "the truncated key never collided: the test exercises nothing"
