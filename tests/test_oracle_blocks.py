"""Pins for oracle/blocks.py (no GPU)."""
import random

import numpy as np
import pytest

from conftest import golden
from oracle.blocks import BlockManager, NoSpace, chain_hashes, fnv1a64
from oracle.ordering import KnowledgeTree


def test_fnv1a64_published_vectors():
    g = golden("fnv1a64_vectors.txt")
    assert f"{fnv1a64(b''):016x}" == g["empty"]
    assert f"{fnv1a64(b'a'):016x}" == g["a"]
    assert f"{fnv1a64(b'foobar'):016x}" == g["foobar"]


def test_chain_hand_worked_and_prefix_sensitivity():
    g = golden("fnv1a64_vectors.txt")
    ch = chain_hashes(np.arange(32), salt=0)
    assert f"{ch[0]:016x}" == g["block0_tokens_0_15_parent_0"]
    assert f"{ch[1]:016x}" == g["block1_tokens_16_31_parent_h0"]
    alone = chain_hashes(np.arange(16, 32), salt=0)[0]
    assert f"{alone:016x}" == g["block1_tokens_16_31_parent_0"]
    assert alone != ch[1]                       # PAPER.md:33 prefix sensitivity
    assert f"{chain_hashes(np.zeros(16, dtype=np.int32))[0]:016x}" == g["sixteen_zeros_parent_0"]
    assert len(chain_hashes(np.arange(47))) == 2     # partial last block is never hashed


def test_chain_matches_independent_struct_pack():
    import struct
    toks = [7, 70000, 2**31 - 1] + list(range(13)) + list(range(100, 116))
    h = 0x1234
    exp = []
    for i in range(2):
        msg = struct.pack("<Q", h) + struct.pack("<16i", *toks[16 * i:16 * i + 16])
        x = 0xCBF29CE484222325
        for b in msg:
            x = ((x ^ b) * 0x100000001B3) % (1 << 64)
        h = x
        exp.append(h)
    assert chain_hashes(toks, salt=0x1234) == exp


def _scenario_setup():
    rng = np.random.default_rng(123)
    docs = {c: rng.integers(0, 32000, 32, dtype=np.int32) for c in "ABCDEFG"}
    return docs, rng


def _prompt(docs, order, q):
    return np.concatenate([docs[d] for d in order] + [q])


def test_hand_worked_block_table_scenario():
    g = golden("block_table_scenario.txt")
    docs, rng = _scenario_setup()
    T, bm = KnowledgeTree(8), BlockManager(16, eager_register=True)
    for name in ["req1", "req2", "req3", "req4"]:
        retr, order, depth, m, table, free, evict = [x.split() for x in g[name].split("|")]
        O, d = T.order(retr)
        assert (O, d) == (order, int(depth[0])), name
        T.observe(O)
        req, tab, c = bm.lookup(_prompt(docs, O, rng.integers(0, 32000, 20, dtype=np.int32)))
        assert c == 16 * int(m[0]), name
        assert tab == [int(x) for x in table], name
        bm.release(req)
        assert bm.free_list() == [int(x) for x in free], name
        assert bm.evictions == int(evict[0]), name
        bm.check_invariants()
    for name in ["req5a", "req5b"]:
        retr, order, depth, m = [x.split() for x in g[name].split("|")]
        O, d = T.order(retr)
        assert (O, d) == (order, int(depth[0])), name
        assert bm.match(_prompt(docs, O, rng.integers(0, 32000, 20, dtype=np.int32))) == int(m[0]), name
    assert T.brute_force_permutations(["C", "B", "A"])[1] == int(g["req5b_brute_force_depth"])


def test_figure1_retrieval_order_gets_zero_blocks():
    g = golden("block_table_scenario.txt")
    docs, rng = _scenario_setup()
    bm = BlockManager(16)
    req, _, _ = bm.lookup(_prompt(docs, "ABC", rng.integers(0, 32000, 20, dtype=np.int32)))
    bm.release(req)
    assert bm.match(_prompt(docs, "CAD", rng.integers(0, 32000, 20, dtype=np.int32))) == int(g["req2_retrieval_m"])
    assert bm.match(_prompt(docs, "ACD", rng.integers(0, 32000, 20, dtype=np.int32))) == 2


def test_fully_cached_prompt_keeps_one_suffix_block():
    # reading: cap m at floor((n-1)/16) so at least one query row remains
    bm = BlockManager(8)
    t = np.arange(32, dtype=np.int32)
    r, tab, c = bm.lookup(t); bm.release(r)
    r2, tab2, c2 = bm.lookup(t)
    assert c == 0 and c2 == 16 and tab2[0] == tab[0] and tab2[1] != tab[1]
    bm.release(r2); bm.check_invariants()


def test_no_space_leaves_state_untouched():
    bm = BlockManager(4)
    r, tab, c = bm.lookup(np.arange(40, dtype=np.int32))          # 3 blocks pinned
    snapshot = (list(bm.ref), bm.free_list(), dict(bm.index), bm.evictions)
    with pytest.raises(NoSpace):
        bm.lookup(np.arange(100, 140, dtype=np.int32))            # needs 3, only 1 free
    assert snapshot == (list(bm.ref), bm.free_list(), dict(bm.index), bm.evictions)
    bm.release(r); bm.check_invariants()


def _brute_match(registered_prefixes, tokens):
    """plain definition: leading full blocks whose entire token prefix equals a resident registered one."""
    n = len(tokens); m = 0
    while m < (n - 1) // 16 and tuple(tokens[: 16 * (m + 1)]) in registered_prefixes:
        m += 1
    return m


@pytest.mark.parametrize("seed", range(10))
def test_random_ops_invariants_and_plain_definition(seed):
    rng = random.Random(seed)
    nrng = np.random.default_rng(seed)
    docs = [nrng.integers(0, 50, 16 * rng.randint(1, 3), dtype=np.int32) for _ in range(6)]
    bm = BlockManager(24, eager_register=bool(seed % 2))
    live = []
    for step in range(120):
        if live and (rng.random() < 0.45 or len(live) > 3):
            bm.release(live.pop(rng.randrange(len(live))))
        else:
            order = rng.sample(range(6), rng.randint(1, 3))
            toks = np.concatenate([docs[d] for d in order] + [nrng.integers(0, 50, rng.randint(0, 20), dtype=np.int32)])
            registered = {tuple(np.frombuffer(k, dtype="<i4")) for k in bm.index}
            expect_m = _brute_match(registered, list(toks))
            try:
                req, tab, c = bm.lookup(toks)
                assert c == 16 * expect_m
                assert len(tab) == -(-len(toks) // 16)
                live.append(req)
            except NoSpace:
                pass
        bm.check_invariants()
