"""Pins for the NEXT-4 part of the oracle (oracle/blocks.py: BlockManager.extend; oracle/attention.py with an arbitrary
number of tokens already in the pool) — SURVEY.md 8(f) NEXT-4, PAPER.md:253-283 (continuous batching: chunked prefill and
decode rows share a launch with prefill suffixes).  Hand-worked block tables, the plain-definition invariants, and
'growing a request token by token == admitting the long sequence at once'."""
import numpy as np
import pytest

from oracle import attention as oattn
from oracle.blocks import BlockManager, NoSpace


def test_extend_hand_worked():
    """NB = 8.  A 20-token prompt takes blocks 0,1 (block 0 full and registered, block 1 partial).  +11 tokens -> 31: still
    2 blocks, nothing new registered.  +1 -> 32: block 1 is complete and registered.  +1 -> 33: block 2 is popped from
    the head of the free list.  A second request with the same 32 leading tokens then hits blocks 0 and 1."""
    rng = np.random.default_rng(3)
    t = rng.integers(0, 32000, 64, dtype=np.int32)
    bm = BlockManager(8)
    req, table, c = bm.lookup(t[:20])
    assert (table, c) == ([0, 1], 0) and len(bm.index) == 1
    assert bm.extend(req, t[20:31]) == [0, 1] and len(bm.index) == 1
    assert bm.extend(req, t[31:32]) == [0, 1] and len(bm.index) == 2
    assert bm.extend(req, t[32:33]) == [0, 1, 2] and len(bm.index) == 2
    assert bm.free_list() == [3, 4, 5, 6, 7]
    bm.check_invariants()
    req2, table2, c2 = bm.lookup(np.concatenate([t[:32], rng.integers(0, 32000, 5, dtype=np.int32)]))
    assert (table2, c2) == ([0, 1, 3], 32)
    bm.release(req)
    bm.release(req2)
    assert bm.free_list() == [4, 5, 6, 7, 2, 3, 1, 0]            # reverse block order per request, shared blocks last
    bm.check_invariants()


def test_extend_no_space_leaves_state_untouched():
    rng = np.random.default_rng(4)
    bm = BlockManager(3)
    req, table, _ = bm.lookup(rng.integers(0, 32000, 40, dtype=np.int32))
    before = (list(bm.free_list()), dict(bm.index), list(bm.ref))
    with pytest.raises(NoSpace):
        bm.extend(req, rng.integers(0, 32000, 20, dtype=np.int32))     # 60 tokens need 4 blocks
    assert (list(bm.free_list()), dict(bm.index), list(bm.ref)) == before
    assert bm.extend(req, rng.integers(0, 32000, 8, dtype=np.int32)) == table
    bm.check_invariants()


@pytest.mark.parametrize("seed", range(5))
def test_growth_equals_one_shot(seed):
    """lookup(n0 tokens) + extend() in random pieces gives the same block table, the same registered prefixes and the
    same free list as one lookup of the whole sequence on a fresh manager."""
    rng = np.random.default_rng(seed)
    n = int(rng.integers(40, 200))
    t = rng.integers(0, 32000, n, dtype=np.int32)
    a, b = BlockManager(32), BlockManager(32)
    n0 = int(rng.integers(1, n))
    req, _, _ = a.lookup(t[:n0])
    pos = n0
    while pos < n:
        step = int(rng.integers(1, 24))
        table = a.extend(req, t[pos:pos + step])
        pos = min(n, pos + step)
        a.check_invariants()
    req_b, table_b, _ = b.lookup(t)
    assert table == table_b and set(a.index) == set(b.index) and a.free_list() == b.free_list()
    a.release(req)
    b.release(req_b)
    assert a.free_list() == b.free_list()


def test_decode_rows_equal_full_recompute():
    """attention of ONE new row over n tokens already in the paged pool (any n, not a multiple of 16) equals row n of the
    full recompute; a chunked prefill (chunks of 37 tokens) equals the one-shot prefill (fp64, up to BLAS summation order)."""
    rng = np.random.default_rng(9)
    Hq, Hkv, D, n = 4, 2, 64, 150
    q, k, v = rng.standard_normal((n, Hq, D)), rng.standard_normal((n, Hkv, D)), rng.standard_normal((n, Hkv, D))
    full = oattn.attention_full(q, k, v, 1e4)
    table = list(rng.permutation(12)[:10])
    pool = oattn.PagedPool(12, Hkv, D)
    outs, pos = [], 0
    for step in [37, 37, 37, 37, 1, 1]:
        outs.append(oattn.attention_suffix(pool, table, pos, q[pos:pos + step], k[pos:pos + step], v[pos:pos + step], 1e4))
        pos += step
    assert pos == n and np.abs(np.concatenate(outs) - full).max() <= 1e-12
