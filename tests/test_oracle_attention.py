"""Pins for oracle/attention.py and oracle/pipeline.py (no GPU)."""
import numpy as np
import pytest
import torch

import tracegen
from oracle import attention as A
from oracle import pipeline as P


def _rand(n, Hq, Hkv, D, seed=0):
    rng = np.random.default_rng(seed)
    return (rng.standard_normal((n, Hq, D)), rng.standard_normal((n, Hkv, D)), rng.standard_normal((n, Hkv, D)))


def test_rope_position_zero_is_identity_and_norm_preserved():
    q, _, _ = _rand(9, 2, 1, 64)
    assert np.array_equal(A.rope(q, np.zeros(9, dtype=int), 1e4), q)
    r = A.rope(q, np.arange(9) * 1000, 5e5)
    np.testing.assert_allclose(np.linalg.norm(r, axis=-1), np.linalg.norm(q, axis=-1), rtol=1e-13)


def test_rope_closed_form_single_pair():
    # D = 2: one pair, angle = p * theta^0 = p  =>  plain 2-D rotation by p radians
    x = np.array([[[1.0, 0.0]], [[0.0, 1.0]]])
    r = A.rope(x, np.array([2, 3]), 12345.0)
    np.testing.assert_allclose(r[0, 0], [np.cos(2.0), np.sin(2.0)], atol=1e-15)
    np.testing.assert_allclose(r[1, 0], [-np.sin(3.0), np.cos(3.0)], atol=1e-15)
    # D = 4: second pair rotates by p * theta^(-2/4) = p / sqrt(theta); pairs are (0,2) and (1,3)  (split-half)
    x4 = np.array([[[0.0, 1.0, 0.0, 0.0]]])
    r4 = A.rope(x4, np.array([5]), 100.0)
    np.testing.assert_allclose(r4[0, 0], [0.0, np.cos(0.5), 0.0, np.sin(0.5)], atol=1e-15)


def test_rope_shift_invariance_of_attention():
    # relative-position property: adding a constant to every position leaves attention unchanged
    q, k, v = _rand(20, 4, 2, 32, seed=3)
    pos = np.arange(20)
    o1 = A.attention_rows(A.rope(q, pos, 1e4), A.rope(k, pos, 1e4), v, pos)
    o2 = A.attention_rows(A.rope(q, pos + 777, 1e4), A.rope(k, pos + 777, 1e4), v, pos)
    np.testing.assert_allclose(o1, o2, atol=1e-12)


def test_probability_rows_sum_to_one_and_causal():
    q, k, v = _rand(33, 4, 2, 16, seed=1)
    pos = np.arange(33)
    o, Pm = A.attention_rows(A.rope(q, pos, 1e4), A.rope(k, pos, 1e4), v, pos, return_probs=True)
    np.testing.assert_allclose(Pm.sum(-1), 1.0, atol=1e-12)
    assert np.all(Pm[:, np.triu_indices(33, 1)[0], np.triu_indices(33, 1)[1]] == 0.0)
    assert np.all(Pm >= 0)


def test_row_zero_constant_v_and_zero_q():
    q, k, v = _rand(17, 4, 2, 16, seed=2)
    o = A.attention_full(q, k, v, 1e4)
    for h in range(4):
        assert np.array_equal(o[0, h], v[0, h // 2])                 # row p=0 => o = v_0 exactly
    vc = np.broadcast_to(np.linspace(-1, 1, 16), v.shape).copy()
    np.testing.assert_allclose(A.attention_full(q, k, vc, 1e4), np.broadcast_to(np.linspace(-1, 1, 16), (17, 4, 16)), atol=1e-13)
    o0 = A.attention_full(np.zeros_like(q), k, v, 1e4)               # Q = 0 => uniform P => running mean of V
    run_mean = np.cumsum(v, axis=0) / np.arange(1, 18)[:, None, None]
    np.testing.assert_allclose(o0, run_mean.repeat(2, axis=1), atol=1e-13)


def test_against_pure_python_loops():
    q, k, v = _rand(7, 2, 1, 8, seed=4)
    o = A.attention_full(q, k, v, 1e4)
    ref = A.attention_rows_loops(q.tolist(), k.tolist(), v.tolist(), 1e4, rows=[0, 3, 6], g=2)
    for (p, h), vec in ref.items():
        np.testing.assert_allclose(o[p, h], vec, atol=1e-13)


def test_against_torch_sdpa_fp64_with_rotate_half():
    # library special case: torch SDPA (causal, repeated KV heads) on independently roped inputs
    n, Hq, Hkv, D, theta = 40, 4, 2, 32, 5e5
    q, k, v = _rand(n, Hq, Hkv, D, seed=5)
    tq, tk, tv = (torch.from_numpy(x) for x in (q, k, v))
    inv = 1.0 / (theta ** (torch.arange(0, D, 2, dtype=torch.float64) / D))
    fr = torch.outer(torch.arange(n, dtype=torch.float64), inv)
    emb = torch.cat([fr, fr], -1)
    cos, sin = emb.cos()[:, None, :], emb.sin()[:, None, :]

    def rot_half(x):
        return torch.cat([-x[..., D // 2:], x[..., : D // 2]], -1)

    rq, rk = tq * cos + rot_half(tq) * sin, tk * cos + rot_half(tk) * sin
    o = torch.nn.functional.scaled_dot_product_attention(
        rq.permute(1, 0, 2)[None], rk.permute(1, 0, 2).repeat_interleave(2, 0)[None],
        tv.permute(1, 0, 2).repeat_interleave(2, 0)[None], is_causal=True)[0].permute(1, 0, 2)
    np.testing.assert_allclose(A.attention_full(q, k, v, theta), o.numpy(), atol=1e-12)


def test_suffix_equals_full_recompute_through_paged_pool():
    n, c, Hq, Hkv, D = 75, 32, 4, 2, 16
    q, k, v = _rand(n, Hq, Hkv, D, seed=6)
    full = A.attention_full(q, k, v, 1e4)
    pool = A.PagedPool(16, Hkv, D)
    table = [9, 3, 14, 0, 7]
    pool.append(table, 0, k[:c], v[:c], 1e4)                 # an "earlier request" wrote the prefix
    out = A.attention_suffix(pool, table, c, q[c:], k[c:], v[c:], 1e4)
    assert np.array_equal(out, full[c:])


def test_bf16_conversion_helpers():
    x = np.array([1.0, -2.5, 3.140625, 1e-3, 65504.0, 1.00390625, 1.01171875], dtype=np.float32)
    bits = tracegen.f32_to_bf16_bits(x)
    ref = torch.from_numpy(x).to(torch.bfloat16)
    assert np.array_equal(bits.view(np.int16), ref.view(torch.int16).numpy())
    np.testing.assert_array_equal(tracegen.bf16_bits_to_f64(bits), ref.double().numpy())


@pytest.mark.parametrize("strategy", ["retrieval", "greedy"])
def test_pipeline_cfg1_prefix_cached_equals_full_recompute(strategy):
    trace = tracegen.make_trace(tracegen.CONFIGS[1])
    res = P.run_trace(trace, strategy)
    assert len(res.requests) == 4
    hits = 0
    for rr in res.requests:
        full = P.full_recompute(trace, rr)
        assert rr.out.shape == (trace.cfg.n - rr.n_cached, 2, 64)
        assert np.array_equal(rr.out, full[rr.n_cached:])
        hits += rr.n_cached
    if strategy == "greedy":
        assert hits > 0


def test_pipeline_greedy_never_fewer_hits_than_retrieval_cfg1_and_bruteforce():
    trace = tracegen.make_trace(tracegen.CONFIGS[1])
    g = P.run_trace(trace, "greedy", compute=False)
    r = P.run_trace(trace, "retrieval", compute=False)
    assert sum(x.n_cached for x in g.requests) >= sum(x.n_cached for x in r.requests)


def test_pipeline_waves_on_tiny_pool():
    import dataclasses
    cfg = dataclasses.replace(tracegen.CONFIGS[1], NB=30, admission="waves", n_req=4)
    trace = tracegen.make_trace(cfg)
    res = P.run_trace(trace, "greedy")
    assert res.waves >= 2
    for rr in res.requests:
        assert np.array_equal(rr.out, P.full_recompute(trace, rr)[rr.n_cached:])


def test_flops_formula():
    # 4*Hq*D*[n(n+1)/2 - c(c+1)/2]: count (row,key) pairs by brute force
    n, c = 37, 16
    pairs = sum(p + 1 for p in range(c, n))
    assert P.attention_flops(2, 8, n, c) == 4 * 2 * 8 * pairs
