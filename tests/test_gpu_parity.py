"""GPU parity tests (-m gpu): the CUDA path, called through the C ABI (ctypes binding), against the fp64 oracle
on the same seeded inputs, element by element.

Bars (BASELINE.json north_star): bit-exact for orders / block tables / n_cached; RoPE'd bf16 values within
1 bf16 ulp of the fp64 result; attention outputs max|d| <= 2e-2 and ||d||2/||ref||2 <= 1e-2 against the fp64 oracle.
"""
import numpy as np
import pytest

import tracegen
from oracle import attention as oattn
from oracle.pipeline import full_recompute, run_trace
from paper_2606_19667_b200 import Context, CwError
from paper_2606_19667_b200.engine import TraceRunner

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

MAX_ABS, REL_L2 = 2e-2, 1e-2          # north_star tolerances for bf16 attention outputs


@pytest.fixture(scope="module")
def dev():
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device (there is no CPU fallback)")
    return "cuda:0"


def to_dev(bits: np.ndarray, dev):
    return torch.from_numpy(np.ascontiguousarray(bits).view(np.int16)).view(torch.bfloat16).to(dev)


def to_bits(t) -> np.ndarray:
    return t.contiguous().view(torch.int16).cpu().numpy().view(np.uint16)


def rand_bits(rng, *shape):
    return tracegen.f32_to_bf16_bits(rng.standard_normal(shape, dtype=np.float32))


def assert_close_attn(got_bits, ref, what=""):
    got = tracegen.bf16_bits_to_f64(got_bits).reshape(ref.shape)
    d = got - ref
    max_abs = float(np.abs(d).max())
    rel = float(np.linalg.norm(d) / np.linalg.norm(ref))
    assert np.isfinite(got).all(), f"{what}: non-finite output"
    assert max_abs <= MAX_ABS and rel <= REL_L2, f"{what}: max_abs={max_abs:.3e} rel_l2={rel:.3e}"
    return max_abs, rel


def assert_bf16_ulp(got_bits, ref, what=""):
    """|got - ref| <= 1 bf16 ulp of ref (ulp <= 2^-7 |ref|), plus the subnormal floor."""
    got = tracegen.bf16_bits_to_f64(got_bits).reshape(ref.shape)
    err = np.abs(got - ref)
    bound = np.abs(ref) * 2.0 ** -7 + 1e-30
    bad = err > bound
    assert not bad.any(), f"{what}: {bad.sum()} elements off by more than 1 bf16 ulp (max err {err.max():.3e})"


def unpack_q_roped(flat_bits, s, Hq, Hkv, D):
    """tile-packed q_roped slice of one request (cacheweaver.h: cw_q_roped_offset) -> plain [s, Hq, D]."""
    g = Hq // Hkv
    tpt = 128 // g
    tok, head, d = np.meshgrid(np.arange(s), np.arange(Hq), np.arange(D), indexing="ij")
    kvh, hh, t = head // g, head % g, tok // tpt
    row = (tok % tpt) * g + hh
    rows = np.minimum(tpt, s - t * tpt) * g
    off = kvh * s * g * D + t * (tpt * g) * D + (d // 64) * rows * 64 + row * 64 + ((((d % 64) // 8) ^ (row % 8)) * 8) + d % 8
    assert np.array_equal(np.sort(off.ravel()), np.arange(s * Hq * D)), "the layout must be a permutation"
    return flat_bits.reshape(-1)[off]


class Batch:
    """Hand-built varlen batch: request r has n_cached c[r] (multiple of 16) and suffix length s[r]; block tables are
    a seeded permutation of the pool.  The prefix K/V is written by a first cw_append_kv call with c = 0."""

    def __init__(self, dev, Hq, Hkv, D, cs, ss, theta=5e5, seed=0, NB=None):
        rng = np.random.default_rng(seed)
        self.dev, self.Hq, self.Hkv, self.D, self.theta = dev, Hq, Hkv, D, theta
        self.cs, self.ss = list(cs), list(ss)
        self.B = len(cs)
        self.ns = [c + s for c, s in zip(cs, ss)]
        nblk = [-(-n // 16) for n in self.ns]
        self.max_blocks = max(nblk)
        NB = NB or sum(nblk) + 3
        perm = rng.permutation(NB).astype(np.int32)
        self.tables = np.zeros((self.B, self.max_blocks), dtype=np.int32)
        o = 0
        for r in range(self.B):
            self.tables[r, :nblk[r]] = perm[o:o + nblk[r]]
            o += nblk[r]
        self.q = [rand_bits(rng, n, Hq, D) for n in self.ns]
        self.k = [rand_bits(rng, n, Hkv, D) for n in self.ns]
        self.v = [rand_bits(rng, n, Hkv, D) for n in self.ns]
        self.ctx = Context(NB, Hq, Hkv, D, 4, rope_theta=theta, max_position=max(self.ns), device=dev)
        self.d_tables = torch.from_numpy(self.tables).to(dev)

    def _append(self, lo, hi):
        """append positions lo[r]..hi[r]-1 of every request (rows with hi==lo contribute nothing)."""
        lens = [h - l for l, h in zip(lo, hi)]
        cu = np.zeros(self.B + 1, dtype=np.int32)
        cu[1:] = np.cumsum(lens)
        T = int(cu[-1])
        cat = lambda xs: np.concatenate([x[l:h] for x, l, h in zip(xs, lo, hi)], axis=0)
        q, k, v = (to_dev(cat(x), self.dev) for x in (self.q, self.k, self.v))
        qr = torch.empty_like(q)
        d_cu = torch.from_numpy(cu).to(self.dev)
        nc = np.asarray(lo, dtype=np.int32)
        d_nc = torch.from_numpy(nc).to(self.dev)
        self.ctx.cw_append_kv(q, k, v, qr, d_cu, d_nc, self.d_tables, self.max_blocks, self.B, T)
        return qr, cu, nc, d_cu, d_nc, T

    def run(self):
        if any(self.cs):
            self._append([0] * self.B, self.cs)
        qr, cu, nc, d_cu, d_nc, T = self._append(self.cs, self.ns)
        out = torch.full_like(qr, float("nan"))
        d_work = torch.empty(self.ctx.cw_attn_work_ints(self.B, T), dtype=torch.int32, device=self.dev)
        d_kv_len = torch.from_numpy(np.asarray(self.ns, dtype=np.int32)).to(self.dev)
        self.ctx.cw_prefill_attn(qr, out, d_cu, d_nc, self.d_tables, self.max_blocks, self.B, T, max(self.ss), max(self.ns),
                                 d_work, d_kv_len=d_kv_len)
        torch.cuda.synchronize()
        self.work_header = d_work[:8].cpu().numpy()          # [claim counter, error flags, fallbacks, items, ...]
        assert self.work_header[1] == 0, "a request descriptor was rejected on the device"
        return to_bits(qr), to_bits(out), cu

    def oracle(self, r):
        f = tracegen.bf16_bits_to_f64
        return oattn.attention_full(f(self.q[r]), f(self.k[r]), f(self.v[r]), self.theta)[self.cs[r]:]


# ---- kernel 1: fused RoPE + KV scatter --------------------------------------------------------------------
@pytest.mark.parametrize("Hq,Hkv,D", [(2, 1, 64), (32, 8, 128), (28, 4, 128)])
def test_append_kv_pool_contents_and_q_roped(dev, Hq, Hkv, D):
    b = Batch(dev, Hq, Hkv, D, cs=[0, 32, 16], ss=[37, 5, 130], seed=1)
    qr_bits, _, cu = b.run()
    f = tracegen.bf16_bits_to_f64
    for r in range(b.B):
        n, c = b.ns[r], b.cs[r]
        pos = np.arange(n)
        k_ref = oattn.rope(f(b.k[r]), pos, b.theta)
        q_ref = oattn.rope(f(b.q[r]), pos, b.theta)[c:]
        qr = unpack_q_roped(qr_bits[cu[r]:cu[r + 1]], n - c, Hq, Hkv, D)
        assert_bf16_ulp(qr, q_ref, f"q_roped r={r}")
        flat = qr_bits[cu[r]:cu[r + 1]].reshape(-1)
        for (t, h, d) in [(0, 0, 0), (n - c - 1, Hq - 1, D - 1), ((n - c) // 2, Hq // 2, 37)]:
            assert flat[b.ctx.cw_q_roped_offset(n - c, t, h, d)] == qr[t, h, d]
        k_out = torch.empty(n, Hkv, D, dtype=torch.bfloat16, device=dev)
        v_out = torch.empty_like(k_out)
        d_table = torch.from_numpy(b.tables[r]).to(dev)
        b.ctx.cw_gather_kv(d_table, n, k_out, v_out)
        torch.cuda.synchronize()
        assert_bf16_ulp(to_bits(k_out), k_ref, f"pool K r={r}")
        assert np.array_equal(to_bits(v_out), b.v[r]), "pool V must be a bit-exact copy"
        # the documented pool layout (cw_pool_offset) addresses the same elements
        kp = to_bits(b.ctx.k_pool)
        for (p, h, d) in [(0, 0, 0), (n - 1, Hkv - 1, D - 1), (n // 2, 0, D // 2 + 3), (17 % n, Hkv - 1, 9)]:
            off = b.ctx.cw_pool_offset(int(b.tables[r, p // 16]), h, p % 16, d)
            assert kp[off] == to_bits(k_out)[p, h, d]


def test_append_kv_position_zero_is_identity(dev):
    b = Batch(dev, 4, 2, 128, cs=[0], ss=[1], seed=2)
    qr_bits, out_bits, _ = b.run()
    assert np.array_equal(unpack_q_roped(qr_bits, 1, 4, 2, 128)[0], b.q[0][0])   # RoPE at p = 0 is the identity
    # row p = 0 attends only key 0: o = v_0 exactly (bit-exact bf16)
    g = 2
    for h in range(4):
        assert np.array_equal(out_bits[0, h], b.v[0][0, h // g])


def test_append_kv_skips_tokens_with_invalid_descriptors(dev):
    """cacheweaver.h (cw_append_kv): the descriptors live on the device, so a bad one cannot be rejected by the call; a token
    whose table entry is not a pool block, or whose position has no RoPE row / no table slot, must write NOTHING (no store
    outside the pool, no rotation by a clamped position), and every other token is written as usual."""
    Hq, Hkv, D = 8, 2, 128
    b = Batch(dev, Hq, Hkv, D, cs=[0, 0, 0], ss=[40, 33, 20], seed=11)
    for r in range(3):                              # unused table slots: not a block either (the Batch helper pads with 0)
        b.tables[r, -(-b.ns[r] // 16):] = -1
    good = b.tables.copy()
    b.tables[1, 1] = b.ctx.NB + 7                   # request 1, positions 16..31: not a pool block
    b.tables[2, 0] = -1                             # request 2, positions 0..15: negative id
    b.d_tables = torch.from_numpy(b.tables).to(dev)
    kp0, vp0 = b.ctx.k_pool.clone(), b.ctx.v_pool.clone()          # zero-filled pools
    qr, cu, nc, d_cu, d_nc, T = b._append([0, 0, 0], b.ns)
    # a second launch whose positions run past max_position (= 40) and past the table (3 blocks = 48 positions)
    d_nc2 = torch.from_numpy(np.asarray([30, 30, 30], dtype=np.int32)).to(dev)
    kp1, vp1 = b.ctx.k_pool.clone(), b.ctx.v_pool.clone()
    b.ctx.cw_append_kv(*(to_dev(np.concatenate(x, axis=0), dev) for x in (b.q, b.k, b.v)), torch.empty_like(qr), d_cu, d_nc2,
                       b.d_tables, b.max_blocks, b.B, T)
    torch.cuda.synchronize()
    f = tracegen.bf16_bits_to_f64
    kp, vp = to_bits(kp1), to_bits(vp1)
    for r in range(3):
        k_ref = oattn.rope(f(b.k[r]), np.arange(b.ns[r]), b.theta)
        for p in range(b.ns[r]):
            skipped = (r == 1 and 16 <= p < 32) or (r == 2 and p < 16)
            blk = int(good[r, p // 16])
            off = b.ctx.cw_pool_offset(blk, 1, p % 16, 5)
            if skipped:       # the block the table SHOULD have named was never touched
                assert kp[off] == 0 and vp[off] == 0
            else:
                assert abs(tracegen.bf16_bits_to_f64(kp[off:off + 1])[0] - k_ref[p, 1, 5]) <= 2.0 ** -7 * abs(k_ref[p, 1, 5]) + 1e-30   # 1 bf16 ulp
                assert vp[off] == b.v[r][p, 1, 5]
    # second launch: positions 30..39 are valid for every request and rewritten with other rows' data; positions >= 40 skipped.
    # What matters here: it ran without a fault and left every block of the pool that no valid (request, position) names alone.
    used = {int(good[r, p // 16]) for r in range(3) for p in range(b.ns[r])}
    kp2 = to_bits(b.ctx.k_pool).reshape(b.ctx.NB, -1)
    for blk in range(b.ctx.NB):
        if blk not in used:
            assert not kp2[blk].any(), f"block {blk} is in no table but was written"


# ---- kernel 2: varlen paged causal GQA attention ----------------------------------------------------------
@pytest.mark.parametrize("Hq,Hkv,D,cs,ss", [
    (2, 1, 64, [0], [224]),                                  # cfg-1 shape, cold
    (2, 1, 64, [64, 0, 192], [160, 1, 32]),                  # cfg-1 shape, cached prefixes, 1-row request
    (32, 8, 128, [0, 256], [300, 48 + 256]),                 # 8B shape, several tiles + ragged tails
    (32, 8, 128, [1280], [48]),                              # query-only suffix after a long hit
    (28, 4, 128, [512, 0], [77, 129]),                       # Qwen shape, g = 7 (rows of a head straddle tiles)
    (64, 8, 128, [128], [200]),                              # 70B shape, g = 8
])
def test_attention_matches_oracle(dev, Hq, Hkv, D, cs, ss):
    b = Batch(dev, Hq, Hkv, D, cs, ss, seed=3)
    _, out_bits, cu = b.run()
    for r in range(b.B):
        assert_close_attn(out_bits[cu[r]:cu[r + 1]], b.oracle(r), f"r={r} c={cs[r]} s={ss[r]}")


def test_attention_many_small_requests(dev):
    """2100 requests of 1-3 suffix rows: more requests than the schedule kernel keeps in shared memory (its large-batch
    path), far more items than CTAs, every item a ragged tile."""
    rng = np.random.default_rng(21)
    B = 2100
    cs = (16 * rng.integers(0, 2, size=B)).tolist()
    ss = rng.integers(1, 4, size=B).tolist()
    b = Batch(dev, 2, 1, 64, cs, ss, seed=22)
    _, out_bits, cu = b.run()
    assert b.work_header[3] == B                                  # one item per request (1 kv head, < 2 tiles)
    for r in range(0, B, 7):
        assert_close_attn(out_bits[cu[r]:cu[r + 1]], b.oracle(r), f"r={r}")


def test_attention_constant_v_and_zero_q(dev):
    """V == const => o == const; Q == 0 => o = running mean of V."""
    b = Batch(dev, 8, 2, 128, cs=[0], ss=[300], seed=4)
    b.q[0][:] = 0
    _, out_bits, _ = b.run()
    v = tracegen.bf16_bits_to_f64(b.v[0])
    mean = np.cumsum(v, axis=0) / np.arange(1, 301)[:, None, None]
    ref = np.repeat(mean, 4, axis=1)
    assert_close_attn(out_bits, ref, "running mean")


def test_empty_batch_and_bad_descriptors(dev):
    b = Batch(dev, 2, 1, 64, cs=[0], ss=[20], seed=5)
    z = torch.zeros(4, dtype=torch.int32, device=dev)
    e = torch.empty(0, 2, 64, dtype=torch.bfloat16, device=dev)
    b.ctx.cw_append_kv(e, e, e, e, z, z, z, 1, 0, 0)                           # B = T = 0: OK, no launch
    b.ctx.cw_prefill_attn(e, e, z, z, z, 1, 0, 0, 0, 0, z)
    q = torch.zeros(20, 2, 64, dtype=torch.bfloat16, device=dev)
    with pytest.raises(CwError):                                               # max_kv_len beyond the block table
        b.ctx.cw_prefill_attn(q, torch.empty_like(q), z, z, b.d_tables, b.max_blocks, 1, 20, 20, 16 * b.max_blocks + 1, z)
    # descriptors live on the device: an invalid one (here n_cached + s beyond max_kv_len) is rejected there — the request
    # produces no output and the error flag of the work header is set
    d_cu = torch.tensor([0, 20], dtype=torch.int32, device=dev)
    d_nc = torch.tensor([16], dtype=torch.int32, device=dev)
    work = torch.zeros(b.ctx.cw_attn_work_ints(1, 20), dtype=torch.int32, device=dev)
    out = torch.full_like(q, float("nan"))
    b.ctx.cw_prefill_attn(q, out, d_cu, d_nc, b.d_tables, b.max_blocks, 1, 20, 20, 20, work)
    torch.cuda.synchronize()
    assert int(work[1]) == 1 and int(work[3]) == 0 and bool(torch.isnan(out).all())
    with pytest.raises(CwError):                                               # q_roped aliases q
        b.ctx.cw_append_kv(q, q, q, q, z, z, b.d_tables, b.max_blocks, 1, 20)


# ---- whole path on the BASELINE.json traces ---------------------------------------------------------------
@pytest.mark.parametrize("strategy", ["greedy", "retrieval", "sorted", "recency", "exhaustive", "greedy_feedback",
                                      "greedy_resident"])
def test_trace_cfg1_all_rows(dev, strategy):
    trace = tracegen.make_trace(tracegen.CONFIGS[1])
    ref = run_trace(trace, strategy)
    run = TraceRunner(trace, strategy, device=dev)
    recs = run.run()
    assert len(recs) == len(ref.requests)
    for a, o in zip(recs, ref.requests):
        assert a.order == o.order and a.depth == o.depth and a.n_cached == o.n_cached
        assert a.table.tolist() == list(o.table)
        assert_close_attn(a.out, o.out, f"cfg1 {strategy} r={a.r}")
        # prefix-cached == full recompute of the same ordered prompt
        assert_close_attn(a.out, full_recompute(trace, o)[o.n_cached:], f"cfg1 {strategy} r={a.r} vs full")


@pytest.mark.parametrize("strategy", ["greedy", "greedy_feedback", "greedy_resident", "exhaustive"])
def test_trace_with_eviction_all_rows(dev, strategy):
    """A pool that holds only ~4 prompts, 30 wave-admitted requests: blocks the trie still believes resident are evicted
    (PAPER.md:129).  Orders, depths, tables bit-exact and every output row within tolerance, for the plain arm and the
    NEXT-1 arms (feedback / residency-aware) — a stale block table entry or a false hit changes K/V and fails."""
    import dataclasses
    cfg = dataclasses.replace(tracegen.CONFIGS[1], name="evict-gpu", seed=5, n_docs=8, doc_len=32, n_req=30, k=3, n_shared=2,
                              q_len=20, NB=32, H=16, admission="waves")
    trace = tracegen.make_trace(cfg)
    ref = run_trace(trace, strategy)
    recs = TraceRunner(trace, strategy, device=dev).run()
    assert ref.evictions > 0 and len(recs) == len(ref.requests)
    for a, o in zip(recs, ref.requests):
        assert (a.order, a.depth, a.n_cached, a.table.tolist(), a.wave) == (o.order, o.depth, o.n_cached, list(o.table), o.wave)
        assert_close_attn(a.out, o.out, f"evict {strategy} r={a.r}")


def test_trace_cfg2_first_requests_all_rows(dev):
    """8B shape, first 6 requests of config 2 (the oracle needs ~2 s per cold request)."""
    trace = tracegen.make_trace(tracegen.CONFIGS[2])
    reqs = list(range(6))
    ref = run_trace(trace, "greedy", requests=reqs)
    recs = TraceRunner(trace, "greedy", device=dev).run(requests=reqs)
    hits = 0
    for a, o in zip(recs, ref.requests):
        assert a.order == o.order and a.n_cached == o.n_cached and a.table.tolist() == list(o.table)
        assert_close_attn(a.out, o.out, f"cfg2 r={a.r} c={a.n_cached}")
        hits += a.n_cached
    assert hits > 0, "the greedy arm must reuse some prefix on config 2"


def test_prefill_host_equals_device_path(dev):
    """cw_prefill_host (pinned host buffers, chunked H2D / compute / D2H pipeline) gives bit-identical outputs to the
    device-buffer calls, and matches the oracle."""
    cs, ss = [0, 64, 0, 256, 16, 0, 128, 0, 32, 0], [130, 200, 1, 48, 300, 77, 64, 129, 500, 31]
    b = Batch(dev, 32, 8, 128, cs, ss, seed=7)
    _, out_dev, cu = b.run()
    b2 = Batch(dev, 32, 8, 128, cs, ss, seed=7)
    b2._append([0] * b2.B, b2.cs)                      # cached prefixes
    cat = lambda xs: np.concatenate([x[c:] for x, c in zip(xs, b2.cs)], axis=0)
    hq, hk, hv = (torch.from_numpy(cat(x).view(np.int16)).view(torch.bfloat16).pin_memory() for x in (b2.q, b2.k, b2.v))
    hout = torch.empty_like(hq).pin_memory()
    T = int(cu[-1])
    ws = torch.empty(b2.ctx.cw_prefill_host_ws_bytes(b2.B, T, b2.max_blocks), dtype=torch.uint8, device=dev)
    for _ in range(2):                                   # second call reuses the streams / events
        hout.zero_()
        b2.ctx.cw_prefill_host(hq, hk, hv, hout, cu, np.asarray(cs, np.int32), b2.tables, b2.max_blocks, b2.B, T, ws)
        got = hout.view(torch.int16).numpy().view(np.uint16)
        assert np.array_equal(got, out_dev)
    for r in range(b.B):
        assert_close_attn(out_dev[cu[r]:cu[r + 1]], b.oracle(r), f"r={r}")


def test_attention_growing_maximum_takes_the_exact_path(dev):
    """Scores that grow by far more than the lazy-rescale threshold from one KV tile to the next (keys scaled up along
    the sequence) force the speculative stale-maximum path to fall back to the exact one and rescale O.  With logits this
    large the bf16 rounding of the roped Q/K alone moves the outputs by more than 2e-2, so the reference here is the
    oracle's attention applied to the oracle's roped Q/K rounded to bf16 (what the pool holds); the plain oracle is
    still checked in relative L2."""
    b = Batch(dev, 8, 2, 128, cs=[0, 128], ss=[700, 400], seed=11)
    for r in range(b.B):
        n = b.ns[r]
        ramp = (1.0 + 7.0 * (np.arange(n) // 128) / max(1, (n - 1) // 128)).astype(np.float32)      # x1 .. x8 per KV tile
        k = tracegen.bf16_bits_to_f64(b.k[r]).astype(np.float32) * ramp[:, None, None]
        b.k[r] = tracegen.f32_to_bf16_bits(k)
    _, out_bits, cu = b.run()
    assert b.work_header[2] > 0, "the speculative softmax path must have fallen back to the exact one"
    check_against_rounded_oracle(b, out_bits, cu)


def check_against_rounded_oracle(b, out_bits, cu):
    f, rnd = tracegen.bf16_bits_to_f64, lambda x: tracegen.bf16_bits_to_f64(tracegen.f32_to_bf16_bits(x.astype(np.float32)))
    for r in range(b.B):
        n, c = b.ns[r], b.cs[r]
        pos = np.arange(n)
        q_r, k_r = rnd(oattn.rope(f(b.q[r]), pos, b.theta)), rnd(oattn.rope(f(b.k[r]), pos, b.theta))
        ref_q = oattn.attention_rows(q_r[c:], k_r, f(b.v[r]), pos[c:])
        assert_close_attn(out_bits[cu[r]:cu[r + 1]], ref_q, f"r={r} (bf16-rounded roped Q/K)")
        got = f(out_bits[cu[r]:cu[r + 1]])
        ref = b.oracle(r)
        assert np.linalg.norm(got - ref) / np.linalg.norm(ref) <= REL_L2


@pytest.mark.parametrize("col", [0, 16, 33, 5])
def test_attention_single_outlier_key_in_a_polynomial_column(dev, col):
    """One key far down the sequence whose logits exceed the running maximum by > 100 nats for many rows.  Columns 0, 1, 16,
    17 (mod 32) of a 64-key chunk take exp2 on the FMA pipe (polynomial + exponent splice): without the upper clamp the
    splice wraps and the row sum stays small, so the overflow check of the speculative path would not fire and the
    dominant key would be dropped.  The fallback counter proves the exact path ran; outputs are checked as in the
    growing-maximum test."""
    b = Batch(dev, 8, 2, 128, cs=[0, 128], ss=[520, 330], seed=13)
    for r in range(b.B):
        p = 64 * 5 + col                                        # chunk 5 of the sequence, chosen column
        k = tracegen.bf16_bits_to_f64(b.k[r]).astype(np.float32)
        k[p] *= 48.0                                            # logits of this key ~ N(0, 48^2): > +100 for ~2 % of the rows
        b.k[r] = tracegen.f32_to_bf16_bits(k)
    _, out_bits, cu = b.run()
    assert b.work_header[2] > 0, "the speculative softmax path must have fallen back to the exact one"
    check_against_rounded_oracle(b, out_bits, cu)


def test_prefill_attn_returns_before_the_stream_reaches_it(dev):
    """cw_prefill_attn reads nothing on the host: with a long cw_append_kv queued in front of it the call returns at once
    (the item list is built by a kernel on the stream), and the host side of the call stays in the tens of microseconds."""
    import time
    Hq, Hkv, D, B, s = 32, 8, 128, 48, 2048
    n = s
    nblk = n // 16
    ctx = Context(B * nblk + 8, Hq, Hkv, D, 4, rope_theta=5e5, max_position=n, device=dev)
    T = B * s
    g = torch.Generator(device=dev)
    g.manual_seed(0)
    q = torch.randn(T, Hq, D, device=dev, dtype=torch.bfloat16, generator=g)
    k = torch.randn(T, Hkv, D, device=dev, dtype=torch.bfloat16, generator=g)
    v = torch.randn(T, Hkv, D, device=dev, dtype=torch.bfloat16, generator=g)
    qr, out = torch.empty_like(q), torch.empty_like(q)
    tables = torch.arange(B * nblk, dtype=torch.int32, device=dev).reshape(B, nblk).contiguous()
    d_cu = (torch.arange(B + 1, dtype=torch.int32, device=dev) * s).contiguous()
    d_nc = torch.zeros(B, dtype=torch.int32, device=dev)
    work = torch.empty(ctx.cw_attn_work_ints(B, T), dtype=torch.int32, device=dev)
    host_us = []
    for it in range(6):
        torch.cuda.synchronize()
        for _ in range(4):                                      # ~1.6 ms of HBM-bound work in front of the attention call
            ctx.cw_append_kv(q, k, v, qr, d_cu, d_nc, tables, nblk, B, T)
        appended = torch.cuda.Event()
        appended.record()
        t0 = time.perf_counter()
        ctx.cw_prefill_attn(qr, out, d_cu, d_nc, tables, nblk, B, T, s, n, work)
        t1 = time.perf_counter()
        still_running = not appended.query()
        host_us.append(1e6 * (t1 - t0))
        assert still_running, "cw_prefill_attn returned only after the work queued in front of it had finished"
    torch.cuda.synchronize()
    assert int(work[1]) == 0 and int(work[3]) == B * Hkv * (s // (2 * (128 // (Hq // Hkv))))
    assert np.median(host_us[1:]) < 60.0, host_us               # ctypes marshalling + two launches


def test_mixed_batch_prefill_chunks_and_decode_rows(dev):
    """NEXT-4: one varlen launch holding a cold prefill, a prefix-cached suffix, the
    second chunk of a chunked prefill (133 tokens already in the pool — not a multiple of 16) and single-token decode rows
    over long contexts.  Every row against the fp64 oracle's full recompute."""
    cs = [0, 256, 133, 1000, 37, 1327, 640]
    ss = [200, 48, 100, 1, 1, 1, 1]
    b = Batch(dev, 32, 8, 128, cs, ss, seed=31)
    _, out_bits, cu = b.run()
    for r in range(b.B):
        assert_close_attn(out_bits[cu[r]:cu[r + 1]], b.oracle(r), f"r={r} past={cs[r]} rows={ss[r]}")


def test_chunked_prefill_and_decode_through_request_handles(dev):
    """cw_lookup, then the prompt's uncached suffix in one cw_prefill_requests call; then cw_extend + cw_prefill_requests
    for two more chunks (37 and 64 tokens) and four decode steps of one token each, sharing launches with a second
    request that is being prefilled.  Outputs equal the oracle's full recompute of the final sequences; block tables equal
    the oracle block manager's."""
    from oracle.blocks import BlockManager
    rng = np.random.default_rng(41)
    Hq, Hkv, D, theta, NB = 8, 2, 128, 5e5, 64
    ctx = Context(NB, Hq, Hkv, D, 4, rope_theta=theta, max_position=512, device=dev)
    obm = BlockManager(NB)
    n_final = [100 + 37 + 64 + 4, 150]
    toks = [rng.integers(0, 32000, n, dtype=np.int32) for n in n_final]
    q = [rand_bits(rng, n, Hq, D) for n in n_final]
    k = [rand_bits(rng, n, Hkv, D) for n in n_final]
    v = [rand_bits(rng, n, Hkv, D) for n in n_final]
    outs = [np.zeros((n, Hq, D), dtype=np.uint16) for n in n_final]
    reqs, oreqs, done = [None, None], [None, None], [0, 0]
    max_blocks = 16

    def launch(batch):                      # batch: list of (request index, tokens now in the sequence)
        rows = [(r, done[r], upto) for r, upto in batch]
        cat = lambda xs: to_dev(np.concatenate([xs[r][lo:hi] for r, lo, hi in rows], axis=0), dev)
        dq, dk, dv = cat(q), cat(k), cat(v)
        T = dq.shape[0]
        qr, out = torch.empty_like(dq), torch.full_like(dq, float("nan"))
        ws = torch.empty(ctx.cw_prefill_requests_ws_bytes(len(rows), T, max_blocks), dtype=torch.uint8, device=dev)
        ctx.cw_prefill_requests([reqs[r] for r, _, _ in rows], dq, dk, dv, qr, out, T, max_blocks, ws)
        torch.cuda.synchronize()
        o, pos = to_bits(out), 0
        for r, lo, hi in rows:
            outs[r][lo:hi] = o[pos:pos + hi - lo]
            pos += hi - lo
            done[r] = hi

    # step 1: request 0 admitted with its first 100 tokens
    reqs[0], table, c = ctx.cw_lookup(toks[0][:100])
    oreqs[0], otable, oc = obm.lookup(toks[0][:100])
    assert (table.tolist(), c) == (otable, oc)
    done[0] = c
    launch([(0, 100)])
    # step 2: request 0 grows by a 37-token chunk; request 1 is admitted (150 tokens) and prefilled in the same launch
    assert ctx.cw_extend(reqs[0], toks[0][100:137]).tolist() == obm.extend(oreqs[0], toks[0][100:137])
    reqs[1], table, c = ctx.cw_lookup(toks[1])
    oreqs[1], otable, oc = obm.lookup(toks[1])
    assert (table.tolist(), c) == (otable, oc)
    done[1] = c
    launch([(0, 137), (1, 150)])
    # step 3: a 64-token chunk, then four decode steps
    assert ctx.cw_extend(reqs[0], toks[0][137:201]).tolist() == obm.extend(oreqs[0], toks[0][137:201])
    launch([(0, 201)])
    for t in range(201, 205):
        assert ctx.cw_extend(reqs[0], toks[0][t:t + 1]).tolist() == obm.extend(oreqs[0], toks[0][t:t + 1])
        launch([(0, t + 1)])
    assert ctx.cw_free_list() == obm.free_list()
    f = tracegen.bf16_bits_to_f64
    for r in range(2):
        assert_close_attn(outs[r], oattn.attention_full(f(q[r]), f(k[r]), f(v[r]), theta), f"request {r}")
    # a later request with the same 201 leading tokens hits every block the chunks completed
    probe = np.concatenate([toks[0][:201], rng.integers(0, 32000, 9, dtype=np.int32)])
    assert ctx.cw_lookup(probe, peek_only=True) == 16 * obm.match(probe) == 192


def test_prefill_requests_equals_separate_calls(dev):
    """cw_prefill_requests (descriptors taken from the request handles, staged and copied by the library, three launches in
    one call) is bit-identical to cw_append_kv + cw_prefill_attn with caller-made descriptors, over two waves that share
    cached blocks."""
    trace = tracegen.make_trace(tracegen.CONFIGS[1])
    outs = {}
    for mode in ("separate", "requests"):
        run = TraceRunner(trace, "greedy", device=dev)
        if mode == "requests":
            ctx = run.ctx

            def prefill_wave(wave, keep_outputs=True, run=run, ctx=ctx):
                q, k, v = run.wave_inputs(wave)
                qr, out = torch.empty_like(q), torch.empty_like(q)
                ws = torch.empty(ctx.cw_prefill_requests_ws_bytes(wave.B, wave.T, wave.max_blocks), dtype=torch.uint8, device=dev)
                ctx.cw_prefill_requests(wave.reqs, q, k, v, qr, out, wave.T, wave.max_blocks, ws)
                torch.cuda.synchronize()
                o = out.view(torch.int16).cpu().numpy().view(np.uint16)
                for bb, rec in enumerate(wave.recs):
                    rec.out = o[wave.cu[bb]: wave.cu[bb + 1]]
            run.prefill_wave = prefill_wave
        recs = run.run()
        outs[mode] = [rec.out.copy() for rec in recs]
    for a, bb in zip(outs["separate"], outs["requests"]):
        assert np.array_equal(a, bb)


def test_prefill_requests_rejects_a_handle_listed_twice_and_leaves_the_handles_unchanged(dev):
    """A handle listed twice would have its rows counted and written twice: CW_ERR_INVALID.  The handles only move on when the
    copy and both launches were enqueued, so the same request can be prefilled by the next (correct) call with its full
    suffix (n_done used to be advanced before anything was enqueued)."""
    Hq, Hkv, D, n = 2, 1, 64, 40
    ctx = Context(8, Hq, Hkv, D, 4, rope_theta=5e5, max_position=64, device=dev)
    req, table, n_cached = ctx.cw_lookup(np.arange(n, dtype=np.int32))
    assert n_cached == 0
    rng = np.random.default_rng(5)
    q2, k2, v2 = to_dev(rand_bits(rng, 2 * n, Hq, D), dev), to_dev(rand_bits(rng, 2 * n, Hkv, D), dev), to_dev(rand_bits(rng, 2 * n, Hkv, D), dev)
    ws = torch.empty(ctx.cw_prefill_requests_ws_bytes(2, 2 * n, 3), dtype=torch.uint8, device=dev)
    with pytest.raises(CwError) as e:
        ctx.cw_prefill_requests([req, req], q2, k2, v2, torch.empty_like(q2), torch.empty_like(q2), 2 * n, 3, ws)
    assert e.value.code == -1 and "twice" in str(e.value)
    # the handle still has all n rows pending: T = n is accepted (T = 0 would be what a moved-on handle asks for)
    q, k, v = q2[:n].contiguous(), k2[:n].contiguous(), v2[:n].contiguous()
    out = torch.full_like(q, float("nan"))
    ctx.cw_prefill_requests([req], q, k, v, torch.empty_like(q), out, n, 3, ws)
    torch.cuda.synchronize()
    assert torch.isfinite(out.float()).all()
    # now the rows are written: a second call has nothing pending and T = n no longer matches
    with pytest.raises(CwError):
        ctx.cw_prefill_requests([req], q, k, v, torch.empty_like(q), out, n, 3, ws)


def test_contexts_on_two_devices_both_get_the_shared_memory_opt_in():
    """The dynamic shared memory opt-in of the attention kernel is per device: a second context on another
    GPU must launch as well.  Needs two visible GPUs."""
    if torch.cuda.device_count() < 2:
        pytest.skip("needs two visible GPUs")
    for d in (0, 1):
        with torch.cuda.device(d):
            b = Batch(f"cuda:{d}", 32, 8, 128, cs=[16], ss=[70], seed=20 + d)
            _, out, cu = b.run()
            assert_close_attn(out[cu[0]:cu[1]], b.oracle(0), f"device {d}")


def test_attention_flags_a_block_table_entry_outside_the_pool(dev):
    """cw_append_kv skips the tokens of a table entry outside [0, NB); cw_prefill_attn used to follow that entry
    into memory outside the pool.  Now the schedule kernel scans the entries every request will read, drops a request with
    a bad one (its output rows keep their fill value) and sets error bit 2 of the work header; the other requests are
    computed, and the device stays healthy (a clean batch afterwards is within tolerance of the oracle)."""
    b = Batch(dev, 32, 8, 128, cs=[0, 32], ss=[100, 40], seed=9)
    bad = b.tables.copy()
    b3 = Batch(dev, 32, 8, 128, cs=[0, 32, 16], ss=[100, 40, 50], seed=9)
    for bb, rows in ((b, [(0, 2, b.ctx.NB + 7), (1, 0, -3)]), (b3, [(1, 3, b3.ctx.NB)])):
        bad = bb.tables.copy()
        for r, i, val in rows:
            bad[r, i] = val
        bb.d_tables = torch.from_numpy(bad).to(dev)
        with pytest.raises(AssertionError, match="rejected on the device"):
            bb.run()
        assert bb.work_header[1] & 4, bb.work_header
    # b: both requests dropped -> no items at all; b3: only request 1 dropped
    assert b.work_header[3] == 0 and b3.work_header[3] > 0
    good = Batch(dev, 32, 8, 128, cs=[0, 32], ss=[100, 40], seed=9)
    _, out, cu = good.run()
    for r in range(good.B):
        assert_close_attn(out[cu[r]:cu[r + 1]], good.oracle(r), f"request {r} after the faulty batch")


def test_append_kv_skips_rows_of_a_non_monotone_cu(dev):
    """with a cu_seqlens_q that is not monotone the rows that fall outside their request's slice are skipped:
    q_roped keeps its fill value there and nothing is written outside the buffer (guard words stay intact)."""
    Hq, Hkv, D, T = 4, 2, 64, 48
    ctx = Context(8, Hq, Hkv, D, 4, rope_theta=5e5, max_position=64, device=dev)
    rng = np.random.default_rng(4)
    q, k, v = to_dev(rand_bits(rng, T, Hq, D), dev), to_dev(rand_bits(rng, T, Hkv, D), dev), to_dev(rand_bits(rng, T, Hkv, D), dev)
    guard = 4096
    buf = torch.full((T * Hq * D + 2 * guard,), 7.0, dtype=torch.bfloat16, device=dev)
    qr = buf[guard:guard + T * Hq * D]
    d_cu = torch.tensor([0, 40, 24, 48], dtype=torch.int32, device=dev)      # request 1 has a negative length
    d_nc = torch.zeros(3, dtype=torch.int32, device=dev)
    d_tables = torch.tensor([[0, 1, 2], [3, 4, 5], [6, 7, 0]], dtype=torch.int32, device=dev)
    ctx.cw_append_kv(q, k, v, qr, d_cu, d_nc, d_tables, 3, 3, T)
    torch.cuda.synchronize()
    assert torch.all(buf[:guard] == 7.0) and torch.all(buf[guard + T * Hq * D:] == 7.0), "store outside q_roped"
    assert torch.isfinite(buf.float()).all()


def test_schedule_in_front_of_append_equals_one_call(dev):
    """cw_attn_schedule needs only the descriptors: enqueued BEFORE cw_append_kv (the pools still hold nothing of the suffix)
    and followed by cw_attn_run, it gives bit for bit what cw_prefill_attn gives, and the same work header."""
    b = Batch(dev, 32, 8, 128, cs=[0, 48, 16, 128], ss=[300, 77, 1, 200], seed=21)
    _, out_ref, cu = b.run()
    hdr_ref = b.work_header.copy()
    b2 = Batch(dev, 32, 8, 128, cs=[0, 48, 16, 128], ss=[300, 77, 1, 200], seed=21)
    b2._append([0] * b2.B, b2.cs)
    cu2 = np.zeros(b2.B + 1, dtype=np.int32)
    cu2[1:] = np.cumsum(b2.ss)
    T = int(cu2[-1])
    d_cu = torch.from_numpy(cu2).to(dev)
    d_nc = torch.from_numpy(np.asarray(b2.cs, dtype=np.int32)).to(dev)
    d_work = torch.empty(b2.ctx.cw_attn_work_ints(b2.B, T), dtype=torch.int32, device=dev)
    b2.ctx.cw_attn_schedule(d_cu, d_nc, b2.d_tables, b2.max_blocks, b2.B, T, max(b2.ss), max(b2.ns), d_work)
    qr, *_ = b2._append(b2.cs, b2.ns)
    out = torch.full_like(qr, float("nan"))
    b2.ctx.cw_attn_run(qr, out, b2.d_tables, b2.max_blocks, b2.B, T, d_work)
    torch.cuda.synchronize()
    assert np.array_equal(to_bits(out), out_ref)
    hdr = d_work[:8].cpu().numpy()
    assert hdr[1] == 0 and hdr[3] == hdr_ref[3]
