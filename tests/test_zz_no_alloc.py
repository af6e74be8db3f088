"""cw_prefill_attn_static: the attention call for callers that cannot allocate device memory.

cw_prefill_attn wants a d_work scratch from the caller.  Code that lives inside another program's process and only ever
sees the tensors of its op (a custom-op slot of an inference server, a plugin), code that runs where the allocator is off
limits (a serving loop after warm-up), or a C caller with no allocator at all has no such buffer to give.  For those the
library carries a 2 MiB work list of its own (one per GPU, shared by all calls) and cw_prefill_attn_static uses it.

This file checks, on the GPU, that the static entry point gives what the existing path gives, on TWO calls in a row: the
second batch is smaller and differently shaped than the first, so the array still holds items of the first call when the
second one runs, and anything the call forgot to reset (claim counter, item count, error flags) would show.  It also
checks that a batch beyond the array's capacity is refused up front.

The file name sorts last on purpose: pytest -x stops at the first failure, and a failure here must not hide the parity
tests.  It builds its own contexts and inputs, so it passes alone in a fresh process as well as after the other files.
"""
import numpy as np
import pytest

import tracegen
from paper_2606_19667_b200 import CW_ERR_INVALID, Context, CwError
from paper_2606_19667_b200.binding import STATIC_WORK_INTS

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

MAX_ABS, REL_L2 = 2e-2, 1e-2          # the tolerance of tests/test_gpu_parity.py (north_star)


def _dev_bf16(rng, dev, *shape):
    bits = tracegen.f32_to_bf16_bits(rng.standard_normal(shape, dtype=np.float32))
    return torch.from_numpy(np.ascontiguousarray(bits).view(np.int16)).view(torch.bfloat16).to(dev)


def _run_both(dev, Hq, Hkv, D, cs, ss, seed):
    """One varlen batch (request r: cs[r] tokens already cached, ss[r] suffix rows) through cw_append_kv, then through
    cw_prefill_attn (caller's scratch) and cw_prefill_attn_static (the library's array).  Returns both outputs as fp64."""
    rng = np.random.default_rng(seed)
    B = len(cs)
    ns = [c + s for c, s in zip(cs, ss)]
    nblk = [-(-n // 16) for n in ns]
    max_blocks, NB = max(nblk), sum(nblk) + 5
    perm = rng.permutation(NB).astype(np.int32)
    tables = np.zeros((B, max_blocks), dtype=np.int32)
    o = 0
    for r in range(B):
        tables[r, :nblk[r]] = perm[o:o + nblk[r]]
        o += nblk[r]
    ctx = Context(NB, Hq, Hkv, D, 4, rope_theta=5e5, max_position=max(ns), device=dev)
    d_tables = torch.from_numpy(tables).to(dev)

    def append(lo, hi):
        lens = [h - l for l, h in zip(lo, hi)]
        cu = np.zeros(B + 1, dtype=np.int32)
        cu[1:] = np.cumsum(lens)
        T = int(cu[-1])
        q, k, v = _dev_bf16(rng, dev, T, Hq, D), _dev_bf16(rng, dev, T, Hkv, D), _dev_bf16(rng, dev, T, Hkv, D)
        qr = torch.empty_like(q)
        d_cu = torch.from_numpy(cu).to(dev)
        d_nc = torch.from_numpy(np.asarray(lo, dtype=np.int32)).to(dev)
        ctx.cw_append_kv(q, k, v, qr, d_cu, d_nc, d_tables, max_blocks, B, T)
        return qr, d_cu, d_nc, T

    if any(cs):
        append([0] * B, cs)                                  # the cached prefix
    qr, d_cu, d_nc, T = append(cs, ns)                       # the suffix rows
    d_kv_len = torch.from_numpy(np.asarray(ns, dtype=np.int32)).to(dev)

    out_ref = torch.full_like(qr, float("nan"))
    d_work = torch.empty(ctx.cw_attn_work_ints(B, T), dtype=torch.int32, device=dev)
    ctx.cw_prefill_attn(qr, out_ref, d_cu, d_nc, d_tables, max_blocks, B, T, max(ss), max(ns), d_work, d_kv_len=d_kv_len)

    out_st = torch.full_like(qr, float("nan"))
    d_status = torch.full((4,), -1, dtype=torch.int32, device=dev)
    ctx.cw_prefill_attn_static(qr, out_st, d_cu, d_nc, d_tables, max_blocks, B, T, max(ss), max(ns), d_status=d_status,
                               d_kv_len=d_kv_len)
    torch.cuda.synchronize()
    hdr_ref, hdr_st = d_work[:4].cpu().numpy(), d_status.cpu().numpy()
    assert hdr_ref[1] == 0 and hdr_st[1] == 0, "a request descriptor was rejected on the device"
    assert hdr_st[3] == hdr_ref[3] > 0, f"item counts differ: static {hdr_st[3]}, caller scratch {hdr_ref[3]}"
    return out_ref.double().cpu().numpy(), out_st.double().cpu().numpy(), int(hdr_st[3])


def _assert_same(ref, got, what):
    assert np.isfinite(ref).all() and np.isfinite(got).all(), f"{what}: non-finite output"
    d = got - ref
    max_abs, rel = float(np.abs(d).max()), float(np.linalg.norm(d) / np.linalg.norm(ref))
    assert max_abs <= MAX_ABS and rel <= REL_L2, f"{what}: max_abs={max_abs:.3e} rel_l2={rel:.3e}"


def test_static_work_list_matches_the_callers_scratch_twice_in_a_row():
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device (there is no CPU fallback)")
    dev = "cuda:0"
    # first call: Llama-3-8B head shape, several tiles per request, cached prefixes, a ragged tail
    ref1, got1, items1 = _run_both(dev, 32, 8, 128, cs=[0, 256, 64, 1024, 16], ss=[517, 130, 1, 333, 64], seed=11)
    _assert_same(ref1, got1, "first call")
    # second call right behind it: another head shape (g = 7, D = 128) and far fewer items, so the array is still full of
    # the first call's items beyond the new count
    ref2, got2, items2 = _run_both(dev, 28, 4, 128, cs=[48, 0], ss=[19, 40], seed=12)
    assert items2 < items1
    _assert_same(ref2, got2, "second call")


def test_static_work_list_refuses_a_batch_beyond_its_capacity():
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device (there is no CPU fallback)")
    dev = "cuda:0"
    ctx = Context(8, 32, 8, 128, 4, rope_theta=5e5, max_position=64, device=dev)
    B, T = 70000, 70000                                       # 8 kv heads x >= 70000 items: beyond 65535
    assert ctx.cw_attn_work_ints(B, T) > STATIC_WORK_INTS
    dummy = torch.zeros(16, dtype=torch.int32, device=dev)    # never dereferenced: the size check comes first
    with pytest.raises(CwError) as e:
        ctx.cw_prefill_attn_static(dummy, dummy, dummy, dummy, dummy, 4, B, T, 1, 64)
    assert e.value.code == CW_ERR_INVALID and "static work list" in str(e.value)
