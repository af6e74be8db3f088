"""GPU parity at BASELINE.json's sizes, in the launch configuration bench.py times (wave admission through
cw_admit_batch, then cw_prefill_requests = ONE cw_append_kv + ONE cw_prefill_attn per wave), checked on sampled outputs the fp64 oracle computes
row by row.  K/V are keyed by the document prefix (tracegen), so a false cache hit, a wrong block table entry or a block
evicted too early changes the sampled rows.
"""
import dataclasses

import numpy as np
import pytest

import tracegen
from oracle import attention as oattn
from oracle.pipeline import run_trace
from paper_2606_19667_b200.engine import admit_waves, make_context

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

MAX_ABS, REL_L2 = 2e-2, 1e-2


def run_waves_on_gpu(trace, strategy, dev):
    """-> list of (wave, out bits uint16 [T, Hq, D]) using the same calls as bench.py's step."""
    cfg = trace.cfg
    ctx = make_context(cfg, dev)
    results = []

    def on_wave(wave):
        rows = tracegen.batch_suffix_qkv(trace, wave.items)
        q, k, v = (torch.from_numpy(x.view(np.int16)).view(torch.bfloat16).to(dev) for x in tracegen.split_qkv(cfg, rows))
        qr, out = torch.empty_like(q), torch.full_like(q, float("nan"))
        ws = torch.empty(ctx.cw_prefill_requests_ws_bytes(wave.B, wave.T, wave.max_blocks), dtype=torch.uint8, device=dev)
        ctx.cw_prefill_requests(wave.reqs, q, k, v, qr, out, wave.T, wave.max_blocks, ws)
        torch.cuda.synchronize()
        hdr = ws[ctx.cw_prefill_requests_work_offset(wave.B, wave.max_blocks):][:16].view(torch.int32).cpu().numpy()
        assert hdr[1] == 0, "a request descriptor was rejected on the device"
        # the descriptors the library staged are the ones the admission reported
        d = ws[: 4 * (2 * wave.B + 1 + wave.B * wave.max_blocks)].view(torch.int32).cpu().numpy()
        assert np.array_equal(d[: wave.B + 1], wave.cu) and np.array_equal(d[wave.B + 1: 2 * wave.B + 1], wave.nc)
        assert np.array_equal(d[2 * wave.B + 1:].reshape(wave.B, wave.max_blocks), wave.tables)
        results.append((wave, out.view(torch.int16).cpu().numpy().view(np.uint16)))

    admit_waves(ctx, trace, strategy, on_wave=on_wave)
    return results


def oracle_rows(trace, r, order, rows, heads=None):
    """fp64 attention outputs of prompt rows `rows` (absolute positions) of request r under `order`: [len(rows), Hq, D]."""
    cfg = trace.cfg
    f = tracegen.bf16_bits_to_f64
    q, k, v = (f(x) for x in tracegen.split_qkv(cfg, tracegen.prompt_qkv(trace, r, order, 0)))
    pos = np.arange(cfg.n)
    rows = np.asarray(rows)
    return oattn.attention_rows(oattn.rope(q[rows], rows, cfg.theta), oattn.rope(k, pos, cfg.theta), v, rows)


def check_sampled(trace, results, n_requests, rows_per_request, seed):
    rng = np.random.default_rng(seed)
    cfg = trace.cfg
    flat = [(wave, out, b) for wave, out in results for b in range(wave.B)]
    picks = rng.choice(len(flat), size=min(n_requests, len(flat)), replace=False)
    picks = sorted(set(picks.tolist()) | {len(flat) - 1})            # always include the last request of the last wave
    worst = (0.0, 0.0)
    n_checked = 0
    for i in picks:
        wave, out, b = flat[i]
        rec = wave.recs[b]
        c, s = rec.n_cached, cfg.n - rec.n_cached
        local = np.unique(np.concatenate([[0, s - 1, min(s - 1, 15), min(s - 1, 16)],
                                          rng.integers(0, s, size=rows_per_request)]))
        ref = oracle_rows(trace, rec.r, rec.order, c + local)
        got = tracegen.bf16_bits_to_f64(out[wave.cu[b]:wave.cu[b + 1]][local])
        d = got - ref
        assert np.isfinite(got).all(), f"request {rec.r}: non-finite output"
        ma, rl = float(np.abs(d).max()), float(np.linalg.norm(d) / np.linalg.norm(ref))
        assert ma <= MAX_ABS and rl <= REL_L2, f"request {rec.r} (wave {rec.wave}, c={c}): max_abs={ma:.3e} rel_l2={rl:.3e}"
        worst = (max(worst[0], ma), max(worst[1], rl))
        n_checked += len(local) * cfg.Hq
    return worst, n_checked


def test_cfg2_full_size_one_wave_sampled_rows():
    """BASELINE.json configs[1] exactly as bench.py launches it: all 64 requests admitted as one wave (eager block
    registration: later requests read blocks written by kernel 1 of the same launch)."""
    dev = "cuda:0"
    cfg = tracegen.CONFIGS[2]
    trace = tracegen.make_trace(cfg)
    results = run_waves_on_gpu(trace, "greedy", dev)
    assert len(results) == 1 and results[0][0].B == 64
    # host path bit-exact against the oracle run in the same admission mode
    ref = run_trace(dataclasses.replace(trace, cfg=dataclasses.replace(cfg, admission="waves")), "greedy", compute=False)
    for rec, o in zip(results[0][0].recs, ref.requests):
        assert (rec.order, rec.n_cached, rec.table.tolist()) == (o.order, o.n_cached, list(o.table))
    assert sum(rec.n_cached for rec in results[0][0].recs) > 0
    worst, n = check_sampled(trace, results, n_requests=5, rows_per_request=24, seed=0)
    assert n >= 4096, n


@pytest.mark.parametrize("base,n_req,NB", [(4, 20, 2600), (5, 5, 1500)])
def test_concurrent_configs_waves_and_eviction_sampled_rows(base, n_req, NB):
    """Qwen2.5-7B-shaped (28q/4kv, g = 7, 5184-token prompts) and 70B-shaped (64q/8kv, 10304-token prompts) configs with
    the request count and pool scaled down together so that the trace still needs several waves and LRU eviction."""
    dev = "cuda:0"
    b = tracegen.CONFIGS[base]
    cfg = dataclasses.replace(b, name=b.name + "-small", n_req=n_req, NB=NB, H=max(1, NB // b.blocks_per_req))
    trace = tracegen.make_trace(cfg)
    results = run_waves_on_gpu(trace, "greedy", dev)
    assert len(results) >= 2, "the scaled-down pool must force several waves"
    ref = run_trace(trace, "greedy", compute=False)
    recs = [rec for wave, _ in results for rec in wave.recs]
    assert len(recs) == len(ref.requests) == n_req
    for rec, o in zip(recs, ref.requests):
        assert (rec.r, rec.order, rec.n_cached, rec.wave, rec.table.tolist()) == (o.r, o.order, o.n_cached, o.wave, list(o.table))
    worst, n = check_sampled(trace, results, n_requests=3, rows_per_request=10, seed=base)
    assert n >= 28 * 30


def run_and_check_wave_by_wave(trace, strategy, dev, requests_per_wave, rows_per_request, seed):
    """Memory-lean variant of run_waves_on_gpu + check_sampled for the full-size concurrent configs: each wave is launched
    exactly as bench.py launches it, sampled rows are checked against the oracle, and the wave's tensors are dropped."""
    import os
    cfg = trace.cfg
    ctx = make_context(cfg, dev)
    rng = np.random.default_rng(seed)
    state = {"checked": 0, "worst": (0.0, 0.0), "waves": 0, "recs": []}

    def on_wave(wave):
        rows = tracegen.batch_suffix_qkv(trace, wave.items, threads=os.cpu_count() or 8)
        q, k, v = (torch.from_numpy(x.view(np.int16)).view(torch.bfloat16).to(dev) for x in tracegen.split_qkv(cfg, rows))
        del rows
        qr, out = torch.empty_like(q), torch.full_like(q, float("nan"))
        ws = torch.empty(ctx.cw_prefill_requests_ws_bytes(wave.B, wave.T, wave.max_blocks), dtype=torch.uint8, device=dev)
        ctx.cw_prefill_requests(wave.reqs, q, k, v, qr, out, wave.T, wave.max_blocks, ws)
        torch.cuda.synchronize()
        hdr = ws[ctx.cw_prefill_requests_work_offset(wave.B, wave.max_blocks):][:16].view(torch.int32).cpu().numpy()
        assert hdr[1] == 0
        picks = sorted(set(rng.choice(wave.B, size=min(requests_per_wave, wave.B), replace=False).tolist()) | {wave.B - 1})
        for b in picks:
            rec = wave.recs[b]
            c, s = rec.n_cached, cfg.n - rec.n_cached
            local = np.unique(np.concatenate([[0, s - 1], rng.integers(0, s, size=rows_per_request)]))
            got = tracegen.bf16_bits_to_f64(out[wave.cu[b] + torch.from_numpy(local).to(dev)].view(torch.int16).cpu().numpy().view(np.uint16))
            ref = oracle_rows(trace, rec.r, rec.order, c + local)
            d = got - ref
            assert np.isfinite(got).all(), f"request {rec.r}: non-finite output"
            ma, rl = float(np.abs(d).max()), float(np.linalg.norm(d) / np.linalg.norm(ref))
            assert ma <= MAX_ABS and rl <= REL_L2, f"request {rec.r} (wave {rec.wave}, c={c}): max_abs={ma:.3e} rel_l2={rl:.3e}"
            state["worst"] = (max(state["worst"][0], ma), max(state["worst"][1], rl))
            state["checked"] += len(local) * cfg.Hq
        state["waves"] += 1
        state["recs"].extend(wave.recs)
        del q, k, v, qr, out, ws

    admit_waves(ctx, trace, strategy, on_wave=on_wave)
    return state


@pytest.mark.parametrize("cfg_id,requests_per_wave,rows_per_request", [(4, 16, 6), (5, 8, 6)])
def test_concurrent_configs_at_full_size(cfg_id, requests_per_wave, rows_per_request):
    """BASELINE.json configs[3] (256 Qwen-shaped requests, 32768-block pool, 3 waves) and configs[4] (32 70B-shaped
    requests, 16384-block pool, 2 waves) at FULL size, launched wave by wave as bench.py does (cw_admit_batch +
    cw_prefill_requests); >= 4096 sampled (request, head, row) outputs against the fp64 oracle; host path bit-exact."""
    cfg = tracegen.CONFIGS[cfg_id]
    trace = tracegen.make_trace(cfg)
    st = run_and_check_wave_by_wave(trace, "greedy", "cuda:0", requests_per_wave, rows_per_request, seed=cfg_id)
    assert st["waves"] >= 2 and st["checked"] >= 4096, st
    ref = run_trace(trace, "greedy", compute=False)
    assert len(st["recs"]) == len(ref.requests) == cfg.n_req
    for rec, o in zip(st["recs"], ref.requests):
        assert (rec.r, rec.order, rec.n_cached, rec.wave, rec.table.tolist()) == (o.r, o.order, o.n_cached, o.wave, list(o.table))


@pytest.mark.parametrize("k,overlap", [(3, 60), (10, 90)])
def test_sweep_cells_sampled_rows(k, overlap):
    """two cells of BASELINE.json configs[2] (the overlap x top-k sweep at the 8B shapes): k = 3 (n = 816) and k = 10
    (n = 2608), all 128 requests admitted as bench.py --sweep does, sampled rows against the oracle."""
    cfg = dataclasses.replace(tracegen.config3(k, overlap), admission="waves")
    trace = tracegen.make_trace(cfg)
    st = run_and_check_wave_by_wave(trace, "greedy", "cuda:0", requests_per_wave=6, rows_per_request=20, seed=k)
    assert st["checked"] >= 4096, st
    ref = run_trace(trace, "greedy", compute=False)
    for rec, o in zip(st["recs"], ref.requests):
        assert (rec.order, rec.n_cached, rec.table.tolist()) == (o.order, o.n_cached, list(o.table))
    assert sum(rec.n_cached for rec in st["recs"]) > 0
