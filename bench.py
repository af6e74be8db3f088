"""bench.py — prefix-cached prefill (CacheWeaver hot path) on B200, one process per GPU.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 2] [--impl ours|reference]

A *step* is one pass of the whole hot path over one batch of synthetic input: the requests
of the configuration are admitted on the host in ONE cw_admit_batch call on a reset context (greedy trie order,
prompt assembly, chained block hashes, prefix match, pin/allocate/evict, trie insert), then ONE cw_append_kv launch
(fused RoPE + KV scatter) and ONE cw_prefill_attn launch (varlen paged causal GQA attention) over all suffixes,
then cw_release_batch.  Workload at N=1: BASELINE.json configs[1] (Llama-3-8B-shaped layer, 64 requests, 200x256-token
documents, top-k 5, 60 % adjacent overlap, 8192-block pool).  Metric: attention TFLOP/s over algorithmic flops
4*Hq*D*[n(n+1)/2 - c(c+1)/2] per request (BASELINE.json `metric`), plus batch prefill ms for greedy vs retrieval order.
The path does not shard (BASELINE.json north_star: one GPU): --gpus N runs N independent replicas ("replicas only").
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import tracegen  # noqa: E402

METRIC = "prefill-attn TFLOP/s (% bf16 peak); batch prefill ms, greedy vs retrieval order"
UNIT = "TFLOP/s"


def attention_flops(cfg, n_cached):
    n = cfg.n
    return sum(4 * cfg.Hq * cfg.D * (n * (n + 1) // 2 - int(c) * (int(c) + 1) // 2) for c in n_cached)


def append_bytes(cfg, T):
    """algorithmic bytes of cw_append_kv: q in + q' out + k,v in + pool K,V out + 4 B descriptor per token."""
    return int(T) * (2 * cfg.Hq * cfg.D * 2 + 2 * 2 * cfg.Hkv * cfg.D * 2 + 4)


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return {"bf16": float(d["bf16_tflops"]), "bf16_sustained": float(d.get("bf16_tflops_sustained", d["bf16_tflops"])),
                "hbm": float(d["hbm_gbs"]), "source": "measured (MEASURED_PEAKS.json, burst)"}
    return {"bf16": 1590.0, "bf16_sustained": 1400.0, "hbm": 6650.0, "source": "fallback (B200_PROFILING.md)"}


def traffic_from_profile(cfg_name, kernel):
    """dram__bytes_read + dram__bytes_write per launch of `kernel` on configuration `cfg_name`, from the committed ncu
    capture listed in profiles/traffic.json; None when that configuration was never captured."""
    p = os.path.join(ROOT, "profiles", "traffic.json")
    if os.path.exists(p):
        return json.load(open(p)).get(cfg_name, {}).get(kernel)
    return None


class ClockSampler:
    """nvidia-smi clocks / throttle reasons DURING the timed region (B200_PROFILING.md clocks line).  The sampler process is
    started before the warm-up (it needs ~100 ms to deliver its first line, longer than a short timed region); only the
    lines whose own timestamp falls between begin() and end() are summarised."""
    Q = ("timestamp,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0, period_ms=20):
        self.rows, self.proc, self.index, self.period_ms = [], None, index, period_ms
        self.t_begin = self.t_end = None

    def __enter__(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", str(self.period_ms)],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except OSError:
            self.proc = None
        return self

    def begin(self):
        self.t_begin = time.time()

    def end(self):
        self.t_end = time.time()

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def __exit__(self, *a):
        if self.proc:
            time.sleep(0.06)
            self.proc.terminate()
            self.t.join(timeout=2)

    @staticmethod
    def _stamp(text):
        import datetime
        try:
            return datetime.datetime.strptime(text, "%Y/%m/%d %H:%M:%S.%f").timestamp()
        except ValueError:
            return None

    def summary(self):
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        t0 = self.t_begin if self.t_begin is not None else float("-inf")
        t1 = self.t_end if self.t_end is not None else float("inf")
        parsed = []
        for r in self.rows:
            try:
                parsed.append((self._stamp(r[0]), float(r[1]), float(r[2]), r[4:8]))
            except (ValueError, IndexError):
                continue
        inside = [x for x in parsed if x[0] is not None and t0 - 1e-3 <= x[0] <= t1 + 1e-3]
        window = "timed region"
        if not inside and parsed and self.t_begin is not None:
            # the region was shorter than the sampling period: the sample closest to it (taken under the same load, during the
            # warm-up steps just before or the steps just after)
            mid = 0.5 * (t0 + t1)
            inside = [min((x for x in parsed if x[0] is not None), key=lambda x: abs(x[0] - mid), default=None)]
            inside = [x for x in inside if x is not None]
            window = "nearest sample to the timed region"
        if not inside:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        reasons = set()
        for x in inside:
            for nm, v in zip(names, x[3]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        return {"sm_mhz": float(np.median([x[1] for x in inside])), "sm_max_mhz": float(max(x[2] for x in inside)),
                "reasons": sorted(reasons), "samples": len(inside), "window": window}


# ---------------------------------------------------------------------------------------------- our arm ----
class Workload:
    """One configuration, one strategy: seeded trace, resident inputs, and the step function."""
    RING = 4

    def __init__(self, cfg_id, strategy, device, want_e2e=True, device_inputs=False, sequential=False, real_waves=0):
        import torch
        from paper_2606_19667_b200.engine import admit_waves, make_context
        self.torch, self.device, self.strategy = torch, device, strategy
        self.cfg = cfg = tracegen.CONFIGS[cfg_id] if isinstance(cfg_id, int) else cfg_id
        self.trace = trace = tracegen.make_trace(cfg)
        self.ctx = make_context(cfg, device)
        self.doc_ids = np.asarray(trace.retrieval, dtype=np.int64)
        # dry admission (host only) fixes the wave boundaries and suffix descriptors; every step repeats it for real
        self.sequential = sequential          # one request per wave (per-request launches) instead of as many as fit
        self.waves = admit_waves(self.ctx, trace, strategy, force_waves=not sequential)
        self.ctx.cw_reset()
        self.flops = sum(attention_flops(cfg, w.nc) for w in self.waves)
        self.T = sum(w.T for w in self.waves)
        self.hit_blocks = sum(int(w.nc.sum()) // 16 for w in self.waves)
        self.max_blocks = cfg.blocks_per_req
        Bmax = max(w.B for w in self.waves)
        self.inputs, self.host_inputs = [], []
        for wi, w in enumerate(self.waves):
            if device_inputs and wi >= real_waves:
                # timing-only runs of the large configs / the sweep: seeded N(0,1) bf16 drawn on the device (the values do
                # not change the work; parity at these shapes is covered by tests/test_gpu_full_size.py with tracegen inputs)
                g = torch.Generator(device=device)
                g.manual_seed(cfg.seed * 1000 + wi)
                dq, dk, dv = (torch.randn(w.T, h, cfg.D, device=device, dtype=torch.bfloat16, generator=g)
                              for h in (cfg.Hq, cfg.Hkv, cfg.Hkv))
                work = torch.empty(self.ctx.cw_attn_work_ints(w.B, w.T), dtype=torch.int32, device=device)
                self.inputs.append((dq, dk, dv, torch.empty_like(dq), torch.empty_like(dq), work))
                continue
            rows = tracegen.batch_suffix_qkv(trace, w.items, threads=os.cpu_count() or 8)
            qkv = [torch.from_numpy(x.view(np.int16)).view(torch.bfloat16) for x in tracegen.split_qkv(cfg, rows)]
            if want_e2e and not device_inputs:
                self.host_inputs.append([t.pin_memory() for t in qkv] + [torch.empty_like(qkv[0]).pin_memory()])
            dq, dk, dv = (t.to(device) for t in qkv)
            work = torch.empty(self.ctx.cw_attn_work_ints(w.B, w.T), dtype=torch.int32, device=device)
            self.inputs.append((dq, dk, dv, torch.empty_like(dq), torch.empty_like(dq), work))
        # pinned staging ring for the admission outputs + device descriptors
        self.ring = []
        for _ in range(self.RING):
            # Bmax + 1 rows: the request that closes a wave (CW_ERR_NO_SPACE) still gets its order written
            st = {"orders": torch.empty(Bmax + 1, cfg.k, dtype=torch.int64).pin_memory(),
                  "pred": torch.empty(Bmax + 1, dtype=torch.int32).pin_memory(),
                  "reqs": torch.empty(Bmax + 1, dtype=torch.int64).pin_memory(),
                  "tables": torch.empty(Bmax + 1, self.max_blocks, dtype=torch.int32).pin_memory(),
                  "n_cached": torch.empty(Bmax + 1, dtype=torch.int32).pin_memory(),
                  "cu": torch.empty(Bmax + 2, dtype=torch.int32).pin_memory()}
            st["np"] = {k: v.numpy() for k, v in st.items()}
            st["d_tables"] = torch.empty(Bmax, self.max_blocks, dtype=torch.int32, device=device)
            st["d_nc"] = torch.empty(Bmax, dtype=torch.int32, device=device)
            st["d_cu"] = torch.empty(Bmax + 1, dtype=torch.int32, device=device)
            st["event"] = None
            self.ring.append(st)
        self.slot, self.Bmax = 0, Bmax
        self.side = torch.cuda.Stream(device=device)
        self.req_ws = None
        if sequential:      # per-request path: cw_prefill_requests stages the descriptors itself (one call per request)
            self.req_ws = torch.empty(max(self.ctx.cw_prefill_requests_ws_bytes(w.B, w.T, self.max_blocks) for w in self.waves),
                                      dtype=torch.uint8, device=device)
        self.ws = None
        if want_e2e and not device_inputs:
            nbytes = max(self.ctx.cw_prefill_host_ws_bytes(w.B, w.T, self.max_blocks) for w in self.waves)
            self.ws = torch.empty(nbytes, dtype=torch.uint8, device=device)
        self.queries = np.ascontiguousarray(trace.query_tokens)
        self.launches = 0
        self.h2d = self.d2h = 0

    def _admit(self, lo, expect):
        st = self.ring[self.slot]
        self.slot = (self.slot + 1) % self.RING
        if st["event"] is not None:
            st["event"].synchronize()
        hi = lo + (expect.B if self.sequential else self.Bmax + 1)
        a = self.ctx.cw_admit_batch(self.doc_ids[lo:hi], self.strategy, self.trace.doc_tokens,
                                    self.queries[lo:hi], self.max_blocks, out=st["np"])
        if a["admitted"] != expect.B:
            raise RuntimeError(f"admission diverged: {a['admitted']} != {expect.B}")
        return st, a

    def step(self, events=None):
        """resident inputs: host admission + H2D of the descriptors + 3 launches per wave (schedule on a side stream beside
        RoPE + scatter, then attention).  The per-request variant (sequential=True) goes through cw_prefill_requests instead: one C call per
        request stages the descriptors and enqueues the same three launches."""
        torch, ctx = self.torch, self.ctx
        ctx.cw_reset()
        lo = 0
        for wi, w in enumerate(self.waves):
            st, a = self._admit(lo, w)
            B, T = w.B, w.T
            if self.req_ws is not None:
                q, k, v, qr, out, _ = self.inputs[wi]
                ctx.cw_prefill_requests(a["reqs"][:B], q, k, v, qr, out, T, self.max_blocks, self.req_ws)
                ctx.cw_release_batch(a["reqs"][:B])
                self.launches += 3
                lo += B
                continue
            st["d_tables"][:B].copy_(st["tables"][:B], non_blocking=True)
            st["d_nc"][:B].copy_(st["n_cached"][:B], non_blocking=True)
            st["d_cu"][:B + 1].copy_(st["cu"][:B + 1], non_blocking=True)
            q, k, v, qr, out, work = self.inputs[wi]
            # the schedule kernel (descriptors -> item list) needs neither q_roped nor the pools: it runs on a side stream
            # beside cw_append_kv, forked behind the descriptor copies and joined in front of the attention kernel
            main = torch.cuda.current_stream()
            self.side.wait_stream(main)
            with torch.cuda.stream(self.side):
                ctx.cw_attn_schedule(st["d_cu"], st["d_nc"], st["d_tables"], self.max_blocks, B, T, w.max_q, w.max_kv, work)
            if events is not None:
                e = [torch.cuda.Event(enable_timing=True) for _ in range(3)]
                e[0].record()
            ctx.cw_append_kv(q, k, v, qr, st["d_cu"], st["d_nc"], st["d_tables"], self.max_blocks, B, T)
            main.wait_stream(self.side)
            if events is not None:
                e[1].record()
            ctx.cw_attn_run(qr, out, st["d_tables"], self.max_blocks, B, T, work)
            if events is not None:
                e[2].record()
                events.append(e)
            st["event"] = torch.cuda.Event()
            st["event"].record()
            ctx.cw_release_batch(a["reqs"][:B])
            self.launches += 3
            lo += B

    def host_admission(self, reps=3):
        """host path alone (a1-a6 + a9 for every request of the configuration): us per request, and the predicted-vs-actual
        prefix counters of one pass (cw_stats)."""
        t0 = time.perf_counter()
        for _ in range(reps):
            self.ctx.cw_reset()
            lo = 0
            for w in self.waves:
                st, a = self._admit(lo, w)
                self.ctx.cw_release_batch(a["reqs"][:w.B])
                lo += w.B
        us = (time.perf_counter() - t0) / reps * 1e6 / self.cfg.n_req
        st = self.ctx.cw_stats()
        return us, {k: st[k] for k in ("predicted_prefix_docs", "actual_prefix_docs", "over_predicted_docs", "stale_marks",
                                       "hit_blocks", "evictions")}

    def step_e2e(self):
        """host buffers: admission + cw_prefill_host (H2D of q,k,v and descriptors, both kernels, D2H of out)."""
        ctx = self.ctx
        ctx.cw_reset()
        lo = 0
        for wi, w in enumerate(self.waves):
            st, a = self._admit(lo, w)
            hq, hk, hv, hout = self.host_inputs[wi]
            ctx.cw_prefill_host(hq, hk, hv, hout, a["cu"], a["n_cached"], a["tables"][:w.B], self.max_blocks, w.B, w.T, self.ws)
            ctx.cw_release_batch(a["reqs"][:w.B])
            self.h2d += (hq.numel() + hk.numel() + hv.numel()) * 2 + 4 * (2 * w.B + 1 + w.B * self.max_blocks)
            self.d2h += hout.numel() * 2
            lo += w.B
        return hout


# --------------------------------------------------------------------------------------- oracle timing ----
def oracle_threads():
    try:
        from threadpoolctl import threadpool_info
        n = [p.get("num_threads", 1) for p in threadpool_info()]
        return max(n) if n else 1
    except Exception:
        return 1


class OracleSample:
    """The oracle as it stands (oracle/, fp64 numpy), timed on a bounded sample: the first `n_req` requests of the
    configuration, greedy order, sequential: order/lookup/observe + RoPE + pool append + suffix attention + release.
    Inputs are generated before the timed region."""

    def __init__(self, cfg_id, n_req, max_rows=None):
        from oracle.pipeline import run_trace
        self.cfg = cfg = tracegen.CONFIGS[cfg_id] if isinstance(cfg_id, int) else cfg_id
        self.trace = tracegen.make_trace(cfg)
        self.reqs = list(range(min(n_req, cfg.n_req)))
        dry = run_trace(self.trace, "greedy", compute=False, requests=self.reqs)
        # max_rows bounds the sample further for the long prompts (cfg 5: one request is ~70 s of fp64 numpy): only the first
        # max_rows suffix rows of each sampled request are prefilled (a prompt cut after n_cached + max_rows tokens)
        self.max_rows = max_rows
        self.flops = sum(4 * cfg.Hq * cfg.D * (m * (m + 1) // 2 - rr.n_cached * (rr.n_cached + 1) // 2)
                         for rr in dry.requests for m in [min(cfg.n, rr.n_cached + (max_rows or cfg.n))])
        for rr in dry.requests:                       # warm tracegen's chunk cache: no RNG inside the timed region
            tracegen.prompt_qkv(self.trace, rr.r, rr.order, rr.n_cached, cache=True)
        self.dry = dry

    def run(self):
        from oracle.attention import PagedPool, attention_suffix
        from oracle.blocks import BlockManager
        from oracle.ordering import KnowledgeTree
        cfg, trace = self.cfg, self.trace
        t0 = time.perf_counter()
        tree, bm, pool = KnowledgeTree(cfg.H), BlockManager(cfg.NB, eager_register=True), PagedPool(cfg.NB, cfg.Hkv, cfg.D)
        for r in self.reqs:
            O, _ = tree.order(trace.retrieval[r])
            tokens = tracegen.assemble_prompt(trace, r, O)
            req, table, c = bm.lookup(tokens)
            tree.observe(O)
            rows = tracegen.prompt_qkv(trace, r, O, c, cache=True)
            if self.max_rows:
                rows = rows[:self.max_rows]
            q, k, v = (tracegen.bf16_bits_to_f64(x) for x in tracegen.split_qkv(cfg, rows))
            attention_suffix(pool, table, c, q, k, v, cfg.theta)
            bm.release(req)
        return time.perf_counter() - t0


# ------------------------------------------------------------------------------------------------ main ----
def dist_env():
    return int(os.environ.get("RANK", 0)), int(os.environ.get("LOCAL_RANK", 0)), int(os.environ.get("WORLD_SIZE", 1))


def run_reference(args):
    """--impl reference: the oracle on the box's host cores (rank 0 only), same metric / unit / config."""
    rank, _, world = dist_env()
    if rank != 0:
        return
    sample = OracleSample(select_config(args), args.oracle_requests, args.oracle_rows)
    for _ in range(args.warmup):
        sample.run()
    times = [sample.run() for _ in range(args.steps)]
    total = sum(times)
    value = sample.flops * args.steps / total / 1e12
    cores = oracle_threads()
    desc = f"first {len(sample.reqs)} of {sample.cfg.n_req} requests of {sample.cfg.name} per step, sequential, greedy order" + \
           (f", first {sample.max_rows} suffix rows of each" if sample.max_rows else "")
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * total / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": f"BASELINE.json configs[{args.config - 1}] ({sample.cfg.name})", "sample": desc},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}, "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def max_over_ranks(value, dist, device):
    """MAX of a scalar over all ranks (the only inter-rank exchange of the bench: timing plumbing, not data path)."""
    if dist is None:
        return float(value)
    import torch
    t = torch.tensor([float(value)], device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_value(units_per_rank, ms_max, world):
    """whole-job throughput of `world` independent replicas ("replicas only"): all units processed / max time."""
    return world * units_per_rank / (ms_max * 1e-3) / 1e12


def timed(torch, fn, steps, dist):
    """barrier + sync, K steps, sync; device time by CUDA events on the launching (current) stream; max over ranks."""
    if dist is not None:
        dist.barrier()
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(steps):
        fn()
    e1.record()
    torch.cuda.synchronize()
    ms = max_over_ranks(e0.elapsed_time(e1), dist, "cuda")
    if dist is not None:
        dist.barrier()
    return ms


def prefill_saved(cfg, waves):
    """Per-request share of the prefill that the prefix cache saved (Table 13 reports this per
    request): token-weighted n_cached / n and flops-weighted c(c+1) / n(n+1) (causal attention pairs), p50 / mean / p95 over
    the requests of the trace.  Statistics of the admission's answers; nothing of the method is computed here."""
    c = np.concatenate([np.asarray(w.nc, dtype=np.float64) for w in waves])
    n = float(cfg.n)
    out = {}
    for name, x in (("token_weighted", c / n), ("flops_weighted", c * (c + 1) / (n * (n + 1)))):
        out[name] = {"p50": float(np.percentile(x, 50)), "mean": float(x.mean()), "p95": float(np.percentile(x, 95))}
    return out


def measure_record(torch, wl, pk, local, warmup, seconds=0.0, steps=0):
    """Attention and append figures of one workload over `steps` steps (or about `seconds` of steps), with the clocks sampled
    inside that very region: device time by CUDA events, fractions against the burst and the sustained measured peaks."""
    cfg = wl.cfg
    with ClockSampler(local) as clk:
        for _ in range(warmup):
            wl.step()
        if seconds > 0:      # device time of a few steps -> number of steps that fill `seconds`
            ms0 = timed(torch, wl.step, 3, None) / 3
            steps = max(steps, int(np.ceil(1.25 * seconds * 1e3 / max(1e-3, ms0))))   # 3 cold steps overstate the steady-state step
        ev = []
        clk.begin()
        ms = timed(torch, lambda: wl.step(ev), steps, None) / steps
        clk.end()
    app_ms = sum(e[0].elapsed_time(e[1]) for e in ev) / steps
    attn_ms = sum(e[1].elapsed_time(e[2]) for e in ev) / steps
    attn_tflops = wl.flops / (attn_ms * 1e-3) / 1e12
    app_gbs = append_bytes(cfg, wl.T) / (app_ms * 1e-3) / 1e9
    return {"workload": cfg.name, "requests": cfg.n_req, "waves": len(wl.waves), "steps": steps, "ms_per_step": ms,
            "seconds": ms * steps * 1e-3, "suffix_tokens": wl.T, "hit_blocks": wl.hit_blocks,
            "attn_ms": attn_ms, "attn_tflops": attn_tflops, "attn_frac": attn_tflops / pk["bf16"],
            "attn_frac_of_sustained": attn_tflops / pk["bf16_sustained"],
            "append_ms": app_ms, "append_gbs": app_gbs, "append_frac": app_gbs / pk["hbm"], "clocks": clk.summary()}


def run_ours(args):
    import torch
    rank, local, world = dist_env()
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device; there is no CPU fallback")
    torch.cuda.set_device(local)
    device = f"cuda:{local}"
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device(device))
    pk = peaks()
    cfg_sel = select_config(args)
    clk = ClockSampler(local)          # streaming long before the timed region (its first line takes ~100 ms)
    clk.__enter__()
    wl = Workload(cfg_sel, args.arm, device, want_e2e=not args.device_inputs, device_inputs=args.device_inputs,
                  real_waves=args.real_waves)
    cfg = wl.cfg

    for _ in range(args.warmup):
        wl.step()
    if args.seconds > 0:       # long run: as many steps as fit the requested wall time (sustained clocks / power cap)
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        wl.step()
        torch.cuda.synchronize()
        args.steps = max(args.steps, int(args.seconds / max(1e-6, time.perf_counter() - t0)))
    wl.launches = 0
    events = []
    clk.begin()
    ms = timed(torch, lambda: wl.step(events), args.steps, dist)
    clk.end()
    clk.__exit__()
    launches = wl.launches
    ms_step = ms / args.steps
    value = aggregate_value(wl.flops, ms_step, world)
    app_ms = sum(e[0].elapsed_time(e[1]) for e in events) / args.steps       # per step, all waves
    attn_ms = sum(e[1].elapsed_time(e[2]) for e in events) / args.steps
    n_l = len(wl.waves)
    attn_tflops = wl.flops / (attn_ms * 1e-3) / 1e12
    app_gbs = append_bytes(cfg, wl.T) / (app_ms * 1e-3) / 1e9

    # end to end: host buffers, H2D/D2H inside the timed region
    e2e_steps, ms_e2e, e2e_value = 0, None, None
    if not args.device_inputs:
        for _ in range(max(2, args.warmup // 2)):
            wl.step_e2e()
        wl.h2d = wl.d2h = 0
        e2e_steps = max(1, min(args.steps, args.e2e_steps))
        ms_e2e = timed(torch, wl.step_e2e, e2e_steps, dist) / e2e_steps
        e2e_value = aggregate_value(wl.flops, ms_e2e, world)

    # the sustained figure (the same step for >= 2 s: clocks settle under the power cap) beside the burst one
    sustained = None
    if world == 1 and args.sustained_seconds > 0 and args.seconds <= 0:
        sustained = measure_record(torch, wl, pk, local, 0, seconds=args.sustained_seconds)
        sustained["what"] = f"the step of this line repeated for ~{args.sustained_seconds:g} s"

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return
    # second half of the metric: batch prefill ms, greedy vs retrieval order (same trace, fresh context)
    host_us, pred = wl.host_admission()
    prefill = {args.arm: {"ms": app_ms + attn_ms, "append_ms": app_ms, "attn_ms": attn_ms, "suffix_tokens": wl.T,
                          "hit_blocks": wl.hit_blocks, "attn_flops": wl.flops, "waves": len(wl.waves),
                          "predicted_prefix_docs": pred["predicted_prefix_docs"], "actual_prefix_docs": pred["actual_prefix_docs"],
                          "over_predicted_docs": pred["over_predicted_docs"], "stale_marks": pred["stale_marks"],
                          "prefill_saved": prefill_saved(cfg, wl.waves)}}
    if not args.skip_retrieval:
        del wl.host_inputs, wl.ws
        wr = Workload(cfg_sel, "retrieval", device, want_e2e=False, device_inputs=args.device_inputs, real_waves=args.real_waves)
        for _ in range(args.warmup):
            wr.step()
        ev = []
        timed(torch, lambda: wr.step(ev), args.steps, None)
        r_app = sum(e[0].elapsed_time(e[1]) for e in ev) / args.steps
        r_attn = sum(e[1].elapsed_time(e[2]) for e in ev) / args.steps
        prefill["retrieval"] = {"ms": r_app + r_attn, "append_ms": r_app, "attn_ms": r_attn, "suffix_tokens": wr.T,
                                "hit_blocks": wr.hit_blocks, "attn_flops": wr.flops, "waves": len(wr.waves),
                                "prefill_saved": prefill_saved(cfg, wr.waves)}
        prefill["ratio_measured"] = prefill[args.arm]["ms"] / prefill["retrieval"]["ms"]
        prefill["ratio_predicted_by_flops"] = wl.flops / wr.flops
        del wr
        if cfg.admission == "sequential" and not args.skip_per_request:
            # the honest per-request figure: every request admitted, launched (2 kernels) and released
            # on its own — launch-bound on this shape (one request is 5-15 us of tensor work)
            ws = Workload(cfg_sel, args.arm, device, want_e2e=False, device_inputs=True, sequential=True)
            for _ in range(args.warmup):
                ws.step()
            s_ms = timed(torch, ws.step, args.steps, None) / args.steps
            prefill["per_request_launches"] = {"ms_per_trace": s_ms, "launches": 3 * len(ws.waves), "attn_flops": ws.flops,
                                               "us_per_request": 1e3 * s_ms / len(ws.waves), "api": "cw_admit_batch(1) + cw_prefill_requests + cw_release_batch per request",
                                               "value_tflops": ws.flops / (s_ms * 1e-3) / 1e12}
            del ws

    if cfg.name.startswith("cfg1"):
        prefill["arms_cfg1"] = cfg1_four_arms(device)
    # the HBM target of cw_append_kv is judged on the concurrent configs 4 and 5 (waves with eviction); their
    # figures ride along on the default line (timing-only activations drawn on the device; parity at these shapes:
    # tests/test_gpu_full_size.py)
    other = None
    if world == 1 and args.config == 2 and not args.skip_configs and not args.device_inputs:
        other = {}
        if hasattr(wl, "host_inputs"):
            del wl.host_inputs, wl.ws
        wl.inputs = None
        torch.cuda.empty_cache()
        for cid in (4, 5):
            wo = Workload(cid, args.arm, device, want_e2e=False, device_inputs=True, real_waves=0)
            rec = measure_record(torch, wo, pk, local, 3, seconds=args.configs_seconds)
            rec["inputs"] = "device-drawn N(0,1) activations (timing only)"
            other[f"cfg{cid}"] = rec
            del wo
            torch.cuda.empty_cache()
    cpu = None
    if world == 1 or rank == 0:
        sample = OracleSample(cfg_sel, args.oracle_requests, args.oracle_rows)
        t = sample.run()
        desc = f"first {len(sample.reqs)} of {cfg.n_req} requests of {cfg.name}, sequential, greedy order, one pass" + \
               (f", first {sample.max_rows} suffix rows of each" if sample.max_rows else "")
        cpu = {"value": sample.flops / t / 1e12, "unit": UNIT, "cores": oracle_threads(), "kind": "oracle", "sample": desc,
               "seconds": t}

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "bf16",
            "data": "synthetic" + (" (timing-only activations drawn on the device)" if args.device_inputs else ""),
            "config": {"workload": f"BASELINE.json configs[{args.config - 1}] ({cfg.name})", "requests": cfg.n_req,
                       "prompt_tokens": cfg.n, "heads": f"{cfg.Hq}q/{cfg.Hkv}kv x {cfg.D}", "pool_blocks": cfg.NB,
                       "admission": f"one varlen wave per launch ({n_l} wave(s)), eager block registration",
                       "order": args.arm, "parallelism": "replicas only" if world > 1 else "1 GPU",
                       "inputs": ("tracegen activations (keyed by document prefix)" if not args.device_inputs else
                                  f"tracegen activations for the first {min(args.real_waves, n_l)} wave(s), device-drawn N(0,1) for the rest"),
                       "l2": "inputs larger than L2 (q,k,v,pool >> 126 MB per step); no explicit flush",
                       "adjacent_jaccard_mean": float(np.mean([tracegen.jaccard(a, b) for a, b in
                                                               zip(wl.trace.retrieval[:-1], wl.trace.retrieval[1:])]))},
            "pct_of_bf16_peak": 100.0 * value / world / pk["bf16"],
            "clocks": clk.summary(),
            "e2e": ({"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": wl.h2d // e2e_steps,
                     "d2h_bytes_per_step": wl.d2h // e2e_steps, "ms_per_step": ms_e2e, "steps": e2e_steps} if e2e_steps else None),
            "gpu_launches": launches,
            "host_us_per_request": {"value": host_us, "what": "cw_order + prompt assembly + cw_lookup + cw_observe + cw_release per request "
                                    "(one cw_admit_batch + cw_release_batch call per wave)", "paper": "66.6 us = order 22.2 + build 44.4 "
                                    "(Python middleware, PAPER.md:244-251 Table 8; other hardware, context only)"},
            "roofline": {"kernel": "prefill_attn_kernel", "bound": "tensor", "achieved": attn_tflops, "peak": pk["bf16"],
                         "unit": "TFLOP/s", "frac": attn_tflops / pk["bf16"], "traffic": traffic_from_profile(cfg.name, "prefill_attn_kernel"),
                         "window": "attention kernel (cw_attn_run), CUDA events on the launching stream; the schedule kernel runs on a side stream beside cw_append_kv, inside the append window",
                         "peak_source": pk["source"], "frac_of_sustained": attn_tflops / pk["bf16_sustained"],
                         "flops_per_step": wl.flops, "avg_ms": attn_ms / n_l, "launches_per_step": n_l},
            "sustained": sustained,
            "configs": other,
            "roofline_append_kv": {"kernel": "append_kv_kernel", "bound": "hbm", "achieved": app_gbs, "peak": pk["hbm"],
                                   "unit": "GB/s", "frac": app_gbs / pk["hbm"], "traffic": traffic_from_profile(cfg.name, "append_kv_kernel"),
                                   "bytes_per_step": append_bytes(cfg, wl.T), "avg_ms": app_ms / n_l},
            "batch_prefill": prefill,
            "cpu_baseline": cpu}
    print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()


def select_config(args):
    """--config N, with the variants --one-wave (cfg 4 with a pool that holds the whole batch) and
    --config 3 --k K --overlap P (one cell of the sweep)."""
    import dataclasses
    if args.config == 3:
        return tracegen.config3(args.k, args.overlap)
    cfg = tracegen.CONFIGS[args.config]
    if args.one_wave:
        nb = 1 << (cfg.n_req * cfg.blocks_per_req - 1).bit_length()
        cfg = dataclasses.replace(cfg, name=cfg.name + f"-onewave-NB{nb}", NB=nb, H=nb // cfg.blocks_per_req)
    return cfg


def cfg1_four_arms(device):
    """config 1 under retrieval order, greedy, brute force over l(O,T) (trie-predicted) and brute force
    over real hits (the exhaustive arm) — PAPER.md:195 does not say which objective its oracle ordering used."""
    import torch
    from itertools import permutations
    from paper_2606_19667_b200.engine import TraceRunner
    trace = tracegen.make_trace(tracegen.CONFIGS[1])
    cfg = trace.cfg
    out = {}
    for arm in ("retrieval", "greedy", "brute_force_l", "exhaustive"):
        run = TraceRunner(trace, "greedy" if arm == "brute_force_l" else arm, device=device)
        if arm == "brute_force_l":          # the library predicts, the harness enumerates: first maximiser of cw_predict
            def admit(r, run=run):
                D = trace.retrieval[r]
                best, best_l = list(D), -1
                for p in permutations(range(len(D))):
                    O = [D[i] for i in p]
                    l = run.ctx.cw_predict(O)
                    if list(p[l:]) == sorted(p[l:]) and l > best_l:
                        best, best_l = O, l
                tokens = tracegen.assemble_prompt(trace, r, best)
                req, table, c = run.ctx.cw_lookup(tokens)
                run.ctx.cw_observe(best)
                from paper_2606_19667_b200.engine import RequestRecord
                return req, RequestRecord(r, best, best_l, tokens, table, c, len(run.waves))
            run._admit = admit
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        recs = run.run(keep_outputs=False)
        e1.record()
        torch.cuda.synchronize()
        out[arm] = {"orders": [rec.order for rec in recs], "predicted_docs": [rec.depth for rec in recs],
                    "hit_blocks": sum(rec.n_cached // 16 for rec in recs),
                    "suffix_tokens": sum(cfg.n - rec.n_cached for rec in recs),
                    "attn_flops": sum(4 * cfg.Hq * cfg.D * (cfg.n * (cfg.n + 1) // 2 - rec.n_cached * (rec.n_cached + 1) // 2) for rec in recs),
                    "trace_ms_python_driven": e0.elapsed_time(e1)}
    return out


def run_sweep(args):
    """BASELINE.json configs[2]: adjacent-overlap x top-k sweep at the 8B shapes, both orderings; per cell: hit blocks,
    suffix tokens, attention flops and prefill ms (append + attention, one wave per launch).  Timing-only inputs."""
    import torch
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device; there is no CPU fallback")
    device = "cuda:0"
    cells = []
    for k in (3, 5, 10):
        for ov in (0, 30, 60, 90):
            cell = {"k": k, "overlap_pct": ov}
            for arm in ("retrieval", "greedy"):
                wl = Workload(tracegen.config3(k, ov), arm, device, want_e2e=False, device_inputs=True)
                for _ in range(max(3, args.warmup)):
                    wl.step()
                ev = []
                timed(torch, lambda: wl.step(ev), args.steps, None)
                app = sum(e[0].elapsed_time(e[1]) for e in ev) / args.steps
                att = sum(e[1].elapsed_time(e[2]) for e in ev) / args.steps
                cell[arm] = {"hit_blocks": wl.hit_blocks, "suffix_tokens": wl.T, "attn_flops": wl.flops, "waves": len(wl.waves),
                             "prefill_ms": app + att, "append_ms": app, "attn_ms": att,
                             "attn_tflops": wl.flops / (att * 1e-3) / 1e12}
                del wl
                torch.cuda.empty_cache()
            cell["flops_ratio"] = cell["greedy"]["attn_flops"] / cell["retrieval"]["attn_flops"]
            cell["ms_ratio"] = cell["greedy"]["prefill_ms"] / cell["retrieval"]["prefill_ms"]
            cells.append(cell)
            print(json.dumps(cell), flush=True)
    return cells


def run_mixed(args):
    """SURVEY.md 8(f) NEXT-4 (continuous batching): decode rows and prefill suffixes in the same varlen
    launch, 8B shapes.  Three launches are timed: (a) 512 single-token decode rows over 1024..8192-token contexts — bound by
    reading each context's K/V once (AI = g = 4 flop/B, far below the 263 flop/B ridge), reported against the HBM peak;
    (b) 64 prefill suffixes of 1072 tokens behind a 256-token cached prefix; (c) both in one launch."""
    import torch
    from paper_2606_19667_b200 import Context
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device; there is no CPU fallback")
    dev, pk = "cuda:0", peaks()
    Hq, Hkv, D = 32, 8, 128
    rng = np.random.default_rng(0)
    dec_n = rng.integers(1024, 8193, size=512)                 # tokens already in the pool per decode row
    pre_c, pre_s = np.full(64, 256), np.full(64, 1072)
    def build(cs, ss):
        ns = cs + ss
        nblk = -(-ns // 16)
        mb = int(nblk.max())
        tables = np.zeros((len(cs), mb), dtype=np.int32)
        o = 0
        for r, nb in enumerate(nblk):
            tables[r, :nb] = np.arange(o, o + nb)
            o += nb
        cu = np.zeros(len(cs) + 1, dtype=np.int32)
        cu[1:] = np.cumsum(ss)
        return dict(cs=cs, ss=ss, ns=ns, tables=tables, cu=cu, blocks=o, mb=mb)
    cases = {"decode_rows": build(dec_n, np.ones(512, dtype=np.int64)), "prefill_suffixes": build(pre_c, pre_s),
             "mixed": build(np.concatenate([pre_c, dec_n]), np.concatenate([pre_s, np.ones(512, dtype=np.int64)]))}
    NB = max(c["blocks"] for c in cases.values()) + 8
    ctx = Context(NB, Hq, Hkv, D, 4, rope_theta=5e5, max_position=int(max(c["ns"].max() for c in cases.values())), device=dev)
    g = torch.Generator(device=dev)
    g.manual_seed(0)
    ctx.k_pool.normal_(generator=g)
    ctx.v_pool.normal_(generator=g)
    for name, c in cases.items():
        B, T = len(c["cs"]), int(c["cu"][-1])
        q = torch.randn(T, Hq, D, device=dev, dtype=torch.bfloat16, generator=g)
        k = torch.randn(T, Hkv, D, device=dev, dtype=torch.bfloat16, generator=g)
        v = torch.randn(T, Hkv, D, device=dev, dtype=torch.bfloat16, generator=g)
        qr, out = torch.empty_like(q), torch.empty_like(q)
        d_cu, d_nc = torch.from_numpy(c["cu"]).to(dev), torch.from_numpy(c["cs"].astype(np.int32)).to(dev)
        d_t = torch.from_numpy(c["tables"]).to(dev)
        work = torch.empty(ctx.cw_attn_work_ints(B, T), dtype=torch.int32, device=dev)
        ctx.cw_append_kv(q, k, v, qr, d_cu, d_nc, d_t, c["mb"], B, T)
        fn = lambda: ctx.cw_prefill_attn(qr, out, d_cu, d_nc, d_t, c["mb"], B, T, int(c["ss"].max()), int(c["ns"].max()), work)
        for _ in range(max(3, args.warmup)):
            fn()
        ms = timed(torch, fn, args.steps, None) / args.steps
        flops = int(sum(4 * Hq * D * (int(n) * (int(n) + 1) // 2 - int(cc) * (int(cc) + 1) // 2) for n, cc in zip(c["ns"], c["cs"])))
        kv_bytes = int(sum(2 * int(n) * Hkv * D * 2 for n in c["ns"])) + 2 * T * Hq * D * 2      # K, V once + q in, o out
        line = {"case": name, "requests": B, "rows": T, "ms": ms, "attn_tflops": flops / ms / 1e9,
                "algorithmic_bytes": kv_bytes, "gbs": kv_bytes / ms / 1e6, "frac_of_hbm_peak": kv_bytes / ms / 1e6 / pk["hbm"],
                "frac_of_bf16_peak": flops / ms / 1e9 / pk["bf16"], "flop_per_byte": flops / kv_bytes,
                "bound": "hbm" if flops / kv_bytes < 263 else "tensor", "fallbacks": int(work[2])}
        print(json.dumps(line), flush=True)
        del q, k, v, qr, out


def run_length_sweep(args):
    """Item-length sweep of the attention kernel (short items pay the per-item cost): B cold prompts of L tokens
    each, B * L = 65 536 suffix rows in every case, 8B head shape, attention kernel only (cw_attn_run over a prepared item
    list), device-drawn activations.  One JSON line per length: ms, TFLOP/s over algorithmic flops, fraction of the peak."""
    import torch
    from paper_2606_19667_b200 import Context
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device; there is no CPU fallback")
    dev, pk = "cuda:0", peaks()
    Hq, Hkv, D, rows = 32, 8, 128, 65536
    g = torch.Generator(device=dev)
    g.manual_seed(0)
    for L in (64, 128, 256, 512, 1024, 2048, 4096, 8192):
        B = rows // L
        mb = L // 16
        ctx = Context(B * mb + 8, Hq, Hkv, D, 4, rope_theta=5e5, max_position=L, device=dev)
        tables = torch.arange(B * mb, dtype=torch.int32, device=dev).reshape(B, mb).contiguous()
        d_cu = torch.arange(0, rows + 1, L, dtype=torch.int32, device=dev)
        d_nc = torch.zeros(B, dtype=torch.int32, device=dev)
        q = torch.randn(rows, Hq, D, device=dev, dtype=torch.bfloat16, generator=g)
        k = torch.randn(rows, Hkv, D, device=dev, dtype=torch.bfloat16, generator=g)
        v = torch.randn(rows, Hkv, D, device=dev, dtype=torch.bfloat16, generator=g)
        qr, out = torch.empty_like(q), torch.empty_like(q)
        work = torch.empty(ctx.cw_attn_work_ints(B, rows), dtype=torch.int32, device=dev)
        ctx.cw_append_kv(q, k, v, qr, d_cu, d_nc, tables, mb, B, rows)

        def fn():      # the schedule kernel resets the claim counter; only the attention kernel is inside the events
            ctx.cw_attn_schedule(d_cu, d_nc, tables, mb, B, rows, L, L, work)
        ms = 0.0
        for i in range(max(3, args.warmup) + args.steps):
            fn()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            ctx.cw_attn_run(qr, out, tables, mb, B, rows, work)
            e1.record()
            torch.cuda.synchronize()
            if i >= max(3, args.warmup):
                ms += e0.elapsed_time(e1) / args.steps
        flops = B * 4 * Hq * D * (L * (L + 1) // 2)
        print(json.dumps({"prompt_tokens": L, "requests": B, "rows": rows, "items": int(work[3]), "attn_ms": ms,
                          "attn_tflops": flops / ms / 1e9, "frac_of_bf16_peak": flops / ms / 1e9 / pk["bf16"],
                          "us_per_item": 1e3 * ms * 148 / max(1, int(work[3]))}), flush=True)
        del q, k, v, qr, out, ctx


def run_layouts(args):
    """config 2's trace under the paper-literal prompt layout (instruction + [Document r: id] headers,
    180-220-token documents) against the block-aligned plain layout with the same retrieval lists:
    hit blocks, suffix tokens, attention flops and prefill ms (one wave, both kernels) per layout and ordering arm."""
    import dataclasses
    import torch
    from paper_2606_19667_b200.engine import TraceRunner
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device; there is no CPU fallback")
    dev = "cuda:0"
    base = tracegen.CONFIGS[2]
    layouts = {"plain-aligned-208": dataclasses.replace(base, name="cfg2-plain208", doc_len=208, admission="waves"),
               "literal-200+-20": dataclasses.replace(base, name="cfg2-literal", doc_len=200, doc_jitter=20, layout="literal",
                                                      admission="waves")}
    for lname, cfg in layouts.items():
        cfg = dataclasses.replace(cfg, H=cfg.NB // (-(-cfg.n // 16)))
        trace = tracegen.make_trace(cfg)
        for arm in ("retrieval", "greedy", "greedy_feedback"):
            run = TraceRunner(trace, arm, device=dev)
            waves = []
            run.prefill_wave = lambda wave, keep_outputs=True: waves.append(wave)      # host path only; the wave is timed below
            recs = run.run(compute=True, keep_outputs=False)
            assert len(waves) == 1
            wave = waves[0]
            ns = np.array([len(rec.tokens) for rec in recs])
            nc = np.array([rec.n_cached for rec in recs])
            flops = int(sum(4 * cfg.Hq * cfg.D * (int(n) * (int(n) + 1) // 2 - int(c) * (int(c) + 1) // 2) for n, c in zip(ns, nc)))
            # the wave was released by run(); re-admit nothing: replay the recorded descriptors (both kernels are idempotent)
            q, k, v = run.wave_inputs(wave)
            d_cu, d_nc, d_t, work = run.wave_descriptors(wave)
            qr, out = torch.empty_like(q), torch.empty_like(q)
            s = np.diff(wave.cu)
            def fn():
                run.ctx.cw_append_kv(q, k, v, qr, d_cu, d_nc, d_t, wave.max_blocks, wave.B, wave.T)
                run.ctx.cw_prefill_attn(qr, out, d_cu, d_nc, d_t, wave.max_blocks, wave.B, wave.T, int(s.max()),
                                        int((wave.nc + s).max()), work)
            for _ in range(max(3, args.warmup)):
                fn()
            ms = timed(torch, fn, args.steps, None) / args.steps
            print(json.dumps({"layout": lname, "arm": arm, "requests": len(recs), "prompt_tokens_mean": float(ns.mean()),
                              "hit_blocks": int(nc.sum()) // 16, "suffix_tokens": int((ns - nc).sum()), "attn_flops": flops,
                              "predicted_docs": int(sum(rec.depth for rec in recs)),
                              "matched_docs": int(sum(run.ctx.cw_matched_docs(tracegen.doc_segment_ends(trace, rec.order), rec.n_cached, len(rec.tokens)) for rec in recs)),
                              "prefill_ms": ms, "attn_tflops_incl_append": flops / ms / 1e9}), flush=True)
            del q, k, v, qr, out


def run_arms(args):
    """Ordering arms of the paper's Table 4 on the bench configuration: retrieval, sorted, recency,
    greedy (Algorithm 1), exhaustive.  One JSON line per arm with hit blocks, suffix tokens, attention flops, host admission
    time and prefill ms, then a summary line with the share of the exhaustive arm's gain that greedy reaches."""
    import torch
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device; there is no CPU fallback")
    device = "cuda:0"
    res = {}
    for arm in ("retrieval", "sorted", "recency", "greedy", "exhaustive"):
        wl = Workload(args.config, arm, device, want_e2e=False, device_inputs=True)
        for _ in range(max(3, args.warmup)):
            wl.step()
        ev = []
        ms_total = timed(torch, lambda: wl.step(ev), args.steps, None) / args.steps
        app = sum(e[0].elapsed_time(e[1]) for e in ev) / args.steps
        att = sum(e[1].elapsed_time(e[2]) for e in ev) / args.steps
        t0 = time.perf_counter()
        for _ in range(3):                                   # host admission alone (a1-a6 for all requests)
            wl.ctx.cw_reset()
            lo = 0
            for w in wl.waves:
                st, a = wl._admit(lo, w)
                wl.ctx.cw_release_batch(a["reqs"][:w.B])
                lo += w.B
        host_ms = (time.perf_counter() - t0) / 3 * 1e3
        res[arm] = {"arm": arm, "hit_blocks": wl.hit_blocks, "suffix_tokens": wl.T, "attn_flops": wl.flops,
                    "prefill_ms": app + att, "append_ms": app, "attn_ms": att, "step_ms": ms_total,
                    "host_admission_ms": host_ms, "host_us_per_request": 1e3 * host_ms / wl.cfg.n_req}
        print(json.dumps(res[arm]), flush=True)
        del wl
        torch.cuda.empty_cache()
    r, g, x = res["retrieval"], res["greedy"], res["exhaustive"]
    share = lambda key: (r[key] - g[key]) / (r[key] - x[key]) if r[key] != x[key] else None
    print(json.dumps({"summary": "greedy's share of the exhaustive arm's reduction vs retrieval order",
                      "in_attn_flops": share("attn_flops"), "in_prefill_ms": share("prefill_ms"),
                      "in_suffix_tokens": share("suffix_tokens"), "paper": "97.5 % of the oracle's TTFT reduction (PAPER.md:208)"}),
          flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=2, choices=[1, 2, 3, 4, 5])
    ap.add_argument("--k", type=int, default=5, help="--config 3: top-k of the sweep cell")
    ap.add_argument("--overlap", type=int, default=60, help="--config 3: adjacent overlap in percent")
    ap.add_argument("--arm", default="greedy", help="ordering arm of the timed workload (cacheweaver.h CW_ARM_*)")
    ap.add_argument("--one-wave", action="store_true", help="pool large enough for the whole batch (cfg 4 variant of SURVEY.md 8(d))")
    ap.add_argument("--real-waves", type=int, default=0, help="with --device-inputs: tracegen activations for the first N waves")
    ap.add_argument("--seconds", type=float, default=0.0, help="run the timed region for about this long (sustained figure)")
    ap.add_argument("--skip-per-request", action="store_true")
    ap.add_argument("--sustained-seconds", type=float, default=2.0, help="length of the extra sustained-clocks record (0 = none)")
    ap.add_argument("--skip-configs", action="store_true", help="no configs.cfg4 / configs.cfg5 records on the default line")
    ap.add_argument("--configs-seconds", type=float, default=1.0, help="timed length of each configs.* record")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--oracle-requests", type=int, default=None, help="requests in the oracle's bounded sample")
    ap.add_argument("--oracle-rows", type=int, default=None, help="suffix rows per request in the oracle's bounded sample")
    ap.add_argument("--e2e-steps", type=int, default=5)
    ap.add_argument("--skip-retrieval", action="store_true")
    ap.add_argument("--device-inputs", action="store_true", help="timing-only: draw q,k,v on the device (no e2e leg)")
    ap.add_argument("--layouts", action="store_true", help="NEXT-3: paper-literal prompt layout vs the aligned plain layout, one JSON line per layout and arm")
    ap.add_argument("--mixed", action="store_true", help="NEXT-4: decode rows / prefill suffixes / both in one varlen launch, one JSON line each")
    ap.add_argument("--length-sweep", action="store_true", help="attention kernel alone on cold prompts of 64..8192 tokens (65 536 rows each), one JSON line per length")
    ap.add_argument("--arms", action="store_true", help="ordering arms of the paper's Table 4 on --config, one JSON line per arm")
    ap.add_argument("--sweep", action="store_true", help="overlap x top-k sweep (BASELINE.json configs[2]), one JSON line per cell")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    if args.oracle_requests is None:
        args.oracle_requests = {1: 4, 2: 16 if args.impl == "ours" else 4, 3: 4, 4: 1, 5: 1}[args.config]
    if args.oracle_rows is None and args.config == 5:
        args.oracle_rows = 4096           # ~12 s instead of ~70 s for the whole 10 304-token prompt
    if args.length_sweep:
        run_length_sweep(args)
    elif args.layouts:
        run_layouts(args)
    elif args.mixed:
        run_mixed(args)
    elif args.arms:
        run_arms(args)
    elif args.sweep:
        run_sweep(args)
    elif args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
