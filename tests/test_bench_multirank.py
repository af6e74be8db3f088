"""N > 1 path of bench.py on CPU (gloo, world_size 2): the path does not shard ("replicas only"), so the
only inter-rank logic is the MAX over ranks of the timed region and the sum of the replicas' work; the reference arm must
print on rank 0 only."""
import json
import os
import subprocess
import sys

import pytest

from conftest import ROOT

WORKER = r'''
import os, sys, json
sys.path.insert(0, os.environ["CW_ROOT"])
import torch, torch.distributed as dist
import bench
dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
ms = bench.max_over_ranks(10.0 + 5.0 * rank, dist, "cpu")          # rank 1 is the slow one
val = bench.aggregate_value(1e12, ms, world)
dist.barrier()
open(os.path.join(os.environ["CW_OUT"], f"rank{rank}.json"), "w").write(json.dumps({"rank": rank, "ms": ms, "value": val}))
dist.destroy_process_group()
'''


def _torchrun(args, env_extra=None, timeout=240):
    env = dict(os.environ, CW_ROOT=ROOT, MASTER_ADDR="127.0.0.1", OMP_NUM_THREADS="2")
    env.update(env_extra or {})
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr", "127.0.0.1",
           "--master-port", "29533"] + args
    return subprocess.run(cmd, capture_output=True, text=True, env=env, timeout=timeout, cwd=ROOT)


def test_max_over_ranks_and_replica_sum(tmp_path):
    w = tmp_path / "worker.py"
    w.write_text(WORKER)
    r = _torchrun([str(w)], {"CW_OUT": str(tmp_path)})
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [json.loads((tmp_path / f"rank{k}.json").read_text()) for k in range(2)]
    assert sorted(l["rank"] for l in lines) == [0, 1]
    for l in lines:
        assert l["ms"] == 15.0                                       # max over ranks, on every rank
        assert l["value"] == pytest.approx(2 * 1e12 / 15e-3 / 1e12)  # 2 replicas' units / max time


def test_reference_arm_prints_on_rank_zero_only():
    r = _torchrun(["bench.py", "--impl", "reference", "--gpus", "2", "--steps", "1", "--warmup", "0", "--config", "1"])
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [json.loads(l) for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    d = lines[0]
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["cpu_baseline"]["kind"] == "oracle"
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["value"] > 0 and d["unit"] == "TFLOP/s"


def test_oracle_sample_with_row_bound_counts_the_rows_it_computes():
    """bench.py's bounded oracle sample (`--oracle-rows`, default for config 5): the flops it reports are those of the
    rows the oracle really computes — a prompt cut after n_cached + max_rows tokens — and the full sample is unchanged."""
    sys.path.insert(0, ROOT)
    import bench
    import tracegen
    cfg = tracegen.CONFIGS[1]
    full = bench.OracleSample(1, 2)
    cut = bench.OracleSample(1, 2, max_rows=40)
    ncs = [rr.n_cached for rr in full.dry.requests]
    assert full.flops == bench.attention_flops(cfg, ncs)
    want = sum(4 * cfg.Hq * cfg.D * sum(p + 1 for p in range(c, min(cfg.n, c + 40))) for c in ncs)
    assert cut.flops == want and cut.flops < full.flops
    assert cut.run() > 0 and full.run() > 0
