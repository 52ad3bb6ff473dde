"""bench.py's N > 1 logic (replicas only) on CPU with gloo, world_size 2:
per-rank inputs differ, the step time is the max over ranks, the value aggregates all ranks,
and only rank 0 of the reference arm does work."""
import json
import os
import subprocess
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import os, sys, json
sys.path.insert(0, %r)
import numpy as np, torch, torch.distributed as dist
import workloads as w
import bench                                                       # the functions under test are bench.py's own
dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
cfg = w.get_config(1)
m = w.random_unit_vectors(bench.rank_seed(cfg, rank), cfg.n)       # per-rank replica input
ms_local = 3.0 + 2.0 * rank                                        # pretend device times
ms = bench.max_over_ranks(ms_local, dist, device="cpu")
chk = torch.tensor([float(m.sum())], dtype=torch.float64)
gathered = [torch.zeros(1, dtype=torch.float64) for _ in range(world)]
dist.all_gather(gathered, chk)
dist.barrier()
if rank == 0:
    print(json.dumps({"ms": ms, "value": bench.job_value(world, cfg.ncell, ms),
                      "sums": [g.item() for g in gathered]}))
dist.destroy_process_group()
""" % ROOT


def test_replica_aggregation_gloo_world2(tmp_path):
    """bench.py's own rank_seed / max_over_ranks / job_value under a world_size-2 gloo group."""
    script = tmp_path / "worker.py"
    script.write_text(WORKER)
    env = dict(os.environ, MASTER_ADDR="127.0.0.1")
    r = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node=2",
                        "--master-addr", "127.0.0.1", "--master-port", "29613", str(script)],
                       capture_output=True, text=True, env=env, timeout=300)
    assert r.returncode == 0, r.stderr[-2000:]
    line = [l for l in r.stdout.splitlines() if l.startswith("{")][-1]
    out = json.loads(line)
    assert out["ms"] == 5.0                                  # max over ranks, not the mean
    assert out["value"] == pytest.approx(2 * 16 * 16 * 2 / 5e-3)
    assert out["sums"][0] != out["sums"][1]                  # independent replicas


def test_rank_helpers_single_process():
    sys.path.insert(0, ROOT)
    import bench
    import workloads as w
    cfg = w.get_config(4)
    assert bench.rank_seed(cfg, 0) == cfg.seed and bench.rank_seed(cfg, 3) == cfg.seed + 3000
    assert bench.max_over_ranks(2.5) == 2.5                  # no process group: the local time
    assert bench.job_value(8, 1000, 2.0) == 8 * 1000 / 2e-3


def test_byte_model_matches_design():
    sys.path.insert(0, ROOT)
    import bench
    k, total = bench.byte_model((512, 512, 128), 4)
    n = 512 * 512 * 128
    # 93*s B/cell up to the (nz+1)/nz and (n+1)^3 corrections (< 1.5 %)
    assert 93 * 4 * n <= total <= 1.015 * 93 * 4 * n
    assert k["S6"] == 9 * n * 4
    k1, t1 = bench.byte_model((128, 32, 1), 8)
    assert k1["S1"] == 3 * 4096 * 8 + 3 * 4096 * 16


def test_reference_arm_other_ranks_do_no_work():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2"],
                       capture_output=True, text=True, env=env, timeout=120)
    assert r.returncode == 0 and r.stdout.strip() == ""
