"""The N>1 host logic on CPU (gloo, world_size 2): row partition covers the grid exactly once, the
max-over-ranks reduction bench.py reports, and `--impl reference` printing on rank 0 only."""
import json
import os
import subprocess
import sys

import numpy as np

import gf_workloads as W

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import os, sys, json
sys.path.insert(0, %r)
import torch, torch.distributed as dist
import bench, gf_workloads as W
dist.init_process_group("gloo")
rank, local, world = bench.dist_env()
cfg = bench.workload_for("cfg3_production", world)
first, rows = W.row_partition(cfg["n_im_global"], world, rank)
# the slowest rank's time is the job's time
t = bench.max_over_ranks(10.0 + 5.0 * rank, world)
got = [None] * world
dist.all_gather_object(got, (first, rows))
dist.barrier()
if rank == 0:
    print(json.dumps({"world": world, "parts": got, "tmax": t, "rows_global": cfg["n_im_global"]}))
dist.destroy_process_group()
""" % ROOT


def test_row_partition_is_exact_cover():
    for n_rows in (1, 7, 256, 2048, 4097):
        for world in (1, 2, 3, 8):
            seen = np.zeros(n_rows, dtype=int)
            for r in range(world):
                first, n = W.row_partition(n_rows, world, r)
                seen[first:first + n] += 1
            assert (seen == 1).all()
            sizes = [W.row_partition(n_rows, world, r)[1] for r in range(world)]
            assert max(sizes) - min(sizes) <= 1


def test_world_size_2_gloo(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER)
    env = dict(os.environ, MASTER_ADDR="127.0.0.1")
    out = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node=2",
                          "--master-addr", "127.0.0.1", "--master-port", "29617", str(script)],
                         capture_output=True, text=True, env=env, timeout=300)
    assert out.returncode == 0, out.stderr[-2000:]
    line = [l for l in out.stdout.splitlines() if l.startswith("{")][-1]
    res = json.loads(line)
    assert res["world"] == 2 and res["rows_global"] == 4096
    assert res["parts"] == [[0, 2048], [2048, 2048]]      # weak scaling: 2048 rows per rank, no overlap
    assert res["tmax"] == 15.0


def test_reference_arm_prints_on_rank0_only():
    env = dict(os.environ, RANK="1", LOCAL_RANK="1", WORLD_SIZE="2")
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2"],
                         capture_output=True, text=True, env=env, timeout=300)
    assert out.returncode == 0 and out.stdout.strip() == ""
