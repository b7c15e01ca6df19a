"""Host-side logic of bench.py under world_size 2 (gloo, CPU): the cross-rank reductions of the replicas-only
multi-GPU mode and the reference arm's rank protocol (rank 0 alone runs and prints)."""
from __future__ import annotations

import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

_WORKER = r"""
import os, sys, json
sys.path.insert(0, {root!r})
import torch.distributed as dist
import bench
rank, world = int(os.environ["RANK"]), int(os.environ["WORLD_SIZE"])
dist.init_process_group("gloo")
mx = bench.reduce_over_ranks(10.0 + rank, "max", world, device="cpu")
sm = bench.reduce_over_ranks(100.0 * (rank + 1), "sum", world, device="cpu")
seeds = [bench.replica_seed(4, r) for r in range(world)]
dist.barrier()
dist.destroy_process_group()
if rank == 0:
    print(json.dumps({{"max": mx, "sum": sm, "seeds": seeds}}), flush=True)
"""


def _torchrun(args, timeout=600):
    env = dict(os.environ, OMP_NUM_THREADS="2")
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
           "--master-addr", "127.0.0.1", "--master-port", "29617"] + args
    return subprocess.run(cmd, cwd=ROOT, env=env, capture_output=True, text=True, timeout=timeout)


def test_cross_rank_reductions_gloo(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(_WORKER.format(root=ROOT))
    res = _torchrun([str(script)])
    assert res.returncode == 0, res.stderr[-2000:]
    lines = [l for l in res.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    out = json.loads(lines[0])
    assert out["max"] == 11.0 and out["sum"] == 300.0
    assert out["seeds"][1] == out["seeds"][0] + 1          # replicas differ by their seed only


def test_reference_arm_two_ranks_prints_one_line():
    res = _torchrun(["bench.py", "--impl", "reference", "--gpus", "2", "--steps", "1", "--warmup", "0"])
    assert res.returncode == 0, res.stderr[-2000:]
    lines = [l for l in res.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1, res.stdout
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["value"] > 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["gpu_launches"] == 0
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["e2e"]["d2h_bytes_per_step"] == 0


def test_committed_dram_profile_is_of_the_kernel_sources_as_they_are():
    """bench.py reports roofline.traffic from profiles/r3_k_step_dram.txt only while that capture is of the CUDA
    sources at HEAD (the file carries their hash): a stale profile would silently turn the field into null."""
    import bench
    assert bench._profiled_traffic(4096, 50) is not None, (
        "profiles/r3_k_step_dram.txt is not of the kernel sources as they are (hash %s): re-capture it" % bench.kernel_source_hash())
    assert bench._profiled_traffic(4096, 49) is None
