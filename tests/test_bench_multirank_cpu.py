"""The N > 1 path of bench.py is "replicas only": no collective on the data path,
timings reduced with MAX over ranks, value = units of all ranks / that time.  Covered here with
world_size 2 on the gloo backend (CPU); the reference arm prints on rank 0 only."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import os, sys
sys.path.insert(0, {root!r})
import torch, torch.distributed as dist
import bench
dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
vals = bench.max_over_ranks([1.0 + rank, 10.0 - rank], torch, dist, "cpu")
assert vals == [float(world), 10.0], vals
v = bench.aggregate_value(2e12, vals[0], world)      # 2 TOP per step per rank, `world` ms
assert abs(v - world * 2e12 / (world * 1e-3) / 1e12) < 1e-9
dist.barrier()
dist.destroy_process_group()
sys.stdout.write("rank%dok\n" % rank)
"""


def _torchrun(args, timeout=300):
    env = dict(os.environ, MASTER_ADDR="127.0.0.1")
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
           "--master-addr", "127.0.0.1", "--master-port", "29533"] + args
    return subprocess.run(cmd, capture_output=True, text=True, timeout=timeout, env=env, cwd=ROOT)


def test_max_over_ranks_and_aggregate_world2(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER.format(root=ROOT))
    r = _torchrun([str(script)])
    assert r.returncode == 0, r.stdout + r.stderr
    assert r.stdout.count("ok") == 2 and "rank0" in r.stdout and "rank1" in r.stdout, r.stdout


def test_reference_arm_prints_once_under_torchrun():
    """`bench.py --impl reference` under torchrun: rank 0 alone runs the oracle and prints one JSON
    line with the contract's keys; the other rank exits 0 without work."""
    r = _torchrun([os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1", "--warmup", "0",
                   "--workload", "tiny"])
    assert r.returncode == 0, r.stdout + r.stderr
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1, r.stdout
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["gpu_launches"] == 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["e2e"]["h2d_bytes_per_step"] == 0
    assert d["value"] > 0 and d["unit"] == "TOPS"
