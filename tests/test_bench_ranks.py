"""bench.py's multi-rank plumbing on CPU: two gloo ranks (the path shards as independent replicas):
max-over-ranks timing, sum-over-ranks counts, and the reference arm printing one line from rank 0 only."""
from __future__ import annotations

import json
import os
import socket
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import os, sys
sys.path.insert(0, os.environ["ECPUSH_ROOT"])
import torch.distributed as dist
import bench
dist.init_process_group("gloo")
rank, world, local = bench.dist_env()
assert world == 2 and dist.get_rank() == rank
mx = bench.max_over_ranks([1.0 + rank, 5.0 - 3 * rank], world, backend_device="cpu")
sm = bench.sum_over_ranks(10.0 * (rank + 1), world, backend_device="cpu")
assert mx == [2.0, 5.0], mx
assert sm == 30.0, sm
dist.barrier()
dist.destroy_process_group()
print(f"rank {rank} ok")
"""


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def test_two_gloo_ranks_reduce_times_and_counts(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER)
    env = dict(os.environ, ECPUSH_ROOT=ROOT)
    out = subprocess.run(
        [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node=2", "--master-addr", "127.0.0.1",
         "--master-port", str(_free_port()), str(script)], env=env, capture_output=True, text=True, timeout=300)
    assert out.returncode == 0, out.stdout + out.stderr
    assert "rank 0 ok" in out.stdout and "rank 1 ok" in out.stdout


def test_reference_arm_prints_one_line_from_rank_zero_only():
    """`bench.py --impl reference` under two ranks: rank 0 times the oracle on a bounded sample, rank 1 exits 0
    without work (tier framing, measurement section)."""
    base = [sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--config", "0", "--steps", "1",
            "--warmup", "0", "--gpus", "2"]
    r1 = subprocess.run(base, env=dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1"), capture_output=True,
                        text=True, timeout=300)
    assert r1.returncode == 0 and r1.stdout.strip() == ""
    r0 = subprocess.run(base, env=dict(os.environ, RANK="0", WORLD_SIZE="2", LOCAL_RANK="0"), capture_output=True,
                        text=True, timeout=300)
    assert r0.returncode == 0, r0.stderr
    line = json.loads(r0.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["cpu_baseline"]["kind"] == "oracle"
    assert line["value"] > 0 and line["unit"] == "particles/s" and line["higher_is_better"] is True
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["e2e"]["d2h_bytes_per_step"] == 0
