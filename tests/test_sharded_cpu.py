"""-m "not gpu": host side of multi-GPU nested sampling: the chain partition and the
exchange callback, world_size 2 on gloo."""
import os
import subprocess
import sys

from paper_2509_13307_b200 import nsgpu

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_shard_range_is_a_partition_in_rank_order():
    for k in (0, 1, 7, 500, 501):
        for world in (1, 2, 3, 8):
            per = (k + world - 1) // world
            nxt = 0
            for r in range(world):
                first, count = nsgpu.shard_range(k, r, world)
                assert 0 <= count <= per
                if count:
                    assert first == nxt == r * per        # contiguous blocks: global chain g = r * per + i
                    nxt = first + count
            assert nxt == k


def test_allgather_callback_two_ranks_gloo():
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr",
           "127.0.0.1", "--master-port", "29621", os.path.join(ROOT, "tests", "_sharded_worker.py")]
    out = subprocess.run(cmd, cwd=ROOT, capture_output=True, text=True, timeout=300)
    assert out.returncode == 0, out.stderr[-3000:]
    assert "OK rank 0" in out.stdout and "OK rank 1" in out.stdout


def test_model_comparison_ranks_flag_starts_the_ranks_and_shards_the_chains():
    """`model_comparison --ranks N` re-executes itself under torch.distributed.run; every rank takes the contiguous block of
    chains nsgpu_shard_range gives it.  `--print-shards` stops before any GPU work, so this runs on the CPU."""
    import json, os, subprocess, sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    env = {k: v for k, v in os.environ.items() if k not in ("RANK", "WORLD_SIZE", "LOCAL_RANK", "MASTER_ADDR", "MASTER_PORT")}
    out = subprocess.run([sys.executable, "-m", "paper_2509_13307_b200.examples.model_comparison", "--ranks", "3", "--n-delete", "500",
                          "--print-shards"], cwd=root, capture_output=True, text=True, timeout=300, env=env)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = sorted((json.loads(l) for l in out.stdout.splitlines() if l.startswith("{")), key=lambda d: d["rank"])
    assert [d["rank"] for d in lines] == [0, 1, 2] and all(d["world"] == 3 for d in lines)
    assert [d["chains"] for d in lines] == [[0, 167], [167, 334], [334, 500]]
