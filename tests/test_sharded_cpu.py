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
