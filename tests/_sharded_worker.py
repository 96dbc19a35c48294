"""worker of tests/test_sharded_cpu.py (run under torchrun, gloo): the exchange callback of nsgpu_run_sharded on
host buffers -- rank-ordered all-gather straight into the caller's memory, as the C library expects it."""
import ctypes as C
import os
import sys

import numpy as np
import torch.distributed as dist

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
from paper_2509_13307_b200 import nsgpu  # noqa: E402


def main():
    dist.init_process_group("gloo")
    rank, world = dist.get_rank(), dist.get_world_size()
    k, D = 7, 5                                            # 7 chains on 2 ranks: 4 + 3, one padding row
    per = (k + world - 1) // world
    first, count = nsgpu.shard_range(k, rank, world)
    send = np.full((per, D), -1.0, np.float32)
    for i in range(count):
        send[i] = 100.0 * (first + i) + np.arange(D)        # the row chain first + i produced
    recv = np.zeros((world * per, D), np.float32)
    fn = nsgpu.ALLGATHER_FN(nsgpu.torch_allgather(device=None))
    rc = fn(None, send.ctypes.data_as(C.c_void_p), recv.ctypes.data_as(C.c_void_p), send.nbytes, None)
    assert rc == 0
    for g in range(k):                                      # global chain g sits at row g on every rank
        np.testing.assert_array_equal(recv[g], 100.0 * g + np.arange(D))
    assert np.all(recv[k:] == -1.0)
    # the three-word counter exchange at the end of a run
    cnt = np.array([10 + rank, 20 + rank, rank, 0], np.uint64)
    allc = np.zeros(4 * world, np.uint64)
    assert fn(None, cnt.ctypes.data_as(C.c_void_p), allc.ctypes.data_as(C.c_void_p), cnt.nbytes, None) == 0
    assert list(allc[0::4]) == [10 + r for r in range(world)]
    dist.barrier()
    print(f"OK rank {rank}", flush=True)
    dist.destroy_process_group()


if __name__ == "__main__":
    main()
