"""-m gpu: nsgpu_run_sharded gives every rank the result of nsgpu_run, bit for bit, whatever the number of ranks
(the Philox streams are keyed by the global chain index and the per-theta arithmetic of the likelihood does not
depend on the batch it sits in).  Only one GPU is available: the ranks are THREADS of this process, each with its
own context on cuda:0, and the all-gather is a host-side rendezvous (a barrier and device-to-device copies) -- no
kernel ever waits for another.  This checks the sharding logic, not performance."""
import threading

import numpy as np
import pytest

from paper_2509_13307_b200 import nsgpu
from tests.util import workload

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")


def _run_threads(wl, world, opts):
    barrier = threading.Barrier(world)
    parts = [None] * world
    results = [None] * world
    errors = []

    def make_cb(r):
        def cb(user, send, recv, nbytes, stream):
            try:
                s = torch.as_tensor(nsgpu._RawBuffer(send, nbytes, True), device="cuda:0")
                parts[r] = s.clone()
                torch.cuda.synchronize()
                barrier.wait(timeout=120)
                out = torch.as_tensor(nsgpu._RawBuffer(recv, nbytes * world, True), device="cuda:0")
                out.copy_(torch.cat(parts))
                torch.cuda.synchronize()
                barrier.wait(timeout=120)
                return 0
            except Exception as e:      # noqa: BLE001
                errors.append(repr(e))
                barrier.abort()
                return 1
        return cb

    def worker(r):
        try:
            with nsgpu.Context(wl, max_batch=opts["n_live"]) as ctx:
                results[r] = ctx.run_sharded(rank=r, world=world, allgather=make_cb(r), return_samples=(r == 0), **opts)
        except Exception as e:          # noqa: BLE001
            errors.append(repr(e))
            barrier.abort()

    threads = [threading.Thread(target=worker, args=(r,)) for r in range(world)]
    for t in threads:
        t.start()
    for t in threads:
        t.join(timeout=600)
    assert not errors, errors
    return results


@pytest.mark.parametrize("name,opts,world", [
    ("identity", dict(n_live=200, n_delete=100, n_steps=30, seed=3), 2),
    ("identity", dict(n_live=200, n_delete=100, n_steps=30, seed=3), 3),      # 34 + 34 + 32 chains
    ("tiny_shear", dict(n_live=96, n_delete=48, n_steps=20, seed=5, stop_frac=1e-2), 2),
])
def test_sharded_run_equals_single_gpu_run(name, opts, world):
    wl = workload(name)
    with nsgpu.Context(wl, max_batch=opts["n_live"]) as ctx:
        ref = ctx.run(**opts)
    res = _run_threads(wl, world, opts)
    for r in res:
        for key in ("logZ", "logZ_err", "H", "n_iter", "n_dead", "n_like_evals", "n_failed_moves", "converged"):
            assert r[key] == ref[key], (key, r[key], ref[key])
    np.testing.assert_array_equal(res[0]["logL"], ref["logL"])
    np.testing.assert_array_equal(res[0]["theta"], ref["theta"])
    np.testing.assert_array_equal(res[0]["logw"], ref["logw"])


def test_nccl_allgather_callback_on_device_buffers():
    """the default exchange (torch.distributed all_gather_into_tensor, NCCL) straight on raw device pointers, as
    nsgpu_run_sharded calls it -- a one-rank group is all one GPU allows"""
    import ctypes as C
    import os
    import torch.distributed as dist
    os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
    os.environ.setdefault("MASTER_PORT", "29631")
    dist.init_process_group("nccl", rank=0, world_size=1)
    try:
        send = torch.arange(1000, dtype=torch.float32, device="cuda:0") * 0.5
        recv = torch.zeros(1000, dtype=torch.float32, device="cuda:0")
        fn = nsgpu.ALLGATHER_FN(nsgpu.torch_allgather(device=0))
        rc = fn(None, C.c_void_p(send.data_ptr()), C.c_void_p(recv.data_ptr()), send.numel() * 4, None)
        assert rc == 0
        assert torch.equal(send, recv)
    finally:
        dist.destroy_process_group()
