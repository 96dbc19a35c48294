"""BASELINE.json configs[4]: nested-sampling model comparison, w0waCDM (39-D) vs its LambdaCDM restriction
(37-D), on the synthetic cosmic-shear likelihood (c3a weights; mock data from the LambdaCDM truth).

    python -m paper_2509_13307_b200.examples.model_comparison [--n-live 1000] [--n-delete 500] [--seeds 1]
                                                              [--shape c4|paper-interp|paper] [--batched] [--ranks N]

`--batched` (with --seeds R > 1): the R seeds of a model run as ONE nsgpu_run_multi call that shares every likelihood
batch between them (each result is what the single run returns, bit for bit), the two models on two host threads.

`--shape paper-interp` / `paper` run the same comparison on the paper-shape likelihood (10 bins, 55 spectra,
1025 quadrature nodes; emulator on 103 z nodes + linear interpolation, or on all 1025: PAPER.md L353, L359).

Multi-GPU: `--ranks N` (re-executes itself under `python -m torch.distributed.run --nnodes=1
--nproc-per-node N --master-addr 127.0.0.1`), or launch it under torchrun yourself; every rank holds the live set, evolves its share of
the 500 chains per iteration and all-gathers the new points over NCCL (`Context.run_sharded`); rank 0 prints.

Prints one JSON line per run and a summary with log Z +- error per model, the log Bayes factor, total
likelihood evaluations and wall time.  The mock data vector is produced by the CUDA path itself at the
fiducial point (the product never calls the oracle).
"""
import argparse
import json
import math
import os
import threading
import time

import numpy as np
import torch

from paper_2509_13307_b200 import nsgpu, workloads as W


def _ranks():
    """(rank, world, device) from the torchrun environment; a plain `python -m ...` is one rank on cuda:0"""
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if world == 1:
        return 0, 1, 0
    import torch.distributed as dist
    dev = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(dev)
    dist.init_process_group("nccl")
    return dist.get_rank(), world, dev


def _spawn(n):
    """re-execute this module with n ranks (one per GPU) on this node"""
    import socket
    import subprocess
    import sys
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={n}", "--master-addr", "127.0.0.1",
           "--master-port", str(port), "-m", "paper_2509_13307_b200.examples.model_comparison"] + sys.argv[1:]
    return subprocess.call(cmd)


def _mock_data(wl_w0wa, device=0):
    """d = model_w0wa(theta_0 with w0 = -1, wa = 0) + L eps, shared by both models."""
    n = wl_w0wa.n_data
    wl_w0wa.data, wl_w0wa.chol = np.zeros(n), np.eye(n)
    with nsgpu.Context(wl_w0wa, max_batch=8, device=device) as c0:
        u0 = torch.as_tensor(wl_w0wa.u_fid[None].astype(np.float32), device=f"cuda:{device}")
        m0 = c0.theory_batch(c0.prior_transform(u0)).cpu().numpy()[0]
    wl_w0wa.seed = 1004
    W.attach_data(wl_w0wa, m0, noise=True)
    return wl_w0wa


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--n-live", type=int, default=1000)
    ap.add_argument("--n-delete", type=int, default=500)
    ap.add_argument("--seeds", type=int, default=1)
    ap.add_argument("--stop-frac", type=float, default=1e-3)
    ap.add_argument("--max-iter", type=int, default=100000)
    ap.add_argument("--shape", default="c4", choices=["c4", "paper-interp", "paper"])
    ap.add_argument("--sequential", action="store_true", help="one run after the other")
    ap.add_argument("--concurrent", type=int, default=4, help="runs in flight on one GPU (models x seeds; default 4)")
    ap.add_argument("--ctx-flags", type=int, default=0, help="extra nsgpu_create flags, e.g. 128 = NSGPU_NO_PDL (plain stream ordering)")
    ap.add_argument("--batched", action="store_true", help="all seeds of a model in one nsgpu_run_multi call (shared likelihood batches)")
    ap.add_argument("--ranks", type=int, default=1, help="GPUs: start this many ranks under torch.distributed.run (sharded runs)")
    ap.add_argument("--print-shards", action="store_true",
                    help="print which chains each rank would evolve (nsgpu_shard_range) and exit: needs no GPU")
    args = ap.parse_args()
    if args.ranks > 1 and "WORLD_SIZE" not in os.environ:
        raise SystemExit(_spawn(args.ranks))
    if args.print_shards:
        world, rank = int(os.environ.get("WORLD_SIZE", "1")), int(os.environ.get("RANK", "0"))
        first, count = nsgpu.shard_range(args.n_delete, rank, world)
        print(json.dumps({"rank": rank, "world": world, "chains": [first, first + count], "of": args.n_delete}), flush=True)
        return
    rank, world, dev = _ranks()
    if world > 1 and rank == 0:
        for r in range(world):
            first, count = nsgpu.shard_range(args.n_delete, r, world)
            print(json.dumps({"rank": r, "chains": [first, first + count], "of": args.n_delete}), flush=True)
    if args.shape == "c4":
        full, rest = _mock_data(W.c3a(), dev), W.c4_lcdm()
    else:
        interp = args.shape == "paper-interp"
        full, rest = _mock_data(W.c5(interp, w0wa=True), dev), W.c5(interp, w0wa=False)
    rest.data, rest.chol = full.data, full.chol
    out = {"w0waCDM": [], "LCDM": []}
    lock = threading.Lock()

    def run_model(name, wl, seeds):
        torch.cuda.set_device(dev)
        batched = args.batched and world == 1 and len(seeds) > 1
        mb = max(args.n_live, args.n_delete * len(seeds)) if batched else args.n_live
        with nsgpu.Context(wl, max_batch=mb, device=dev, mlp=nsgpu.MLP_AUTO | args.ctx_flags) as ctx:
            if batched:
                rs = ctx.run_multi(args.n_live, args.n_delete, 5 * wl.D, seeds, stop_frac=args.stop_frac, max_iter=args.max_iter,
                                   return_samples=False)
                for r in rs:
                    r["model"], r["D"], r["n_gpus"], r["batched_with"] = name, wl.D, world, len(seeds)
                    with lock:
                        print(json.dumps(r), flush=True)
                        out[name].append(r)
                return
            for seed in seeds:
                kw = dict(stop_frac=args.stop_frac, max_iter=args.max_iter, seed=seed, return_samples=False)
                if world == 1:
                    r = ctx.run(args.n_live, args.n_delete, 5 * wl.D, **kw)
                else:
                    r = ctx.run_sharded(args.n_live, args.n_delete, 5 * wl.D, rank=rank, world=world, **kw)
                r["model"], r["D"], r["seed"], r["n_gpus"] = name, wl.D, seed, world
                with lock:
                    if rank == 0:
                        print(json.dumps(r), flush=True)
                    out[name].append(r)

    models = (("w0waCDM", full), ("LCDM", rest))
    all_seeds = list(range(1, args.seeds + 1))
    t_all = time.perf_counter()
    n_conc = 1 if (world > 1 or args.sequential) else max(1, args.concurrent)
    if n_conc > 1:
        # The runs are independent and each keeps the GPU only partly busy (batches of <= n_delete proposals, fewer
        # as the chains of an iteration finish): one host thread and one context per worker, each nsgpu_run on its
        # context's own stream, so their kernels share the SMs.  Workers = models x groups of seeds.
        per_model = 1 if args.batched else max(1, min(len(all_seeds), n_conc // 2))
        jobs = [(name, wl, all_seeds[g::per_model]) for name, wl in models for g in range(per_model)]
        threads = [threading.Thread(target=run_model, args=j) for j in jobs]
        for t in threads:
            t.start()
        for t in threads:
            t.join()
        for v in out.values():
            v.sort(key=lambda r: r["seed"])
    else:
        for name, wl in models:
            run_model(name, wl, all_seeds)
    t_all = time.perf_counter() - t_all
    if rank != 0:
        return
    z = {k: np.mean([r["logZ"] for r in v]) for k, v in out.items()}
    e = {k: math.sqrt(np.mean([r["logZ_err"] ** 2 for r in v]) / len(v)) for k, v in out.items()}
    print(json.dumps({"shape": args.shape, "summary": {k: {"logZ": z[k], "err": e[k], "evals": int(np.mean([r["n_like_evals"] for r in v])),
                                       "seconds": float(np.mean([r["seconds"] for r in v])),
                                       "iterations": int(np.mean([r["n_iter"] for r in v]))} for k, v in out.items()},
                      "wall_seconds_all_runs": t_all, "concurrent_runs": n_conc if n_conc == 1 else len(jobs),
                      "logB_LCDM_over_w0wa": z["LCDM"] - z["w0waCDM"],
                      "logB_err": math.hypot(e["LCDM"], e["w0waCDM"])}))


if __name__ == "__main__":
    main()
