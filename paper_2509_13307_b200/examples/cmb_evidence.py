"""The paper's CMB run in shape (Table 2 row "CMB"): evidence of the 6-parameter model
under the cosmic-variance TT likelihood, nested sampling with 1000 live points of which 500 are evolved in parallel.

    python -m paper_2509_13307_b200.examples.cmb_evidence [--seeds S] [--sequential]

Synthetic stand-ins (no trained emulator or Planck best-fit mock in this repo): seeded random-weight TT emulator
6 -> 4 x 512 -> 2507, observed spectrum = a cosmic-variance draw around the model at the fiducial point
(`workloads.cmb_tt`, `attach_cmb_tt_data`).  The paper quotes 12 s on one L4 in fp64 for its run (context, not a
like-for-like comparison).  Prints one JSON line per run and a summary line; with several seeds the runs share the
GPU (one host thread and one context each, see model_comparison.py).
"""
import argparse
import json
import math
import threading
import time

import numpy as np
import torch

from paper_2509_13307_b200 import nsgpu, workloads as W


def _mock_data(wl, device=0):
    """C_l at the fiducial point from the GPU path itself, then a chi^2_{2l+1} draw per multipole."""
    wl.data, wl.chol = np.ones(wl.n_data), None
    with nsgpu.Context(wl, max_batch=8, device=device) as c0:
        u0 = torch.as_tensor(wl.u_fid[None].astype(np.float32), device=f"cuda:{device}")
        m0 = c0.theory_batch(c0.prior_transform(u0)).cpu().numpy()[0]
    return W.attach_cmb_tt_data(wl, m0, noise=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--n-live", type=int, default=1000)
    ap.add_argument("--n-delete", type=int, default=500)
    ap.add_argument("--seeds", type=int, default=1)
    ap.add_argument("--stop-frac", type=float, default=1e-3)
    ap.add_argument("--max-iter", type=int, default=100000)
    ap.add_argument("--sequential", action="store_true", help="one run after the other")
    ap.add_argument("--ctx-flags", type=int, default=0, help="extra nsgpu_create flags, e.g. 128 = NSGPU_NO_PDL")
    args = ap.parse_args()
    wl = _mock_data(W.cmb_tt())
    runs, lock = [], threading.Lock()

    def work(seeds):
        torch.cuda.set_device(0)
        with nsgpu.Context(wl, max_batch=args.n_live, mlp=nsgpu.MLP_AUTO | args.ctx_flags) as ctx:
            for seed in seeds:
                r = ctx.run(args.n_live, args.n_delete, 5 * wl.D, stop_frac=args.stop_frac, max_iter=args.max_iter,
                            seed=seed, return_samples=False)
                r["seed"] = seed
                with lock:
                    print(json.dumps(r), flush=True)
                    runs.append(r)

    seeds = list(range(1, args.seeds + 1))
    n_workers = 1 if args.sequential else min(4, len(seeds))
    t0 = time.perf_counter()
    threads = [threading.Thread(target=work, args=(seeds[g::n_workers],)) for g in range(n_workers)]
    for t in threads:
        t.start()
    for t in threads:
        t.join()
    wall = time.perf_counter() - t0
    z = [r["logZ"] for r in runs]
    print(json.dumps({"workload": wl.name, "D": wl.D, "runs": len(runs), "concurrent_runs": n_workers,
                      "logZ_mean": float(np.mean(z)), "logZ_scatter": float(np.std(z, ddof=1)) if len(z) > 1 else None,
                      "logZ_err_reported": math.sqrt(float(np.mean([r["logZ_err"] ** 2 for r in runs]))),
                      "evals_per_run": int(np.mean([r["n_like_evals"] for r in runs])),
                      "seconds_per_run_inside": float(np.mean([r["seconds"] for r in runs])),
                      "wall_seconds_all_runs": wall}))


if __name__ == "__main__":
    main()
