"""Share of a nested-sampling round spent in the sampler's own kernels (steps a11-a12: slice proposal / update state machine
and compaction) against the likelihood stages (a2-a10) -- SURVEY 8(d), row "slice/select/scan: measured as round overhead".

    python -m paper_2509_13307_b200.examples.round_overhead [--iterations 3] [--workload c4|cmb_tt]

Runs the first few iterations of the BASELINE.json configs[4] run (39-D shear, 1000 live points, 500 deleted per iteration,
195 slice moves) with the library's per-stage CUDA-event timers on and prints the device time per stage and per round.
(The timers add ~20 event records per round, so the absolute round time is a little above an unprofiled run's.)
"""
import argparse
import json

import numpy as np
import torch

from paper_2509_13307_b200 import nsgpu, workloads as W
from paper_2509_13307_b200.examples.model_comparison import _mock_data


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--iterations", type=int, default=3)
    ap.add_argument("--workload", default="c4", choices=["c4", "cmb_tt"])
    args = ap.parse_args()
    if args.workload == "c4":
        wl = _mock_data(W.c3a())
        n_live, n_delete, n_steps = 1000, 500, 5 * wl.D
    else:
        wl = W.cmb_tt()
        wl.data, wl.chol = np.ones(wl.n_data), None
        with nsgpu.Context(wl, max_batch=8) as c0:
            u0 = torch.as_tensor(wl.u_fid[None].astype(np.float32), device="cuda")
            W.attach_cmb_tt_data(wl, c0.theory_batch(c0.prior_transform(u0)).cpu().numpy()[0])
        n_live, n_delete, n_steps = 1000, 500, 30
    with nsgpu.Context(wl, max_batch=n_live) as ctx:
        ctx.run(n_live, n_delete, n_steps, seed=1, max_iter=1, return_samples=False)          # warm-up
        ctx.set_profiling(True)
        ctx.stage_times()
        r = ctx.run(n_live, n_delete, n_steps, seed=1, max_iter=args.iterations, return_samples=False)
        st = ctx.stage_times()
        ctx.set_profiling(False)
    rounds = r["n_rounds"]
    total = sum(ms for ms, _ in st.values())
    out = {"workload": wl.name, "iterations": r["n_iter"], "rounds": rounds, "evaluations": r["n_like_evals"],
           "proposals_per_round": (r["n_like_evals"] - n_live) / rounds, "seconds_sampling": r["seconds_sampling"],
           "device_ms_per_round": total / rounds,
           "stage_us_per_round": {k: 1e3 * ms / rounds for k, (ms, cnt) in st.items() if cnt},
           "sampler_share": st["slice_round"][0] / total}
    print(json.dumps(out))


if __name__ == "__main__":
    main()
