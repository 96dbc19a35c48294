"""Measurement script (not a test: pytest does not collect it) behind profiles/r2_truncation_model.md and the precision
columns of profiles/r2_gemm_pipeline_ab.md.  It lives under tests/ because it compares the CUDA path with the oracle.

    python tests/gemm_precision_probe.py single-layer      # how tcgen05.mma rounds its accumulator: one K = 512 GEMM, 4 sign structures
    python tests/gemm_precision_probe.py c3a [B]           # emulator / log L error of c3a for k-block sizes and k-blocks per TMEM partial

Both drive the kernel parameters through the library's A/B environment variables (NSGPU_BK, NSGPU_KPP, NSGPU_TRUNC_ULPS).
"""
import json
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

import torch  # noqa: E402

from oracle import gaussian, likelihood as LK  # noqa: E402
from paper_2509_13307_b200 import nsgpu, workloads as W  # noqa: E402
from tests.util import loglike_tolerance, theta_of_u, workload  # noqa: E402


def single_layer():
    """One hidden layer: first layer on the CUDA cores, ONE K = 512 output GEMM on the tensor cores, linear output, the
    compensation factor switched off: regress (GPU - oracle) on the oracle output."""
    os.environ["NSGPU_TRUNC_ULPS"] = "0"
    os.environ["NSGPU_BK"] = "64"
    B = 512
    for case in ("random", "positive", "negative", "mixed_bigbias"):
        wl = W.toy(seed=77, width=512, n_out=64, n_hidden=1)
        em = wl.emulators[0]
        if case in ("positive", "negative"):
            em.alpha[0][:] = 40.0; em.beta[0][:] = 0.0          # ReLU-like hidden layer: h >= 0
            em.W[1][:] = np.abs(em.W[1]) * (-1.0 if case == "negative" else 1.0)
            em.b[1][:] = 0.0
        if case == "mixed_bigbias":
            em.b[1][:] = 5.0
        wl.data = np.zeros(wl.n_data); wl.chol = np.eye(wl.n_data)
        theta = theta_of_u(wl, W.u_prior_set(wl, B))
        ref = LK.emulate(wl, theta.astype(np.float64), 0)[:, 0, :]
        for kpp in ("1", "2", "4", "8"):
            os.environ["NSGPU_KPP"] = kpp
            with nsgpu.Context(wl, max_batch=B, mlp=nsgpu.MLP_TC) as ctx:
                got = ctx.emulate_batch(torch.as_tensor(theta, device="cuda"), 0).cpu().numpy().astype(np.float64)[:, 0, :]
            d = (got - ref).ravel()
            x = (ref - (em.b[1][None, :] if case == "mixed_bigbias" else 0)).ravel()
            A = np.stack([x, np.ones_like(x)], 1)
            sl, ic = np.linalg.lstsq(A, d, rcond=None)[0]
            res = d - A @ np.array([sl, ic])
            print(json.dumps({"case": case, "k_blocks_per_partial": kpp, "slope": float(sl), "intercept": float(ic),
                              "rms_output": float(np.sqrt(np.mean(x * x))), "rms_residual": float(np.sqrt(np.mean(res * res)))}), flush=True)


def c3a(B):
    wl = workload("c3a")
    theta = theta_of_u(wl, np.concatenate([W.u_post_set(wl, B // 2), W.u_prior_set(wl, B // 2)]))
    th64 = theta.astype(np.float64)
    ref_spec = LK.emulate(wl, th64, 0)
    ref_ll = LK.loglike(wl, th64)
    chi2 = -2.0 * (ref_ll - gaussian.log_norm(wl.chol))
    tol = loglike_tolerance(chi2)
    em = wl.emulators[0]
    tref = (np.log10(ref_spec) - em.out_mean) / em.out_std
    os.environ.pop("NSGPU_TRUNC_ULPS", None)
    for bk, kpps in (("64", ("1", "2")), ("32", ("2", "4", "8"))):
        for kpp in kpps:
            os.environ["NSGPU_BK"], os.environ["NSGPU_KPP"] = bk, kpp
            with nsgpu.Context(wl, max_batch=B) as ctx:
                t = torch.as_tensor(theta, device="cuda")
                spec = ctx.emulate_batch(t, 0).cpu().numpy().astype(np.float64)
                ll = ctx.loglike_batch(t).cpu().numpy()
            d = ((np.log10(spec) - em.out_mean) / em.out_std - tref).ravel()
            x = tref.ravel()
            err = np.abs(ll - ref_ll)
            print(json.dumps({"BK": bk, "k_blocks_per_partial": kpp, "rms_dt": float(np.sqrt(np.mean(d * d))),
                              "slope": float(np.dot(d, x) / np.dot(x, x)), "max_rel_P": float(np.max(np.abs(spec - ref_spec) / ref_spec)),
                              "max_dlogL_chi2_le_2000": float(err[chi2 <= 2000].max()), "max_dlogL_over_tol": float(np.max(err / tol))}), flush=True)


if __name__ == "__main__":
    mode = sys.argv[1] if len(sys.argv) > 1 else "single-layer"
    if mode == "single-layer":
        single_layer()
    else:
        c3a(int(sys.argv[2]) if len(sys.argv) > 2 else 256)
