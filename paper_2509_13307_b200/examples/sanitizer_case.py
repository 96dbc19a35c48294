"""The smallest run that goes through every kernel family of the hot path, for `compute-sanitizer` (memcheck, racecheck,
synccheck; one tool per GPU call, B200_PROFILING.md) and for quick checks after a kernel change:

    compute-sanitizer --tool memcheck python -m paper_2509_13307_b200.examples.sanitizer_case

  1. c3a (39-D shear, 512-wide emulator, 50 z nodes) at B = 64: first layer, tcgen05 GEMMs as single CTAs, -- forced
     with NSGPU_MLP_CLUSTER -- as CTA pairs that multicast the weight tiles, and as the fused multi-layer kernel (all
     three must agree bit for bit), resident projection, DMMA chi^2;
  2. a width-64 shear model with the streaming projection kernels and the tiled chi^2;
  3. the CMB binning path (three emulators) and the cosmic-variance TT likelihood at small sizes;
  4. a short nested-sampling run (slice rounds, compaction, deletion + evidence scan, live covariance, error-bar kernel).
Data vectors come from the CUDA path itself (no oracle): the run only has to finish with finite numbers that agree
between the launch configurations.  Prints one summary line."""
import numpy as np
import torch

from paper_2509_13307_b200 import nsgpu, workloads as W


def _attach(wl, flags=0):
    n = wl.n_data
    wl.data, wl.chol = (np.ones(n), None) if wl.theory.kind == W.THEORY_CMB_TT_CV else (np.zeros(n), np.eye(n))
    with nsgpu.Context(wl, max_batch=4, mlp=flags) as c0:
        u0 = torch.as_tensor(wl.u_fid[None].astype(np.float32), device="cuda")
        m0 = c0.theory_batch(c0.prior_transform(u0)).cpu().numpy()[0]
    if wl.theory.kind == W.THEORY_CMB_TT_CV:
        return W.attach_cmb_tt_data(wl, m0)
    return W.attach_data(wl, m0)


def main():
    out = {}
    wl = _attach(W.c3a())
    u = torch.as_tensor(np.concatenate([W.u_post_set(wl, 32), W.u_prior_set(wl, 32)]).astype(np.float32), device="cuda")
    res = []
    for flags in (nsgpu.MLP_TC | nsgpu.MLP_LAYERED | nsgpu.MLP_NO_CLUSTER, nsgpu.MLP_TC | nsgpu.MLP_LAYERED | nsgpu.MLP_CLUSTER,
                  nsgpu.MLP_TC | nsgpu.MLP_FUSED):
        with nsgpu.Context(wl, max_batch=64, mlp=flags) as ctx:
            res.append(ctx.loglike_batch(ctx.prior_transform(u)).cpu().numpy())
    assert np.all(np.isfinite(res[0])) and np.array_equal(res[0], res[1]) and np.array_equal(res[0], res[2])
    out["c3a_B64_pairs_and_fused_equal_single"] = True
    ws = _attach(W.shear(seed=22, w0wa=True, n_z_emu=11, n_z=11, width=64, n_hidden=2, n_k=40, n_chi=150, n_ell=11, n_tomo=5,
                         z_max=3.0, n_ia_terms=1, n_m_terms=2, name="s64p"), nsgpu.SHEAR_STREAM)
    us = torch.as_tensor(W.u_post_set(ws, 40).astype(np.float32), device="cuda")
    with nsgpu.Context(ws, max_batch=40, mlp=nsgpu.SHEAR_STREAM | nsgpu.CHI2_TILED) as ctx:
        a = ctx.loglike_batch(ctx.prior_transform(us)).cpu().numpy()
    with nsgpu.Context(ws, max_batch=40) as ctx:
        b = ctx.loglike_batch(ctx.prior_transform(us)).cpu().numpy()
    assert np.all(np.isfinite(a)) and np.max(np.abs(a - b)) < 1e-6 * np.max(np.abs(a))
    out["streaming_vs_resident_max_rel"] = float(np.max(np.abs(a - b) / np.abs(a)))
    for name, wl2 in (("tiny_cmb", W.tiny_cmb()), ("tiny_cmb_tt", W.cmb_tt(seed=9, width=64, n_hidden=2, ell_max=131))):
        wl2 = _attach(wl2)
        u2 = torch.as_tensor(W.u_post_set(wl2, 33, scale=2e-4).astype(np.float32), device="cuda")
        with nsgpu.Context(wl2, max_batch=33) as ctx:
            ll = ctx.loglike_batch(ctx.prior_transform(u2)).cpu().numpy()
        assert np.all(np.isfinite(ll))
        out[name + "_finite"] = True
    wg = W.toy_identity(D=4)
    with nsgpu.Context(wg, max_batch=128) as ctx:
        r = ctx.run(128, 64, 8, seed=1, return_samples=False)
    assert r["converged"] and abs(r["logZ"]) <= 3.0 * r["logZ_err"] + 0.1
    out["ns_logZ"] = round(r["logZ"], 3)
    print("sanitizer_case ok:", out)


if __name__ == "__main__":
    main()
