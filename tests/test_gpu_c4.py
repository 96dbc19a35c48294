"""-m gpu: pins for BASELINE.json configs[4], the 39-D w0wa cosmic-shear model against its 37-D LambdaCDM restriction
(P:L127, L131 run settings; Table 2 row).  log Z has no closed form here and the oracle's own nested sampling is
far too slow at 39-D (1e8 evaluations x 0.01 s), so SURVEY 8(c.4) pins what can be pinned:
  * the restricted 37-D run against a 39-D run whose w0, wa priors are collapsed onto (-1, 0): same likelihood, same
    code path, two different random walks -- the evidences must agree within their errors;
  * per-point log L of the final live set of a run against the oracle;
  * seed-to-seed scatter of log Z against the reported error bar.
Sizes are reduced (500 live / 250 deleted, stop at 0.1) to keep the suite short; the full-size comparison is
`python -m paper_2509_13307_b200.examples.model_comparison` (profiles/r2_c4_model_comparison.md).
The sampler itself is pinned at the full configs[4] settings by the closed-form run in tests/test_gpu_sampler.py."""
import copy
import math

import numpy as np
import pytest

from oracle import gaussian, likelihood as LK
from paper_2509_13307_b200 import nsgpu, workloads as W
from tests.util import loglike_tolerance, workload

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")

N_LIVE, N_DELETE, STOP = 500, 250, 0.1


def _collapsed_w0wa():
    """c3a with the w0, wa priors shrunk onto (-1, 0): theta_w0 = -1 exactly in float32, |theta_wa| <= 1e-9."""
    wl = copy.deepcopy(workload("c3a"))
    th = wl.theory
    wl.prior_p0[th.idx_w0], wl.prior_p1[th.idx_w0] = -1.0 - 1e-9, -1.0 + 1e-9
    wl.prior_p0[th.idx_wa], wl.prior_p1[th.idx_wa] = -1e-9, 1e-9
    return wl


def test_restricted_run_equals_run_with_collapsed_priors_and_live_set_matches_oracle():
    rest, full = workload("c4_lcdm"), _collapsed_w0wa()
    np.testing.assert_array_equal(rest.data, full.data)          # same mock, same covariance (seed 1003)
    with nsgpu.Context(rest, max_batch=N_LIVE) as c37:
        r37 = c37.run(N_LIVE, N_DELETE, 5 * rest.D, stop_frac=STOP, seed=1)
    with nsgpu.Context(full, max_batch=N_LIVE) as c39:
        r39 = c39.run(N_LIVE, N_DELETE, 5 * full.D, stop_frac=STOP, seed=1)
        # the collapsed model's likelihood at the restricted run's live points equals the restricted likelihood
        live37 = r37["theta"][-N_LIVE:]
        lifted = np.insert(live37, 6, np.array([[-1.0], [0.0]], np.float32).repeat(N_LIVE, axis=1), axis=1)
        l39 = c39.loglike_batch(torch.as_tensor(lifted, device="cuda")).cpu().numpy()
    for r in (r37, r39):
        assert r["converged"] and r["n_failed_moves"] == 0 and r["n_iter"] > 20
        assert r["logZ_err"] == pytest.approx(r["logZ_err_analytic"], rel=0.35)
    np.testing.assert_array_equal(l39, r37["logL"][-N_LIVE:])
    assert abs(r37["logZ"] - r39["logZ"]) <= 3.0 * math.hypot(r37["logZ_err"], r39["logZ_err"]), (r37["logZ"], r39["logZ"])
    assert r37["H"] == pytest.approx(r39["H"], rel=0.1)
    # the collapsed dimensions stayed collapsed
    assert np.all(r39["theta"][:, 6] == -1.0) and np.max(np.abs(r39["theta"][:, 7])) <= 1e-9
    # per-point parity of the final live set (the points evidence accumulates at) against the oracle: all 500
    ref = LK.loglike(rest, live37.astype(np.float64))
    chi2 = -2.0 * (ref - gaussian.log_norm(rest.chol))
    err = np.abs(r37["logL"][-N_LIVE:] - ref)
    assert np.all(err <= loglike_tolerance(chi2)), (err / loglike_tolerance(chi2)).max()
    assert np.all(chi2 <= 2000.0)                                # the whole live set is in the absolute-tolerance regime
    # nested sampling's own bookkeeping: live points carry equal weights, weights sum to 1
    w = np.exp(r37["logw"])
    assert w.sum() == pytest.approx(1.0, abs=1e-9)


def test_seed_scatter_of_the_restricted_model_is_consistent_with_the_reported_error():
    wl = workload("c4_lcdm")
    n, k = 300, 150
    zs, errs = [], []
    with nsgpu.Context(wl, max_batch=n) as ctx:
        for seed in (11, 12, 13, 14, 15):
            r = ctx.run(n, k, 5 * wl.D, stop_frac=STOP, seed=seed, return_samples=False)
            assert r["converged"] and r["n_failed_moves"] == 0
            zs.append(r["logZ"]); errs.append(r["logZ_err"])
    assert np.std(zs, ddof=1) < 2.5 * np.mean(errs), (zs, errs)
    assert np.std(zs, ddof=1) > 0.1 * np.mean(errs)               # ... and the seeds really are different runs
