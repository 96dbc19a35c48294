"""Pins for oracle/nested.py (a11-a14): evidence weights, slice-step validity, closed-form log Z."""
import math
import os

import numpy as np
import pytest
from scipy import stats

from oracle import gaussian, likelihood as LK, nested
from oracle.philox import Stream
from paper_2509_13307_b200 import workloads as W


def test_hand_computed_weights_4_live_2_delete(golden_dir):
    w0, w1, Z, logX_after = np.loadtxt(os.path.join(golden_dir, "ns_weights_4live_2delete.txt"))
    logL = [math.log(3.0), math.log(1.0), math.log(4.0), math.log(2.0)]
    dead, logw, n_j, logX, logZ, Lstar = nested.delete_lowest(logL, 2, 0.0, -np.inf)
    assert dead == [1, 3] and list(n_j) == [4, 3]
    np.testing.assert_allclose(np.exp(logw), [w0, w1], rtol=1e-14)
    assert logZ == pytest.approx(math.log(Z), abs=1e-14) and logX == pytest.approx(logX_after, abs=1e-15)
    assert Lstar == pytest.approx(math.log(2.0))


def test_ties_are_ordered_by_index():
    dead = nested.delete_lowest([1.0, 0.5, 0.5, 0.5], 2, 0.0, -np.inf)[0]
    assert dead == [1, 2]


def test_constant_likelihood_gives_log_Z_equal_log_L():
    """weights telescope: sum_j w_j + X_final = 1 at any stopping point."""
    c = 3.7
    r = nested.run(lambda u: np.full(len(u), c), 2, 20, 10, 1, stop_frac=1e-3, seed=3, max_iter=5)
    assert r["logZ"] == pytest.approx(c, abs=1e-12)
    assert r["H"] == pytest.approx(0.0, abs=1e-12)


def test_batch_error_factor():
    assert nested.batch_error_factor(1000, 1) == pytest.approx(1.0)
    assert nested.batch_error_factor(1000, 500) == pytest.approx(1.4427, rel=2e-3)      # 1/ln 2 as n -> inf
    assert nested.batch_error_factor(200, 100) == pytest.approx(1.0 / math.log(2.0), rel=1e-2)


def test_live_cholesky_is_the_sample_covariance_factor():
    rng = np.random.default_rng(0)
    u = rng.random((50, 4))
    L = nested.live_cholesky(u)
    np.testing.assert_allclose(L @ L.T, np.cov(u.T) + 1e-12 * np.eye(4), rtol=1e-12)
    assert np.allclose(L, np.tril(L))


def test_slice_move_in_one_dimension_samples_the_interval_uniformly():
    """1-D: constraint L > L* <=> x in (0.2, 0.5); output must be uniform there whatever x0 is."""
    f = lambda pts: np.where((pts[:, 0] > 0.2) & (pts[:, 0] < 0.5), 1.0, -1.0)
    x0 = np.full((400, 1), 0.21)
    xs, ls, ne, nf = nested.evolve_chains(f, x0, np.ones(400), np.array([[0.05]]), 0.0, 3, 11, 1)
    assert np.all((xs > 0.2) & (xs < 0.5)) and np.all(ls == 1.0) and nf == 0
    assert stats.kstest((xs[:, 0] - 0.2) / 0.3, "uniform").pvalue > 1e-3


def test_slice_chain_uniform_in_ellipsoid_and_respects_box():
    wl = W.toy_identity(D=4)
    f = lambda u: LK.loglike_u(wl, u)
    rng = np.random.default_rng(0)
    c = 9.0
    Lstar = -0.5 * c + gaussian.log_norm(wl.chol)
    z = rng.standard_normal((300, 4))
    z = z / np.linalg.norm(z, axis=1)[:, None] * rng.random((300, 1)) ** 0.25 * math.sqrt(c) * 0.999
    u0 = 0.5 + z @ wl.chol.T
    l0 = f(u0)
    xs, ls, ne, nf = nested.evolve_chains(f, u0[:150], l0[:150], nested.live_cholesky(u0), Lstar, 12, 1, 1)
    assert np.all(ls > Lstar) and np.all((xs >= 0) & (xs <= 1)) and nf == 0
    np.testing.assert_allclose(ls, f(xs), rtol=1e-12)
    v = (-2.0 * (ls - gaussian.log_norm(wl.chol)) / c) ** 2.0          # (r/R)^D, D = 4
    assert stats.kstest(v, "uniform").pvalue > 1e-3
    assert 3.0 < ne / (150 * 12) < 9.0


def test_out_of_box_proposals_cost_no_likelihood_call():
    calls = []
    def f(pts):
        calls.append(pts.copy()); return np.ones(len(pts))
    nested.evolve_chains(f, np.full((5, 2), 0.5), np.ones(5), 0.3 * np.eye(2), 0.0, 2, 5, 1)
    allp = np.concatenate(calls)
    assert np.all((allp >= 0) & (allp <= 1))


def test_gaussian_in_box_log_Z_and_H_closed_form():
    """identity theory, tight correlated Gaussian centred in the cube: log Z = 0 (normalised L),
    H = -1/2 ln((2 pi e)^D det Sigma).  Two seeds, each within 3 sigma; k = n/2."""
    D = 3
    wl = W.toy_identity(D=D, sigma=0.05)
    Sigma = wl.chol @ wl.chol.T
    H_exact = -0.5 * math.log((2 * math.pi * math.e) ** D * np.linalg.det(Sigma))
    for seed in (1, 2):
        r = nested.run(lambda u: LK.loglike_u(wl, u), D, 80, 40, 5 * D, seed=seed)
        assert r["converged"]
        assert abs(r["logZ"]) < 3.0 * r["logZ_err"]
        assert r["logZ_err"] == pytest.approx(r["logZ_err_analytic"], rel=0.25)
        assert r["H"] == pytest.approx(H_exact, abs=0.8)
        w = np.exp(r["logw"])
        assert w.sum() == pytest.approx(1.0, abs=1e-10)
        mean = w @ r["u"]
        np.testing.assert_allclose(mean, 0.5, atol=0.03)


def test_single_deletion_agrees_with_batch_deletion():
    """batch deletion 'does not introduce new approximations' -- k = 1 and k = n/2 both
    recover the closed form."""
    D = 2
    wl = W.toy_identity(D=D, sigma=0.05)
    r1 = nested.run(lambda u: LK.loglike_u(wl, u), D, 30, 1, 4, seed=4)
    rk = nested.run(lambda u: LK.loglike_u(wl, u), D, 30, 15, 4, seed=4)
    assert abs(r1["logZ"]) < 3.0 * r1["logZ_err"] + 0.1 and abs(rk["logZ"]) < 3.0 * rk["logZ_err"] + 0.1
    assert abs(r1["logZ"] - rk["logZ"]) < 3.0 * math.hypot(r1["logZ_err"], rk["logZ_err"])


def test_stream_definition():
    """draw j of (seed, chain, iteration, tag) is philox(ctr=(j, chain, iteration, tag), key=(seed lo, seed hi))."""
    from oracle.philox import philox4x32_10, u01
    s = Stream((7 << 32) | 9, 5, 3, 1)
    a = s.uniform(); b = s.uniform()
    w0 = philox4x32_10(np.array([0, 5, 3, 1], np.uint32), np.array([9, 7], np.uint32))
    w1 = philox4x32_10(np.array([1, 5, 3, 1], np.uint32), np.array([9, 7], np.uint32))
    assert a == float(u01(w0[0])) and b == float(u01(w1[0]))
