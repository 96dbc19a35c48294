"""Pins for oracle/gaussian.py (a10), oracle/prior.py (a1) and oracle/philox.py."""
import math
import os

import numpy as np
import pytest
from scipy.special import erfinv

from oracle import gaussian as G, philox, prior


def test_identity_covariance_is_sum_of_squares():
    rng = np.random.default_rng(0)
    r = rng.standard_normal((5, 7))
    np.testing.assert_allclose(G.chi2(np.eye(7), r, np.zeros(7)), np.sum(r * r, axis=1), rtol=1e-14)


def test_diagonal_covariance():
    rng = np.random.default_rng(1)
    s = 0.5 + rng.random(6)
    m, d = rng.standard_normal((4, 6)), rng.standard_normal(6)
    np.testing.assert_allclose(G.chi2(np.diag(s), m, d), np.sum(((m - d) / s) ** 2, axis=1), rtol=1e-13)


def test_residual_equal_to_cholesky_column_has_unit_chi2():
    rng = np.random.default_rng(2)
    A = rng.standard_normal((8, 8)); L = np.linalg.cholesky(A @ A.T + np.eye(8))
    d = rng.standard_normal(8)
    for j in range(8):
        w = G.whiten(L, (L[:, j])[None, :])
        want = np.zeros(8); want[j] = 1.0
        np.testing.assert_allclose(w[0], want, atol=1e-12)
        assert G.chi2(L, (d + L[:, j])[None, :], d)[0] == pytest.approx(1.0, abs=1e-12)


def test_3x3_explicit_inverse_and_sign_convention():
    C = np.array([[4.0, 1.0, 0.5], [1.0, 3.0, 0.2], [0.5, 0.2, 2.0]])
    # cofactor inverse written out
    det = (C[0, 0] * (C[1, 1] * C[2, 2] - C[1, 2] * C[2, 1]) - C[0, 1] * (C[1, 0] * C[2, 2] - C[1, 2] * C[2, 0])
           + C[0, 2] * (C[1, 0] * C[2, 1] - C[1, 1] * C[2, 0]))
    cof = np.empty((3, 3))
    for i in range(3):
        for j in range(3):
            sub = np.delete(np.delete(C, i, 0), j, 1)
            cof[i, j] = (-1) ** (i + j) * (sub[0, 0] * sub[1, 1] - sub[0, 1] * sub[1, 0])
    Cinv = cof.T / det
    L = np.linalg.cholesky(C)
    m, d = np.array([[1.0, -2.0, 0.5]]), np.array([0.3, 0.1, -0.7])
    r = (m - d)[0]
    assert G.chi2(L, m, d)[0] == pytest.approx(r @ Cinv @ r, rel=1e-13)
    want = -0.5 * (r @ Cinv @ r) - 0.5 * math.log((2 * math.pi) ** 3 * det)
    assert G.loglike(L, m, d)[0] == pytest.approx(want, rel=1e-13)
    # the upper-triangular factor (a transposed operand) gives a different chi2
    assert abs(G.chi2(L.T.copy(), m, d)[0] - r @ Cinv @ r) > 1e-3


def test_log_det_against_eigenvalues():
    rng = np.random.default_rng(3)
    A = rng.standard_normal((6, 6)); C = A @ A.T + 0.5 * np.eye(6)
    want = -0.5 * (6 * math.log(2 * math.pi) + np.sum(np.log(np.linalg.eigvalsh(C))))
    assert G.log_norm(np.linalg.cholesky(C)) == pytest.approx(want, rel=1e-13)


def test_prior_transform_uniform_endpoints_and_gaussian_quantiles():
    kind = np.array([0, 1, 0]); p0 = np.array([-3.0, 0.01, 2.0]); p1 = np.array([1.0, 0.02, 4.0])
    th = prior.transform(kind, p0, p1, np.array([[0.0, 0.5, 1.0], [0.25, 0.8413447460685429, 0.5]]))
    np.testing.assert_allclose(th[0], [-3.0, 0.01, 4.0], atol=1e-15)
    np.testing.assert_allclose(th[1], [-2.0, 0.03, 3.0], atol=1e-12)     # Phi(1) = 0.84134...
    u = np.array([1e-6, 0.1, 0.3, 0.77, 1 - 1e-6])
    got = prior.transform(np.array([1]), np.array([0.0]), np.array([1.0]), u[:, None])[:, 0]
    np.testing.assert_allclose(got, math.sqrt(2.0) * erfinv(2.0 * u - 1.0), rtol=1e-10)


def test_in_support():
    kind = np.array([0, 1]); p0 = np.array([0.0, 0.0]); p1 = np.array([1.0, 1.0])
    th = np.array([[0.5, 9.0], [1.5, 0.0], [-0.1, 0.0], [0.5, np.nan]])
    assert prior.in_support(kind, p0, p1, th).tolist() == [True, False, False, False]


def test_philox_known_answers(golden_dir):
    for line in open(os.path.join(golden_dir, "philox4x32_10_kat.txt")):
        if line.startswith("#") or not line.strip():
            continue
        w = [int(x, 16) for x in line.split()]
        got = philox.philox4x32_10(np.array(w[0:4], np.uint32), np.array(w[4:6], np.uint32))
        assert [int(x) for x in got] == w[6:10]


def test_philox_vectorised_matches_scalar_and_stream_blocks():
    ctr = np.array([[i, 7, 3, 0] for i in range(130)], np.uint32)
    key = np.array([42, 0], np.uint32)
    bulk = philox.philox4x32_10(ctr, key)
    s = philox.Stream(42, 7, 3, 0)
    for i in range(130):
        assert np.array_equal(s.words(), bulk[i])
        assert np.array_equal(philox.philox4x32_10(ctr[i], key), bulk[i])


def test_u01_open_interval_and_box_muller_moments():
    assert 0.0 < philox.u01(0) < philox.u01(0xFFFFFFFF) < 1.0
    ctr = np.zeros((20000, 4), np.uint32); ctr[:, 0] = np.arange(20000)
    w = philox.philox4x32_10(ctr, np.array([1, 2], np.uint32))
    a, b = philox.box_muller(w[:, 0], w[:, 1])
    z = np.concatenate([a, b])
    assert abs(z.mean()) < 0.02 and abs(z.var() - 1.0) < 0.03 and abs(np.mean(a * b)) < 0.02
