"""Pins for oracle/emulator.py (steps a2-a4): hand-computed net, linear collapses, ReLU limit,
brute-force loops, de-standardisation special case."""
import os
import types

import numpy as np
import pytest

from oracle import emulator as E


def _emu(W, b, alpha, beta, in_mean, in_std, out_mean, out_std, out_kind=0):
    f = lambda a: np.asarray(a, np.float32)
    return types.SimpleNamespace(n_in=W[0].shape[0], n_hidden=len(W) - 1, width=W[0].shape[1],
                                 n_out=W[-1].shape[1], out_kind=out_kind, W=[f(w) for w in W],
                                 b=[f(x) for x in b], alpha=[f(a) for a in alpha], beta=[f(x) for x in beta],
                                 in_mean=f(in_mean), in_std=f(in_std), out_mean=f(out_mean), out_std=f(out_std))


def _random_emu(rng, n_in, width, n_out, n_hidden, out_kind=0):
    W, b, al, be = [], [], [], []
    fi = n_in
    for _ in range(n_hidden):
        W.append(rng.standard_normal((fi, width))); b.append(rng.standard_normal(width))
        al.append(rng.standard_normal(width)); be.append(rng.standard_normal(width)); fi = width
    W.append(rng.standard_normal((fi, n_out))); b.append(rng.standard_normal(n_out))
    return _emu(W, b, al, be, rng.standard_normal(n_in), 0.5 + rng.random(n_in),
                rng.standard_normal(n_out), 0.5 + rng.random(n_out), out_kind)


def test_hand_computed_2_3_2(golden_dir):
    want = np.loadtxt(os.path.join(golden_dir, "mlp_2_3_2_hand.txt"))
    emu = _emu([np.array([[1, 0, -1], [0.5, 2, 1]]), np.array([[1, 2], [0, 1], [-2, 0.5]])],
               [[0, 0.5, -0.5], [0.125, -0.25]], [[0, 2, -1]], [[0.5, 0, 1]],
               [0, 0], [1, 1], [1, -1], [2, 0.5])
    got = E.mlp_raw(emu, np.array([[1.0, 2.0]]))[0]
    np.testing.assert_allclose(got, want, rtol=0, atol=1e-14)


def test_transposed_weight_would_fail():
    """y = x.W + b with W [fan_in, fan_out]: a non-square first layer pins the orientation."""
    emu = _emu([np.array([[1.0, 2.0, 3.0]]), np.array([[1.0], [10.0], [100.0]])],
               [[0, 0, 0], [0]], [[0, 0, 0]], [[1, 1, 1]], [0], [1], [0], [1])
    assert E.mlp_raw(emu, np.array([[2.0]]))[0, 0] == pytest.approx(2 + 40 + 600)


def test_beta_one_is_product_of_matrices():
    rng = np.random.default_rng(1)
    emu = _random_emu(rng, 5, 7, 4, 3)
    emu.beta = [np.ones(7, np.float32) for _ in range(3)]
    X = rng.standard_normal((6, 5))
    x = (X - emu.in_mean.astype(float)) / emu.in_std.astype(float)
    for l in range(4):
        x = np.einsum("mi,ij->mj", x, emu.W[l].astype(float)) + emu.b[l].astype(float)
    want = x * emu.out_std.astype(float) + emu.out_mean.astype(float)
    np.testing.assert_allclose(E.mlp_raw(emu, X), want, rtol=1e-13, atol=1e-13)


def test_alpha_zero_is_linear_with_half_one_plus_beta():
    rng = np.random.default_rng(2)
    emu = _random_emu(rng, 3, 5, 2, 2)
    emu.alpha = [np.zeros(5, np.float32) for _ in range(2)]
    X = rng.standard_normal((4, 3))
    x = (X - emu.in_mean.astype(float)) / emu.in_std.astype(float)
    for l in range(2):
        x = (x @ emu.W[l].astype(float) + emu.b[l].astype(float)) * 0.5 * (1.0 + emu.beta[l].astype(float))
    want = (x @ emu.W[2].astype(float) + emu.b[2].astype(float)) * emu.out_std.astype(float) + emu.out_mean.astype(float)
    np.testing.assert_allclose(E.mlp_raw(emu, X), want, rtol=1e-13, atol=1e-13)


def test_relu_limit():
    """beta = 0, alpha -> large: sigma(alpha t) t -> max(t, 0)."""
    t = np.array([-3.0, -0.5, 0.25, 2.0])
    got = E.activation(t, np.full(4, 1e4), np.zeros(4))
    np.testing.assert_allclose(got, np.maximum(t, 0.0), atol=1e-12)
    # and the overflow-safe sigmoid does not overflow
    assert np.all(np.isfinite(E.sigmoid(np.array([-1e5, 1e5]))))


def test_matmul_form_equals_triple_loop():
    rng = np.random.default_rng(3)
    emu = _random_emu(rng, 4, 6, 5, 3)
    X = rng.standard_normal((3, 4))
    got = E.mlp_raw(emu, X)
    for m in range(3):
        np.testing.assert_allclose(got[m], E.mlp_forward_loops(emu, X[m]), rtol=1e-12, atol=1e-12)


def test_sigma_out_zero_gives_exp10_of_mu_out():
    rng = np.random.default_rng(4)
    emu = _random_emu(rng, 3, 4, 6, 2, out_kind=1)
    emu.out_std = np.zeros(6, np.float32)
    got = E.mlp_forward(emu, rng.standard_normal((5, 3)))
    np.testing.assert_array_equal(got, np.broadcast_to(10.0 ** emu.out_mean.astype(float), (5, 6)))


def test_activation_formula_by_value():
    # (beta + sigma(alpha x)(1-beta)) x at alpha=1, beta=0.25, x=ln 3: sigma = 3/4
    x = np.log(3.0)
    assert E.activation(np.array([x]), np.array([1.0]), np.array([0.25]))[0] == pytest.approx((0.25 + 0.75 * 0.75) * x, abs=1e-15)
