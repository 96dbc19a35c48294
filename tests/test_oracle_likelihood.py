"""Pins for oracle/cmb.py (a9) and oracle/likelihood.py (end-to-end a2-a10)."""
import types

import numpy as np
import pytest

from oracle import cmb, gaussian, likelihood as LK, prior
from paper_2509_13307_b200 import workloads as W


def _theta(wl, u):
    return prior.transform(wl.prior_kind, wl.prior_p0, wl.prior_p1, u)


def test_cmb_binning_of_constant_spectra_and_calibration():
    wl = W.tiny_cmb()
    th = wl.theory
    n_out = wl.emulators[0].n_out
    spectra = [np.full(n_out, 2.0), np.full(n_out, -3.0), np.full(n_out, 5.0)]
    theta = _theta(wl, wl.u_fid); theta[th.cal_index] = 2.0
    m = cmb.model_vector(th, theta, spectra)
    assert m.shape == (23,)
    np.testing.assert_allclose(m[:9], 2.0 / 4.0, rtol=1e-7)      # rows sum to 1 (fp32 weights), / A_cal^2
    np.testing.assert_allclose(m[9:16], -3.0 / 4.0, rtol=1e-7)
    np.testing.assert_allclose(m[16:], 5.0 / 4.0, rtol=1e-7)


def test_cmb_binning_matrix_structure():
    wl = W.cmb()
    th = wl.theory
    assert wl.n_data == 613 and wl.D == 7 and len(th.bin_col) == (2508 - 29) + 2 * (1996 - 29)   # reading C2
    rows = np.diff(th.bin_ptr)
    assert rows[:215].min() >= 11 and rows[:215].max() <= 12 and rows[215:].min() >= 9 and rows[215:].max() <= 10
    # bin of a linear ramp = the ramp at the bin centre
    n_out = 2507
    ramp = np.arange(2, 2509, dtype=float)
    theta = _theta(wl, wl.u_fid)
    m = cmb.model_vector(th, theta, [ramp, ramp, ramp])
    lo = th.bin_col[th.bin_ptr[0]] + 2; hi = th.bin_col[th.bin_ptr[1] - 1] + 2
    assert m[0] == pytest.approx(0.5 * (lo + hi) / theta[6] ** 2, rel=1e-6) and lo == 30
    # block diagonal: TE rows only touch TE columns
    c = th.bin_col[th.bin_ptr[215]:th.bin_ptr[215 + 199]]
    assert c.min() >= n_out and c.max() < 2 * n_out


def test_configs_have_the_baseline_shapes():
    assert (W.c2().D, W.c2().n_data, W.c2().emulators[0].n_in, W.c2().emulators[0].n_out) == (37, 300, 7, 420)
    a, b = W.c3a(), W.c3b()
    assert (a.D, a.n_data, a.emulators[0].n_in, a.theory.n_z_emu, b.theory.n_z_emu, b.theory.n_z) == (39, 300, 9, 50, 12, 50)
    r = W.c4_lcdm()
    assert r.D == 37 and r.emulators[0].n_in == 9 and list(r.theory.emu_in_idx[6:8]) == [-1, -1]
    np.testing.assert_array_equal(r.emulators[0].W[2], a.emulators[0].W[2])     # same weights as c3a
    t = W.toy()
    assert (t.D, t.n_data, t.emulators[0].width, t.emulators[0].n_hidden) == (6, 100, 128, 4)


@pytest.mark.parametrize("make", [W.tiny_shear, W.tiny_cmb, lambda: W.toy(width=16, n_out=10)])
def test_permutation_and_batch_size_invariance(make):
    wl = make()
    m0 = LK.theory(wl, _theta(wl, wl.u_fid[None]))[0]
    (W.attach_toy_data if wl.theory.kind == 1 else W.attach_data)(wl, m0)
    u = W.u_post_set(wl, 7)
    ll = LK.loglike_u(wl, u)
    perm = np.array([3, 0, 6, 1, 5, 2, 4])
    np.testing.assert_allclose(LK.loglike_u(wl, u[perm]), ll[perm], rtol=1e-12)
    for i in range(7):
        assert LK.loglike_u(wl, u[i:i + 1])[0] == pytest.approx(ll[i], rel=1e-12)


def test_noiseless_data_gives_the_normalisation_constant_at_fiducial():
    wl = W.tiny_shear()
    th0 = _theta(wl, wl.u_fid[None])
    W.attach_data(wl, LK.theory(wl, th0)[0], noise=False)
    assert LK.loglike(wl, th0)[0] == pytest.approx(gaussian.log_norm(wl.chol), rel=1e-14)


def test_out_of_support_is_minus_inf():
    wl = W.tiny_cmb()
    th0 = _theta(wl, wl.u_fid[None])
    W.attach_data(wl, LK.theory(wl, th0)[0])
    bad = th0.copy(); bad[0, 2] = 5.0        # h outside U(0.64, 0.982)
    far = th0.copy(); far[0, 6] = 1.5        # A_cal: Gaussian prior, unbounded -> finite
    out = LK.loglike(wl, np.concatenate([th0, bad, far]))
    assert np.isfinite(out[0]) and out[1] == -np.inf and np.isfinite(out[2])


def test_restricted_lcdm_equals_w0wa_model_at_w0_minus1_wa_0():
    """c4: the 37-D restriction is the 39-D model with w0 = -1, wa = 0 (same code path, same weights)."""
    full = W.shear(seed=7, w0wa=True, n_z_emu=9, n_z=9, width=48, n_hidden=2, n_k=37, n_chi=23, n_ell=6, n_tomo=3)
    rest = W.shear(seed=7, fix_w0wa=True, n_z_emu=9, n_z=9, width=48, n_hidden=2, n_k=37, n_chi=23, n_ell=6, n_tomo=3)
    tr = _theta(rest, W.u_prior_set(rest, 3))
    tf = np.insert(tr, 6, np.array([[-1.0], [0.0]]).repeat(3, axis=1), axis=1)
    np.testing.assert_allclose(LK.theory(rest, tr), LK.theory(full, tf), rtol=1e-13)


def test_emulate_tap_shapes():
    wl = W.tiny_shear()
    out = LK.emulate(wl, _theta(wl, W.u_prior_set(wl, 2)))
    assert out.shape == (2, wl.theory.n_z_emu, wl.theory.n_k) and np.all(out > 0)
