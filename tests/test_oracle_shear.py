"""Pins for oracle/shear.py (steps a5-a8): closed forms and special cases."""
import math
import types

import numpy as np
import pytest
from scipy.interpolate import CubicSpline

from oracle import shear as S
from paper_2509_13307_b200 import workloads as W


def _th(n_chi=100, z_max=2.0, n_z=50, n_k=60, k_min=1e-6, k_max=1e4, n_ell=4, n_tomo=2):
    return types.SimpleNamespace(n_chi=n_chi, z_max=z_max, n_z=n_z, n_z_emu=n_z, n_k=n_k, k_min=k_min,
                                 k_max=k_max, n_ell=n_ell, n_tomo=n_tomo, z_interp=0,
                                 ell=100.0 * 30.0 ** ((np.arange(n_ell) + 0.5) / n_ell))


def test_quadrature_nodes_are_midpoints_in_a():
    a, z, da = S.quadrature_nodes(_th(n_chi=4, z_max=1.0))
    np.testing.assert_allclose(a, [0.9375, 0.8125, 0.6875, 0.5625]); assert da == 0.125
    np.testing.assert_allclose(z, 1 / a - 1)


def test_E_of_z_lcdm_and_w0wa_values():
    # LCDM at z=1, Om=0.3: sqrt(0.3*8 + 0.7)
    assert S.E_of_z(np.array([1.0]), 0.3, -1.0, 0.0)[0] == pytest.approx(math.sqrt(3.1), rel=1e-15)
    # w0=-0.9, wa=0.2 at z=1: DE term (1+z)^{3(1+w0+wa)} e^{-3 wa z/(1+z)} = 2^{0.9} e^{-0.3}
    want = math.sqrt(0.3 * 8 + 0.7 * 2 ** 0.9 * math.exp(-0.3))
    assert S.E_of_z(np.array([1.0]), 0.3, -0.9, 0.2)[0] == pytest.approx(want, rel=1e-15)


@pytest.mark.parametrize("n", [100, 200, 400])
def test_einstein_de_sitter_closed_forms(n):
    """Om = 1: chi(z) = 2 (c/H0) (1 - (1+z)^-1/2), D = a. Midpoint error is O(N^-2)."""
    th = _th(n_chi=n)
    a, z, da = S.quadrature_nodes(th)
    chi, dchi, D, Eq = S.background(a, z, da, 1.0, -1.0, 0.0)
    chi_exact = 2.0 * S.C_OVER_H0 * (1.0 - np.sqrt(a))
    # worst RELATIVE error sits at the first node (chi_0 ~ da) and is first order (8.4e-4 at N=100);
    # the absolute error is second order everywhere
    assert np.max(np.abs(chi / chi_exact - 1.0)) < 1.0e-3 * (100.0 / n)
    scale = (100.0 / n) ** 2
    assert np.max(np.abs(chi - chi_exact)) / chi_exact[-1] < 2.0e-5 * scale
    assert np.max(np.abs(D / a - 1.0)) < 1.0e-3 * (100.0 / n)
    np.testing.assert_allclose(Eq, (1 + z) ** 1.5, rtol=1e-14)
    np.testing.assert_allclose(np.sum(dchi), 2.0 * S.C_OVER_H0 * (1 - math.sqrt(1 / 3.0)), rtol=2e-4 * scale)


def test_convergence_order_of_chi_is_two():
    errs = []
    for n in (100, 200, 400):
        a, z, da = S.quadrature_nodes(_th(n_chi=n))
        chi = S.background(a, z, da, 1.0, -1.0, 0.0)[0]
        errs.append(abs(chi[-1] / (2.0 * S.C_OVER_H0 * (1.0 - math.sqrt(a[-1]))) - 1.0))
    assert 3.5 < errs[0] / errs[1] < 4.5 and 3.5 < errs[1] / errs[2] < 4.5


def test_growth_index_lcdm_value():
    """Om=0.3 LCDM: D(a=0.5)/D(1) from gamma = 0.55 is within 0.5% of the exact growth factor
    0.7789/... (exact LCDM ratio D(z=1)/D(0) = 0.6118 for Om=0.3, e.g. Hamilton 2001 integral)."""
    th = _th(n_chi=400, z_max=1.0)
    a, z, da = S.quadrature_nodes(th)
    D = S.background(a, z, da, 0.3, -1.0, 0.0)[2]
    # exact: D ∝ H(a) ∫_0^a da'/(a' H)^3, evaluated numerically here with a fine trapezoid
    def Dex(ae):
        x = np.linspace(1e-6, ae, 200001); Hx = np.sqrt(0.3 / x ** 3 + 0.7)
        f = 1.0 / (x * Hx) ** 3
        return math.sqrt(0.3 / ae ** 3 + 0.7) * float(np.sum(0.5 * (f[1:] + f[:-1]) * np.diff(x)))
    ratio_exact = Dex(a[-1]) / Dex(1.0)
    assert D[-1] == pytest.approx(ratio_exact, rel=5e-3)
    assert D[0] == pytest.approx(1.0, abs=2e-3)


def test_growth_index_w0wa_hand_computed_golden(golden_dir):
    """reading S13, gamma = 0.55 + 0.05 (1 + w0 + wa/2): the 4-cell grid at Om = 0.3, w0 = -0.8, wa = 0.3 evaluated by
    hand in tests/golden/growth_w0wa_4node.txt (gamma = 0.5675).  `wa` for `wa/2`, a wrong 0.05 or a dropped w0 moves
    ln D by > 1e-4 here; the pin is at 1e-12."""
    import os
    rows = np.loadtxt(os.path.join(golden_dir, "growth_w0wa_4node.txt"))
    a, z, da = S.quadrature_nodes(_th(n_chi=4, z_max=1.0))
    np.testing.assert_array_equal(a, rows[:, 0])
    chi, dchi, D, Eq = S.background(a, z, da, 0.3, -0.8, 0.3)
    np.testing.assert_allclose(Eq ** 2, rows[:, 1], rtol=1e-13)
    np.testing.assert_allclose(np.log(D), rows[:, 4], rtol=1e-12)
    # the hand table is itself consistent: Om(a) = 0.3 a^-3/E^2, and ln D from its own Om(a)^gamma column
    np.testing.assert_allclose(0.3 * rows[:, 0] ** -3 / rows[:, 1], rows[:, 2], rtol=1e-13)
    np.testing.assert_allclose(rows[:, 2] ** 0.5675, rows[:, 3], rtol=1e-13)
    g = rows[:, 3] * 0.125 / rows[:, 0]
    np.testing.assert_allclose(-(np.cumsum(g) - 0.5 * g), rows[:, 4], rtol=1e-13)
    # sensitivity of the pin: the plausible mistakes are far outside it
    for gam in (0.55 + 0.05 * (1 - 0.8 + 0.3), 0.55 + 0.5 * (1 - 0.8 + 0.15), 0.55 + 0.05 * (1 + 0.15), 0.55):
        gq = rows[:, 2] ** gam * 0.125 / rows[:, 0]
        assert np.max(np.abs(-(np.cumsum(gq) - 0.5 * gq) - rows[:, 4])) > 1e-4


@pytest.mark.parametrize("w0,wa", [(-0.8, 0.3), (-1.0, 0.0), (-1.3, -0.6), (-0.6, 0.4)])
def test_growth_against_linear_growth_ode(w0, wa):
    """D(a) of reading S13 against a direct integration of the linear growth equation for the same flat w0wa
    background, D'' + (3/a + dlnE/da) D' = 1.5 Om a^-5 E^-2 D, started deep in matter domination (D = a): the
    growth-index form is a <1% approximation of it (Linder 2005) -- a sign error in the w-dependence of gamma or a
    wrong exponent is not."""
    from scipy.integrate import solve_ivp
    Om = 0.3
    th = _th(n_chi=400, z_max=2.0)
    a, z, da = S.quadrature_nodes(th)
    D = S.background(a, z, da, Om, w0, wa)[2]
    E2 = lambda x: Om * x ** -3 + (1 - Om) * x ** (-3 * (1 + w0 + wa)) * np.exp(-3 * wa * (1 - x))
    def rhs(x, y):
        h = 1e-6 * x
        dlnE = 0.5 * (np.log(E2(x + h)) - np.log(E2(x - h))) / (2 * h)
        return [y[1], -(3.0 / x + dlnE) * y[1] + 1.5 * Om / (x ** 5 * E2(x)) * y[0]]
    sol = solve_ivp(rhs, [1e-3, 1.0], [1e-3, 1.0], dense_output=True, rtol=1e-9, atol=1e-12)
    Dex = sol.sol(a)[0] / sol.sol(1.0)[0]
    assert np.max(np.abs(D / Dex - 1.0)) < 1.0e-2
    # and the w-dependence of gamma is needed for that at the dynamical end of the prior: with a constant 0.55 ...
    if (w0, wa) == (-0.6, 0.4):
        assert np.max(np.abs(D / Dex - 1.0)) < 0.6e-2


def test_omega_m_is_physical_density_over_h_squared():
    """reading S11 of the garbled Table-1 row: omega_b = Omega_b h^2, omega_cdm = Omega_cdm h^2, so
    Omega_m = (0.02 + 0.12)/0.7^2 = 2/7; /h instead of /h^2 gives 0.2."""
    th = types.SimpleNamespace(idx_omega_b=2, idx_omega_cdm=0, idx_h=1, idx_w0=-1, idx_wa=-1, idx_eta0=-1, idx_dz=3,
                               idx_ia=4, idx_m=5, n_tomo=1, n_ia_terms=1, n_m_terms=1)
    p = S.physical_parameters(th, np.array([0.12, 0.7, 0.02, 0.01, 0.5, 0.02]))
    assert p["Om"] == pytest.approx(2.0 / 7.0, rel=1e-15)
    assert (p["w0"], p["wa"], p["eta0"]) == (-1.0, 0.0, 0.7)
    assert p["dz"].tolist() == [0.01] and p["A"].tolist() == [[0.5, 0.0, 0.0]] and p["m"].tolist() == [[0.02, 0.0]]
    # through the model: the lensing amplitude of a pure-lensing spectrum scales as Om^2 at fixed distances; check the
    # value the full model_vector uses by comparing two h at fixed omegas on a flat table (C ~ Om^2 x geometry)
    wl = W.tiny_shear()
    from oracle import prior
    t0 = prior.transform(wl.prior_kind, wl.prior_p0, wl.prior_p1, wl.u_fid)
    assert S.physical_parameters(wl.theory, t0)["Om"] == pytest.approx(
        (t0[wl.theory.idx_omega_b] + t0[wl.theory.idx_omega_cdm]) / t0[wl.theory.idx_h] ** 2, rel=1e-15)


@pytest.mark.parametrize("Om,w0,wa,n", [(1.0, -1.0, 0.0, 100), (1.0, -1.0, 0.0, 200), (0.3, -0.8, 0.3, 100), (0.3, -0.8, 0.3, 200)])
def test_ia_window_carries_n_of_chi_normalised_over_comoving_distance(Om, w0, wa, n):
    """eq. A4 weights n_i(chi), a density per unit comoving distance: n_i(chi) dchi = n_i(z) dz, so
    with the reading dz/dchi = E H0/c the quantity -W^I D / (A C1 rho_cr Om) must integrate to 1 over chi on the
    quadrature grid (midpoint rule, O(N^-2)).  A missing or inverted E, or c/H0 for H0/c, breaks the normalisation."""
    th = _th(n_chi=n)
    a, z, da = S.quadrature_nodes(th)
    chi, dchi, D, Eq = S.background(a, z, da, Om, w0, wa)
    nz = S.n_of_z(z, 0.8, 0.1, 0.02)
    WI = S.window_ia(z, nz, np.full(n, 1.7), Om, D, Eq)
    n_chi_density = -WI * D / (1.7 * S.C1_RHOCR * Om)
    assert np.sum(n_chi_density * dchi) == pytest.approx(1.0, abs=2e-4 * (100.0 / n) ** 2)
    # independent of the cosmology-dependent Jacobian: the same sum in z
    assert np.sum(nz * da / a ** 2) == pytest.approx(np.sum(n_chi_density * dchi), rel=1e-13)


def test_ia_window_single_plane_source():
    """n(z) = unit-weight spike at node s (n dz = 1): W^I is -A C1 rho_cr Om / D_s per unit comoving distance of
    that cell, i.e. -A C1 rho_cr Om / (D_s dchi_s), and zero elsewhere."""
    th = _th(n_chi=50)
    a, z, da = S.quadrature_nodes(th)
    chi, dchi, D, Eq = S.background(a, z, da, 0.3, -0.9, 0.2)
    s = 21
    nz = np.zeros(50); nz[s] = 1.0 / (da / a[s] ** 2)
    WI = S.window_ia(z, nz, np.full(50, 0.8), 0.3, D, Eq)
    assert WI[s] == pytest.approx(-0.8 * S.C1_RHOCR * 0.3 / (D[s] * dchi[s]), rel=1e-13)
    assert np.count_nonzero(WI) == 1


def test_single_plane_lensing_kernel():
    """n(z) = delta at node s: W(q) = 1.5 Om (H0/c)^2 (1+z_q) chi_q (chi_s - chi_q)/chi_s for q < s."""
    th = _th(n_chi=50)
    a, z, da = S.quadrature_nodes(th)
    chi = S.background(a, z, da, 0.3, -1.0, 0.0)[0]
    s = 37
    nz = np.zeros(50); nz[s] = 1.0 / (da / a[s] ** 2)          # unit weight n dz = 1
    Wg = S.window_gamma(a, z, da, chi, nz, 0.3)
    want = 1.5 * 0.3 / S.C_OVER_H0 ** 2 * (1 + z) * chi * (chi[s] - chi) / chi[s]
    np.testing.assert_allclose(Wg[:s], want[:s], rtol=1e-13)
    assert np.all(Wg[s:] == 0.0)


def test_window_gamma_equals_suffix_scan_form():
    """A - chi*B with suffix sums A = sum n dz, B = sum n dz/chi (the O(N) form the GPU uses)."""
    rng = np.random.default_rng(0)
    th = _th(n_chi=64)
    a, z, da = S.quadrature_nodes(th)
    chi = S.background(a, z, da, 0.31, -0.8, 0.3)[0]
    nz = rng.random(64)
    w = nz * da / a ** 2
    A = np.concatenate([np.cumsum(w[::-1])[::-1][1:], [0.0]])
    B = np.concatenate([np.cumsum((w / chi)[::-1])[::-1][1:], [0.0]])
    want = 1.5 * 0.31 / S.C_OVER_H0 ** 2 * (1 + z) * chi * (A - chi * B)
    np.testing.assert_allclose(S.window_gamma(a, z, da, chi, nz, 0.31), want, rtol=1e-11, atol=1e-20)


def test_n_of_z_shift_moves_the_mean_up_and_is_normalised():
    z = np.linspace(-1, 3, 40001)
    n = S.n_of_z(z, 0.7, 0.1, 0.05)
    dz = z[1] - z[0]
    assert np.sum(n) * dz == pytest.approx(1.0, rel=1e-9)
    assert np.sum(n * z) * dz == pytest.approx(0.75, rel=1e-9)        # mean = mu + dz  (reading S8)
    assert S.n_of_z(np.array([0.75]), 0.7, 0.1, 0.05)[0] == pytest.approx(1 / (0.1 * math.sqrt(2 * math.pi)))


def test_ia_window_formula():
    # W^I = -A C1rho Om / D * n(z) * E * H0/c  (eq. A4 with n(chi) = n(z) dz/dchi)
    got = S.window_ia(np.array([0.5]), np.array([2.0]), np.array([1.5]), 0.3, np.array([0.8]), np.array([1.3]))
    assert got[0] == pytest.approx(-1.5 * 0.0138768 * 0.3 / 0.8 * 2.0 * 1.3 / 2997.92458, rel=1e-15)
    assert 5e-14 * 2.77536627e11 == pytest.approx(S.C1_RHOCR, rel=1e-5)


def test_extensions_reduce_to_paper_model():
    z = np.linspace(0, 2, 7); ell = np.array([100.0, 550.0, 3000.0])
    np.testing.assert_array_equal(S.ia_amplitude(z, 0.7, 0.0, 0.0), np.full(7, 0.7))
    np.testing.assert_array_equal(S.m_bias(ell, 0.01, 0.0), np.full(3, 0.01))
    assert S.m_bias(np.array([550.0 * 30.0]), 0.0, 1.0)[0] == pytest.approx(1.0)
    assert S.ia_amplitude(np.array([0.62]), 0.0, 1.0, 0.0)[0] == pytest.approx(0.0, abs=1e-15)


def test_spline_reproduces_cubics_and_matches_scipy():
    x = np.linspace(0.0, 2.0, 12); xe = np.linspace(0.0, 2.0, 50)
    c = lambda t: 0.3 * t ** 3 - 1.1 * t ** 2 + 0.4 * t + 2.0
    np.testing.assert_allclose(S.notaknot_spline_eval(x, c(x)[:, None], xe)[:, 0], c(xe), rtol=1e-12, atol=1e-12)
    rng = np.random.default_rng(5)
    Y = rng.standard_normal((12, 9))
    np.testing.assert_allclose(S.notaknot_spline_eval(x, Y, xe), CubicSpline(x, Y)(xe), rtol=1e-10, atol=1e-11)
    # non-uniform nodes as well
    xn = np.sort(rng.random(9)) * 2; xn[0], xn[-1] = 0.0, 2.0
    Yn = rng.standard_normal((9, 3))
    np.testing.assert_allclose(S.notaknot_spline_eval(xn, Yn, xe), CubicSpline(xn, Yn)(xe), rtol=1e-9, atol=1e-10)


def test_table_interpolation_exact_on_bilinear_tables_and_zero_outside():
    th = _th(n_z=5, n_k=11, k_min=1e-2, k_max=10.0)
    zl, lk = S.z_nodes_limber(th), S.log10k_nodes(th)
    table = 1.5 - 0.7 * zl[:, None] + 2.0 * lk[None, :] + 0.3 * zl[:, None] * lk[None, :]
    zq = np.array([0.0, 0.13, 1.0, 1.999, 2.0]); k = np.array([0.01, 0.5, 3.3, 9.99, 10.0])
    want = 10.0 ** (1.5 - 0.7 * zq + 2.0 * np.log10(k) + 0.3 * zq * np.log10(k))
    np.testing.assert_allclose(S.power_at(th, zl, lk, table, zq, k, 0.7), want, rtol=1e-12)
    out = S.power_at(th, zl, lk, table, np.array([0.5, 0.5]), np.array([0.00999, 10.01]), 0.7)
    assert out.tolist() == [0.0, 0.0]
    # baryon template: eta0 = 0.9 lowers log10 P by 0.02 k^2/(k^2+1)
    r = S.power_at(th, zl, lk, table, np.array([0.5]), np.array([1.0]), 0.9) / S.power_at(th, zl, lk, table, np.array([0.5]), np.array([1.0]), 0.7)
    assert r[0] == pytest.approx(10 ** (-0.2 * 0.1 * 0.5), rel=1e-13)


def test_concave_in_z_table_is_underestimated_by_linear_interpolation():
    """the paper's own observation."""
    th = _th(n_z=6, n_k=5, k_min=1e-2, k_max=10.0)
    zl, lk = S.z_nodes_limber(th), S.log10k_nodes(th)
    f = lambda zz: 3.0 - 0.4 * zz ** 2
    table = np.repeat(f(zl)[:, None], 5, axis=1)
    zq = np.linspace(0.01, 1.99, 57)
    got = S.power_at(th, zl, lk, table, zq, np.full(57, 1.0), 0.7)
    assert np.all(got <= 10.0 ** f(zq) * (1 + 1e-14))


@pytest.mark.parametrize("n", [100, 200, 400])
def test_power_law_limber_closed_form(n):
    """P = A k^n_s (z independent), W = chi^p: C(ell) = A (ell+1/2)^n_s chi_max^{2p-1-n_s}/(2p-1-n_s)
    in an EdS background; midpoint error O(N^-2)."""
    th = _th(n_chi=n, n_tomo=1)
    zl, lk = S.z_nodes_limber(th), S.log10k_nodes(th)
    A, ns, p = 3.0e3, -1.2, 2.0
    table = np.repeat((math.log10(A) + ns * lk)[None, :], th.n_z, axis=0)
    a, z, da = S.quadrature_nodes(th)
    chi, dchi, D, Eq = S.background(a, z, da, 1.0, -1.0, 0.0)
    Wg = (chi ** p)[None, :]
    C = S.limber_cl(th, chi, dchi, z, Wg, np.zeros_like(Wg), table, zl, lk, 0.7)[0]
    chi_max = 2.0 * S.C_OVER_H0 * (1.0 - math.sqrt(1.0 / 3.0))
    e = 2 * p - 1 - ns
    want = A * (th.ell + 0.5) ** ns * chi_max ** e / e
    np.testing.assert_allclose(C, want, rtol=2.5e-3 * (100.0 / n) ** 2)


def test_four_term_sum_equals_factored_form():
    rng = np.random.default_rng(7)
    th = _th(n_chi=40, n_tomo=3, n_z=7, n_k=30, k_min=1e-4, k_max=50.0)
    zl, lk = S.z_nodes_limber(th), S.log10k_nodes(th)
    table = rng.standard_normal((7, 30))
    a, z, da = S.quadrature_nodes(th)
    chi, dchi, D, Eq = S.background(a, z, da, 0.3, -1.0, 0.0)
    Wg, Wi = rng.random((3, 40)), -rng.random((3, 40))
    C = S.limber_cl(th, chi, dchi, z, Wg, Wi, table, zl, lk, 0.6)
    Wt = Wg + Wi
    for pidx, (i, j) in enumerate(S.pair_index(3)):
        for b in range(th.n_ell):
            P = S.power_at(th, zl, lk, table, z, (th.ell[b] + 0.5) / chi, 0.6)
            assert C[pidx, b] == pytest.approx(np.sum(dchi / chi ** 2 * Wt[i] * Wt[j] * P), rel=1e-12)
    assert S.pair_index(3) == [(0, 0), (0, 1), (0, 2), (1, 1), (1, 2), (2, 2)]


def test_model_vector_layout_and_m_bias_scaling():
    """pair-major, ell fastest (S16); (1+m_i)(1+m_j) rescaling."""
    wl = W.tiny_shear()
    th = wl.theory
    rng = np.random.default_rng(9)
    table = 2.0 + 0.1 * rng.standard_normal((th.n_z_emu, th.n_k))
    theta = np.array(wl.prior_p0, float).copy()
    from oracle import prior
    theta = prior.transform(wl.prior_kind, wl.prior_p0, wl.prior_p1, wl.u_fid)
    base = theta.copy(); base[th.idx_m:th.idx_m + 2 * th.n_tomo] = 0.0
    m0 = S.model_vector(th, base, table)
    mod = base.copy(); mod[th.idx_m + 2 * 1] = 0.1          # m_{1,0} = 0.1
    m1 = S.model_vector(th, mod, table)
    ratio = (m1 / m0).reshape(-1, th.n_ell)
    want = {(0, 0): 1.0, (0, 1): 1.1, (0, 2): 1.0, (1, 1): 1.21, (1, 2): 1.1, (2, 2): 1.0}
    for pidx, ij in enumerate(S.pair_index(3)):
        np.testing.assert_allclose(ratio[pidx], want[ij], rtol=1e-12)


def test_spline_variant_close_to_full_on_smooth_table():
    """c3b-vs-c3a style check on an injected smooth table (SURVEY §8(d) structure caveat)."""
    full, spl = W.tiny_shear(spline=False), W.tiny_shear(spline=True)
    from oracle import prior
    theta = prior.transform(full.prior_kind, full.prior_p0, full.prior_p1, full.u_fid)
    lk = S.log10k_nodes(full.theory)
    f = lambda zz: (3.0 - 0.8 * (lk[None, :] + 1.0) ** 2 / 3.0) - 0.35 * zz[:, None] + 0.05 * zz[:, None] ** 2
    a = S.model_vector(full.theory, theta, f(S.z_nodes_emulator(full.theory)))
    b = S.model_vector(spl.theory, theta, f(S.z_nodes_emulator(spl.theory)))
    np.testing.assert_allclose(b, a, rtol=5e-3)


def test_single_coefficient_layout_is_the_truncated_expansion():
    """one A_IA and one m per bin.  The (1, 1) parameter layout must give exactly the model of
    the (3, 2) layout with the higher coefficients set to zero, and moving A_i / m_i of ONE bin must change
    exactly the spectra that bin takes part in."""
    import dataclasses
    wl = W.tiny_shear_paper()
    th = wl.theory
    assert (th.n_ia_terms, th.n_m_terms) == (1, 1) and wl.D == 9 + 3 * th.n_tomo
    from oracle import prior
    theta = prior.transform(wl.prior_kind, wl.prior_p0, wl.prior_p1, wl.u_fid)
    rng = np.random.default_rng(3)
    theta[th.idx_ia:th.idx_ia + th.n_tomo] = rng.uniform(-2, 2, th.n_tomo)
    theta[th.idx_m:th.idx_m + th.n_tomo] = rng.uniform(-0.05, 0.05, th.n_tomo)
    table = 2.0 + 0.1 * rng.standard_normal((th.n_z_emu, th.n_k))
    m11 = S.model_vector(th, theta, table)
    # the same physical point in the (3, 2) layout
    nt = th.n_tomo
    wide = np.concatenate([theta[:th.idx_ia],
                           np.stack([theta[th.idx_ia:th.idx_ia + nt], np.zeros(nt), np.zeros(nt)], 1).ravel(),
                           np.stack([theta[th.idx_m:th.idx_m + nt], np.zeros(nt)], 1).ravel()])
    th32 = dataclasses.replace(th, n_ia_terms=3, n_m_terms=2, idx_m=th.idx_ia + 3 * nt)
    np.testing.assert_array_equal(S.model_vector(th32, wide, table), m11)
    # locality: bin 2's amplitude and bias touch only pairs containing bin 2
    for idx in (th.idx_ia + 2, th.idx_m + 2):
        mod = theta.copy(); mod[idx] += 0.3
        changed = (S.model_vector(th, mod, table) != m11).reshape(-1, th.n_ell).any(axis=1)
        assert [bool(c) for c in changed] == [2 in ij for ij in S.pair_index(nt)]
