"""Pins of the cosmic-variance TT likelihood oracle (oracle/cmb_tt.py): the density written out with
lgamma, its normalisation and mean by quadrature, the closed form under a rescaling of the theory, the maximum."""
import math

import numpy as np
from scipy import integrate

from oracle import cmb_tt


def test_matches_the_formula_written_out():
    rng = np.random.default_rng(0)
    ell = np.arange(2, 40)
    c = 10.0 ** rng.normal(-9, 0.3, len(ell))
    ch = c * rng.chisquare(2 * ell + 1) / (2 * ell + 1)
    got = cmb_tt.loglike_spectrum(ell, ch, c[None])[0]
    assert got == np.float64(got) and abs(got - cmb_tt.logpdf_direct(ell, ch, c)) < 1e-9 * abs(got)


def test_density_is_normalised_with_mean_c():
    """int p(Chat | C) dChat = 1 and E[Chat] = C: pins the Jacobian nu / C and the argument nu Chat / C."""
    for l, c in ((2, 3.0), (7, 0.2)):
        p = lambda ch: math.exp(cmb_tt.loglike_spectrum([l], [ch], np.array([[c]]))[0])
        norm, _ = integrate.quad(p, 0, 60 * c, limit=200)
        mean, _ = integrate.quad(lambda ch: ch * p(ch), 0, 60 * c, limit=200)
        assert abs(norm - 1.0) < 1e-7 and abs(mean - c) < 1e-7 * c


def test_rescaled_theory_closed_form_and_maximum():
    """C = a Chat for all l: log L(a) - log L(1) = -1/2 sum nu (1/a + ln a - 1) <= 0, maximal at a = 1."""
    ell = np.arange(2, 300)
    nu = 2.0 * ell + 1.0
    ch = 10.0 ** np.linspace(-9, -11, len(ell))
    base = cmb_tt.loglike_spectrum(ell, ch, ch[None])[0]
    for a in (0.9, 1.0, 1.003, 1.2):
        got = cmb_tt.loglike_spectrum(ell, ch, (a * ch)[None])[0]
        want = -0.5 * np.sum(nu * (1.0 / a + math.log(a) - 1.0))
        assert abs((got - base) - want) < 1e-8 * max(1.0, abs(want))
        assert got <= base + 1e-9


def test_multipoles_are_independent_and_additive():
    ell = np.array([2, 3, 50])
    c = np.array([[1.0, 2.0, 3.0]]); ch = np.array([1.1, 1.7, 3.2])
    total = cmb_tt.loglike_spectrum(ell, ch, c)[0]
    parts = sum(cmb_tt.loglike_spectrum(ell[i:i + 1], ch[i:i + 1], c[:, i:i + 1])[0] for i in range(3))
    assert abs(total - parts) < 1e-12
