"""The paper's own CMB likelihood (section 2.4; reading C5 of DESIGN.md):
a cosmic-variance-limited temperature power spectrum.  "The likelihood for the observed power spectrum, given a
theoretical model C_l(theta), follows a chi-squared distribution of shape 2l+1": with nu_l = 2l+1,

    nu_l Chat_l / C_l(theta)  ~  chi^2_{nu_l}     independently for every multipole l,

so the density of the observed Chat_l is  p(Chat_l | C_l) = (nu_l / C_l) f_{chi^2_nu}(nu_l Chat_l / C_l)  and
log L(theta) = sum_l log p(Chat_l | C_l(theta)), normalisation included (reading L1).  The chi^2 density is the
library primitive `scipy.stats.chi2.logpdf`; `logpdf_direct` writes the same density out with lgamma for the pin.
"""
import math

import numpy as np
from scipy.stats import chi2 as _chi2


def ells(th, n_out):
    return th.ell_min + np.arange(n_out)


def loglike_spectrum(ell, c_hat, c_model):
    """c_model: [B, n_l] theory spectra, c_hat: [n_l] observed.  Returns log L [B] (fp64)."""
    c_model = np.asarray(c_model, np.float64)
    nu = 2.0 * np.asarray(ell, np.float64) + 1.0
    x = nu[None, :] * np.asarray(c_hat, np.float64)[None, :] / c_model
    return np.sum(np.log(nu[None, :] / c_model) + _chi2.logpdf(x, nu[None, :]), axis=1)


def logpdf_direct(ell, c_hat, c_model):
    """the same density from its formula: log(nu/C) + (nu/2 - 1) log x - x/2 - (nu/2) log 2 - lgamma(nu/2)."""
    out = 0.0
    for l, ch, c in zip(ell, c_hat, c_model):
        nu = 2.0 * l + 1.0
        x = nu * ch / c
        out += math.log(nu / c) + (0.5 * nu - 1.0) * math.log(x) - 0.5 * x - 0.5 * nu * math.log(2.0) - math.lgamma(0.5 * nu)
    return out
