"""Shared test helpers: workloads with oracle-made data vectors, tolerance rules."""
import functools
import re
import os

import numpy as np

from oracle import likelihood as LK, prior
from paper_2509_13307_b200 import workloads as W

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

MAKERS = {
    "toy": W.toy, "toy_small": lambda: W.toy(width=16, n_out=10, n_hidden=2), "identity": W.toy_identity,
    "tiny_shear": W.tiny_shear, "tiny_shear_spline": lambda: W.tiny_shear(spline=True),
    "tiny_shear_lcdm": lambda: W.tiny_shear(w0wa=False), "tiny_cmb": W.tiny_cmb,
    "c1": W.cmb, "c2": W.c2, "c3a": W.c3a, "c3b": W.c3b, "c4_lcdm": W.c4_lcdm,
    "toy_w64": lambda: W.toy(width=64, n_out=100, n_hidden=3),
    "tiny_shear_paper": W.tiny_shear_paper, "c5i": lambda: W.c5(True), "c5": lambda: W.c5(False),
    "cmb_tt": W.cmb_tt, "tiny_cmb_tt": lambda: W.cmb_tt(seed=9, width=64, n_hidden=2, ell_max=131),
}


def theta_of_u(wl, u):
    """oracle prior transform, rounded to the float32 the boundary takes (input rounding is not error)."""
    return prior.transform(wl.prior_kind, wl.prior_p0, wl.prior_p1, u).astype(np.float32)


@functools.lru_cache(maxsize=None)
def workload(name, noise=True):
    """Workload with data/covariance attached; the mock data vector comes from the ORACLE at theta_0."""
    wl = MAKERS[name]()
    if wl.theory.kind == 0:
        return wl
    th0 = theta_of_u(wl, wl.u_fid[None]).astype(np.float64)
    m0 = LK.theory(wl, th0)[0]
    if wl.theory.kind == 4:
        W.attach_cmb_tt_data(wl, m0, noise=noise)
    elif wl.theory.kind == 1:
        W.attach_toy_data(wl, m0)
    else:
        W.attach_data(wl, m0, noise=noise)
    return wl


def loglike_tolerance(chi2):
    """reading T2: |dlogL| <= 1e-3 where the oracle chi2 <= 2000, 1e-6 chi2 beyond."""
    chi2 = np.asarray(chi2, np.float64)
    return np.where(chi2 <= 2000.0, 1e-3, 1e-6 * chi2)


def header_exports():
    src = open(os.path.join(ROOT, "include", "nsgpu.h")).read()
    return sorted(set(re.findall(r"\b(nsgpu_[a-z_]+)\s*\(", src)))
