"""Gaussian likelihood against a fixed dense covariance (step a10; "multivariate
Gaussian"; readings L1, L2: normalisation included, lower Cholesky factor)."""
import math
import numpy as np


def whiten(L, r):
    """forward substitution L w = r, written out row by row. r: [B, n] -> w [B, n]."""
    L = np.asarray(L, dtype=np.float64)
    r = np.asarray(r, dtype=np.float64)
    n = L.shape[0]
    w = np.zeros_like(r)
    for i in range(n):
        w[:, i] = (r[:, i] - w[:, :i] @ L[i, :i]) / L[i, i]
    return w


def log_norm(L):
    """-1/2 ln det(2 pi C) = -1/2 (n ln 2pi + 2 sum ln L_ii)."""
    L = np.asarray(L, dtype=np.float64)
    n = L.shape[0]
    return -0.5 * (n * math.log(2.0 * math.pi) + 2.0 * float(np.sum(np.log(np.diag(L)))))


def chi2(L, model, data):
    w = whiten(L, np.asarray(model, np.float64) - np.asarray(data, np.float64)[None, :])
    return np.sum(w * w, axis=1)


def loglike(L, model, data):
    return -0.5 * chi2(L, model, data) + log_norm(L)
