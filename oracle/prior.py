"""Prior transform u in [0,1]^D -> theta (step a1; priors of P:L78-91 Table 1; reading N1:
the sampler lives in the unit hypercube, each dimension has its own transform)."""
import numpy as np
from scipy.special import ndtri  # Phi^-1, library primitive

UNIFORM, GAUSSIAN = 0, 1


def transform(kind, p0, p1, u):
    """kind int[D]; uniform: theta = p0 + (p1-p0) u; gaussian: theta = p0 + p1 Phi^-1(u)."""
    u = np.asarray(u, dtype=np.float64)
    theta = np.empty_like(u)
    for d in range(u.shape[-1]):
        if kind[d] == UNIFORM:
            theta[..., d] = p0[d] + (p1[d] - p0[d]) * u[..., d]
        else:
            theta[..., d] = p0[d] + p1[d] * ndtri(u[..., d])
    return theta


def in_support(kind, p0, p1, theta):
    """True where theta lies inside every uniform box dimension (Gaussian dims are unbounded)."""
    theta = np.asarray(theta, dtype=np.float64)
    ok = np.all(np.isfinite(theta), axis=-1)
    for d in range(theta.shape[-1]):
        if kind[d] == UNIFORM:
            ok &= (theta[..., d] >= p0[d]) & (theta[..., d] <= p1[d])
    return ok
