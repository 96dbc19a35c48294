"""Cosmic-shear theory vector (steps a5-a8): background, windows, z/k interpolation of the
emulated log10 P(k,z), extended-Limber projection (eqs. A1-A4), nuisances
(P:L350-351), with the grid sizes of BASELINE.json configs[2,3] and the readings S1-S21 of
DESIGN.md.  Units: distances in Mpc/h, k in h/Mpc, H0/c = 1/2997.92458 h/Mpc.

Everything is fp64 and written in the order of SURVEY.md §8(c.1) step 2 (a..k).
"""
import math
import numpy as np

C_OVER_H0 = 2997.92458          # c/H0 in Mpc/h
C1_RHOCR = 0.0138768            # C1 rho_cr = 5e-14 x 2.77536627e11 (reading S12)


# ---- a. grids (theta independent) ---------------------------------------------------------
def z_nodes_emulator(th):
    return np.arange(th.n_z_emu, dtype=np.float64) * th.z_max / (th.n_z_emu - 1)


def z_nodes_limber(th):
    return np.arange(th.n_z, dtype=np.float64) * th.z_max / (th.n_z - 1)


def quadrature_nodes(th):
    """midpoint rule in the scale factor on n_chi cells from a=1 down to a_min = 1/(1+z_max)
    ("evenly spaced in scale factor"; reading S3). Returns a_q, z_q, da."""
    a_min = 1.0 / (1.0 + th.z_max)
    da = (1.0 - a_min) / th.n_chi
    a_q = 1.0 - (np.arange(th.n_chi, dtype=np.float64) + 0.5) * da
    return a_q, 1.0 / a_q - 1.0, da


def log10k_nodes(th):
    return np.linspace(math.log10(th.k_min), math.log10(th.k_max), th.n_k)


# ---- b..d. background ---------------------------------------------------------------------
def E_of_z(z, Om, w0, wa):
    """flat w0wa: E^2 = Om (1+z)^3 + (1-Om)(1+z)^{3(1+w0+wa)} exp(-3 wa z/(1+z)) (reading S11)."""
    return np.sqrt(Om * (1.0 + z) ** 3
                   + (1.0 - Om) * (1.0 + z) ** (3.0 * (1.0 + w0 + wa)) * np.exp(-3.0 * wa * z / (1.0 + z)))


def background(a_q, z_q, da, Om, w0, wa):
    """chi_q [Mpc/h], dchi_q, growth D_q (D(z=0)=1 in the continuum), E_q on the quadrature nodes.
    chi: cumulative midpoint rule of dchi = (c/H0) da / (a^2 E); growth: Linder growth index
    gamma = 0.55 + 0.05 (1 + w0 + wa/2), ln D = - int Om(a)^gamma dlna (reading S13)."""
    E_q = E_of_z(z_q, Om, w0, wa)
    f_q = 1.0 / (a_q ** 2 * E_q)
    n = len(a_q)
    chi = np.empty(n)
    run = 0.0
    for q in range(n):
        chi[q] = C_OVER_H0 * (run + 0.5 * f_q[q] * da)
        run += f_q[q] * da
    dchi = C_OVER_H0 * f_q * da
    Om_a = Om * a_q ** -3 / E_q ** 2
    gamma = 0.55 + 0.05 * (1.0 + w0 + 0.5 * wa)
    g_q = Om_a ** gamma * da / a_q
    lnD = np.empty(n)
    run = 0.0
    for q in range(n):
        lnD[q] = -(run + 0.5 * g_q[q])
        run += g_q[q]
    return chi, dchi, np.exp(lnD), E_q


# ---- e..g. source distributions and windows ---------------------------------------------------
def n_of_z(z, mean, sigma, dz):
    """Gaussian n_i(z - dz_i): the mean moves by +dz_i (P:L351 garbled; reading S8), analytic
    normalisation (reading S9)."""
    return np.exp(-0.5 * ((z - mean - dz) / sigma) ** 2) / (sigma * math.sqrt(2.0 * math.pi))


def window_gamma(a_q, z_q, da, chi, nz_q, Om):
    """eq. A3 as the naive O(N^2) sum on the quadrature nodes (outer loop over q, inner
    sum over q' > q):  W(q) = 1.5 Om (H0/c)^2 (1+z_q) chi_q sum_{q'>q} n(z_q') dz_q' (chi_q' - chi_q)/chi_q'."""
    n = len(a_q)
    dz_q = da / a_q ** 2
    W = np.zeros(n)
    for q in range(n):
        s = np.sum(nz_q[q + 1:] * dz_q[q + 1:] * (chi[q + 1:] - chi[q]) / chi[q + 1:])
        W[q] = 1.5 * Om / C_OVER_H0 ** 2 * (1.0 + z_q[q]) * chi[q] * s
    return W


def window_ia(z_q, nz_q, A_q, Om, D_q, E_q):
    """eq. A4 with n_i(chi) = n_i(z) dz/dchi = n_i(z) E (H0/c)."""
    return -A_q * C1_RHOCR * Om / D_q * nz_q * E_q / C_OVER_H0


def ia_amplitude(z, A0, A1, A2):
    """reading S2: A_i(z) = A_{i,0} + A_{i,1} x + A_{i,2} x^2, x = (1+z)/1.62 - 1
    (A_{i,1} = A_{i,2} = 0 is the paper's single amplitude per bin)."""
    x = (1.0 + z) / 1.62 - 1.0
    return A0 + A1 * x + A2 * x * x


def m_bias(ell, m0, m1):
    """reading S2: m_i(ell) = m_{i,0} + m_{i,1} ln(ell/550)/ln 30 (m_{i,1}=0: paper)."""
    return m0 + m1 * np.log(ell / 550.0) / math.log(30.0)


# ---- k. cubic not-a-knot spline in z ----------------------------------------------------------
def notaknot_spline_eval(x, Y, xe):
    """Textbook C^2 cubic spline through (x_i, Y[i,...]) with not-a-knot end conditions,
    evaluated at xe. Second derivatives M from the (dense) tridiagonal system."""
    x = np.asarray(x, np.float64)
    Y = np.asarray(Y, np.float64)
    n = len(x)
    assert n >= 4
    h = np.diff(x)
    A = np.zeros((n, n))
    rhs = np.zeros((n,) + Y.shape[1:])
    A[0, 0], A[0, 1], A[0, 2] = h[1], -(h[0] + h[1]), h[0]
    A[n - 1, n - 3], A[n - 1, n - 2], A[n - 1, n - 1] = h[n - 2], -(h[n - 3] + h[n - 2]), h[n - 3]
    for i in range(1, n - 1):
        A[i, i - 1], A[i, i], A[i, i + 1] = h[i - 1], 2.0 * (h[i - 1] + h[i]), h[i]
        rhs[i] = 6.0 * ((Y[i + 1] - Y[i]) / h[i] - (Y[i] - Y[i - 1]) / h[i - 1])
    M = np.linalg.solve(A, rhs.reshape(n, -1)).reshape(rhs.shape)
    out = np.empty((len(xe),) + Y.shape[1:])
    for e, xv in enumerate(xe):
        i = int(np.clip(np.searchsorted(x, xv, side="right") - 1, 0, n - 2))
        hl, t0, t1 = h[i], x[i + 1] - xv, xv - x[i]
        out[e] = (M[i] * t0 ** 3 + M[i + 1] * t1 ** 3) / (6.0 * hl) \
            + (Y[i] / hl - M[i] * hl / 6.0) * t0 + (Y[i + 1] / hl - M[i + 1] * hl / 6.0) * t1
    return out


# ---- h. interpolation of the log10 P table ------------------------------------------------------
def power_at(th, z_lim, lk, table, zq, k, eta0):
    """P(k, z_q) for arrays zq, k of equal length: linear in z between the bracketing Limber z
    nodes and linear in log10 k between the bracketing k nodes, both applied to log10 P (
    readings S5, S6); baryon template log10 P += -(eta0 - 0.7) 0.1 k^2/(k^2+1) (reading S21);
    P = 0 outside [k_min, k_max]."""
    zq = np.asarray(zq, np.float64)
    k = np.asarray(k, np.float64)
    inside = (k >= th.k_min) & (k <= th.k_max)
    dzl = z_lim[1] - z_lim[0]
    m = np.clip(np.floor(zq / dzl).astype(np.int64), 0, th.n_z - 2)
    t = (zq - z_lim[m]) / dzl
    dlk = lk[1] - lk[0]
    x = np.log10(np.where(inside, k, th.k_min))
    j = np.clip(np.floor((x - lk[0]) / dlk).astype(np.int64), 0, th.n_k - 2)
    s = (x - lk[j]) / dlk
    lo = (1.0 - t) * table[m, j] + t * table[m + 1, j]
    hi = (1.0 - t) * table[m, j + 1] + t * table[m + 1, j + 1]
    y = (1.0 - s) * lo + s * hi
    y = y - (eta0 - 0.7) * 0.1 * k * k / (k * k + 1.0)
    return np.where(inside, 10.0 ** y, 0.0)


def pair_index(n_tomo):
    return [(i, j) for i in range(n_tomo) for j in range(i, n_tomo)]


# ---- i, j. Limber sum ------------------------------------------------------------------------------
def limber_cl(th, chi, dchi, z_q, Wg, Wi, table, z_lim, lk, eta0):
    """eq. A2 on the quadrature nodes, the four terms of eq. A1 computed
    separately and summed. Wg, Wi: [n_tomo, n_chi]. Returns C [n_pairs, n_ell]."""
    pairs = pair_index(th.n_tomo)
    C = np.zeros((len(pairs), th.n_ell))
    for b in range(th.n_ell):
        ell = th.ell[b]
        P = power_at(th, z_lim, lk, table, z_q, (ell + 0.5) / chi, eta0)
        g = dchi / chi ** 2
        for p, (i, j) in enumerate(pairs):
            gg = np.sum(g * Wg[i] * Wg[j] * P)
            gi = np.sum(g * Wg[i] * Wi[j] * P)
            ig = np.sum(g * Wi[i] * Wg[j] * P)
            ii = np.sum(g * Wi[i] * Wi[j] * P)
            C[p, b] = gg + gi + ig + ii
    return C


def _bin_terms(theta, first, n_tomo, n_terms, n_max):
    """[n_tomo, n_max] coefficients, bin-major in theta with n_terms per bin, higher ones zero
    (n_terms = 1: the paper's single amplitude / bias per bin)."""
    out = np.zeros((n_tomo, n_max))
    for i in range(n_tomo):
        for t in range(n_terms):
            out[i, t] = theta[first + n_terms * i + t]
    return out


def physical_parameters(th, theta):
    """unpack one theta row by the parameter map (reading S2)."""
    g = lambda i, default: (float(theta[i]) if i >= 0 else default)
    ob, oc, h = g(th.idx_omega_b, 0.0), g(th.idx_omega_cdm, 0.0), g(th.idx_h, 1.0)
    nt = th.n_tomo
    return dict(Om=(ob + oc) / (h * h), w0=g(th.idx_w0, -1.0), wa=g(th.idx_wa, 0.0),
                eta0=g(th.idx_eta0, 0.7),
                dz=np.array([theta[th.idx_dz + i] for i in range(nt)], np.float64),
                A=_bin_terms(theta, th.idx_ia, nt, th.n_ia_terms, 3),
                m=_bin_terms(theta, th.idx_m, nt, th.n_m_terms, 2))


def emulator_inputs(th, theta, z_nodes):
    """rows (theta_emu..., z_m) for every emulator z node (step a2)."""
    base = np.array([float(theta[i]) if i >= 0 else float(c)
                     for i, c in zip(th.emu_in_idx, th.emu_in_const)], np.float64)
    X = np.empty((len(z_nodes), len(base) + 1))
    X[:, :-1] = base[None, :]
    X[:, -1] = z_nodes
    return X


def model_vector(th, theta, table_emu):
    """theta: one row; table_emu: log10 P on the emulator nodes [n_z_emu, n_k]. Returns model[n_data]."""
    p = physical_parameters(th, theta)
    z_emu, z_lim, lk = z_nodes_emulator(th), z_nodes_limber(th), log10k_nodes(th)
    a_q, z_q, da = quadrature_nodes(th)
    table = np.asarray(table_emu, np.float64)
    if th.z_interp == 2:      # k. cubic spline n_z_emu -> n_z nodes, per k
        table = notaknot_spline_eval(z_emu, table, z_lim)
    chi, dchi, D_q, E_q = background(a_q, z_q, da, p["Om"], p["w0"], p["wa"])
    Wg = np.empty((th.n_tomo, th.n_chi))
    Wi = np.empty((th.n_tomo, th.n_chi))
    for i in range(th.n_tomo):
        nz_q = n_of_z(z_q, th.nz_mean[i], th.nz_sigma, p["dz"][i])
        Wg[i] = window_gamma(a_q, z_q, da, chi, nz_q, p["Om"])
        Wi[i] = window_ia(z_q, nz_q, ia_amplitude(z_q, *p["A"][i]), p["Om"], D_q, E_q)
    C = limber_cl(th, chi, dchi, z_q, Wg, Wi, table, z_lim, lk, p["eta0"])
    out = np.empty(C.size)
    for pidx, (i, j) in enumerate(pair_index(th.n_tomo)):
        mi = m_bias(th.ell, p["m"][i, 0], p["m"][i, 1])
        mj = m_bias(th.ell, p["m"][j, 0], p["m"][j, 1])
        out[pidx * th.n_ell:(pidx + 1) * th.n_ell] = (1.0 + mi) * (1.0 + mj) * C[pidx]
    return out
