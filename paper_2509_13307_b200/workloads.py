"""Seeded synthetic workloads (inputs only) for the nsgpu hot path.

This module is the ONE piece shared by the CUDA path (`paper_2509_13307_b200.nsgpu`),
the oracle (`oracle/`) and the tests/bench.  It holds *no arithmetic of the method*:
it only draws seeded random weights, writes down grids/prior tables/parameter
layouts, and (given a model vector computed by whoever calls it) builds a synthetic
data vector, an SPD covariance and its Cholesky factor.  Neither `oracle/` nor the
CUDA binding is imported here.

Recipes follow SURVEY.md §8(c.3) readings E3/E4/S2/S3/S7/C2 and §8(d) (seeds 1000..1004);
shapes follow BASELINE.json configs[0..4].  The paper's trained CosmoPower weights,
mock data and LSST-like covariance are not available, so these
seeded stand-ins of the same shape are used everywhere.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field
from typing import List, Optional

import numpy as np

# theory kinds (mirrors include/nsgpu.h)
THEORY_IDENTITY = 0
THEORY_EMULATOR = 1
THEORY_CMB_BINNED = 2
THEORY_SHEAR_LIMBER = 3
THEORY_CMB_TT_CV = 4     # the paper's cosmic-variance TT likelihood: chi^2_{2l+1} per multipole

PRIOR_UNIFORM = 0
PRIOR_GAUSSIAN = 1

OUT_LINEAR = 0
OUT_EXP10 = 1

Z_INTERP_NONE = 0      # emulator z nodes are the Limber z nodes
Z_INTERP_CUBIC = 2     # cubic not-a-knot spline from n_z_emu nodes to n_z nodes


@dataclass
class Emulator:
    """One CosmoPower-style MLP: n_in -> n_hidden x width -> n_out (all arrays fp32)."""
    n_in: int
    n_hidden: int
    width: int
    n_out: int
    out_kind: int
    W: List[np.ndarray]        # n_hidden+1 matrices, row-major [fan_in, fan_out]; y = x.W + b
    b: List[np.ndarray]        # n_hidden+1 vectors [fan_out]
    alpha: List[np.ndarray]    # n_hidden vectors [width]
    beta: List[np.ndarray]     # n_hidden vectors [width]
    in_mean: np.ndarray
    in_std: np.ndarray
    out_mean: np.ndarray
    out_std: np.ndarray


@dataclass
class Theory:
    kind: int
    # emulator-input assembly: emulator input j (j < n_theta_in) is theta[emu_in_idx[j]]
    # or the constant emu_in_const[j] when emu_in_idx[j] < 0.  Shear emulators take one
    # more input (z, last) that the theory stage supplies per redshift node.
    emu_in_idx: np.ndarray = field(default_factory=lambda: np.zeros(0, np.int32))
    emu_in_const: np.ndarray = field(default_factory=lambda: np.zeros(0, np.float64))
    # --- cmb_binned ---
    bin_ptr: Optional[np.ndarray] = None    # int32 [n_data+1]
    bin_col: Optional[np.ndarray] = None    # int32 [nnz], columns in [0, n_spec*n_out)
    bin_val: Optional[np.ndarray] = None    # float32 [nnz]
    cal_index: int = -1
    # --- cmb_tt_cv ---
    ell_min: int = 2
    # --- shear_limber ---
    n_z_emu: int = 0
    n_z: int = 0
    n_chi: int = 0
    n_k: int = 0
    n_ell: int = 0
    n_tomo: int = 0
    z_interp: int = Z_INTERP_NONE
    z_max: float = 0.0
    k_min: float = 0.0
    k_max: float = 0.0
    ell: Optional[np.ndarray] = None        # float64 [n_ell]
    nz_mean: Optional[np.ndarray] = None    # float64 [n_tomo]
    nz_sigma: float = 0.0
    # positions in theta (or <0 with the constant used instead): physical parameters
    idx_omega_b: int = -1
    idx_omega_cdm: int = -1
    idx_h: int = -1
    idx_w0: int = -1      # <0 => w0 = -1
    idx_wa: int = -1      # <0 => wa = 0
    idx_eta0: int = -1
    idx_dz: int = -1      # first of n_tomo photo-z shifts
    idx_ia: int = -1      # first of n_ia_terms*n_tomo IA coefficients (A_{i,0..} bin-major)
    idx_m: int = -1       # first of n_m_terms*n_tomo shear-calibration coefficients (m_{i,0..} bin-major)
    n_ia_terms: int = 3   # 3, 2: BASELINE.json configs[2..4]; 1, 1: the paper's single amplitude and bias per bin
    n_m_terms: int = 2


@dataclass
class Workload:
    name: str
    seed: int
    D: int
    prior_kind: np.ndarray      # int32 [D]
    prior_p0: np.ndarray        # float64 [D]  (a | mu)
    prior_p1: np.ndarray        # float64 [D]  (b | sigma)
    emulators: List[Emulator]
    theory: Theory
    n_data: int
    u_fid: np.ndarray           # float64 [D] fiducial point in hypercube coordinates
    param_names: List[str]
    cov_frac: float = 0.05      # f of SURVEY §8(d): sigma_i = f*abs(d_i) + 1e-3*rms(d)
    data: Optional[np.ndarray] = None     # float64 [n_data]
    chol: Optional[np.ndarray] = None     # float64 [n_data, n_data] lower
    notes: str = ""


# ----------------------------------------------------------------------------------------
# emulator weights (reading E3)
# ----------------------------------------------------------------------------------------
def make_emulator(rng: np.random.Generator, n_in: int, n_hidden: int, width: int, n_out: int,
                  out_kind: int, in_mean, in_std, out_mean, out_std) -> Emulator:
    W, b, alpha, beta = [], [], [], []
    fan_in = n_in
    for _ in range(n_hidden):
        W.append((rng.standard_normal((fan_in, width)) * math.sqrt(2.0 / fan_in)).astype(np.float32))
        b.append((0.1 * rng.standard_normal(width)).astype(np.float32))
        alpha.append(rng.standard_normal(width).astype(np.float32))
        beta.append(rng.standard_normal(width).astype(np.float32))
        fan_in = width
    W.append((rng.standard_normal((fan_in, n_out)) * math.sqrt(2.0 / fan_in)).astype(np.float32))
    b.append((0.1 * rng.standard_normal(n_out)).astype(np.float32))
    f32 = lambda a: np.ascontiguousarray(np.asarray(a, dtype=np.float64).astype(np.float32))
    return Emulator(n_in, n_hidden, width, n_out, out_kind, W, b, alpha, beta,
                    f32(in_mean), f32(in_std), f32(out_mean), f32(out_std))


def _prior_arrays(rows):
    kind = np.array([r[0] for r in rows], np.int32)
    p0 = np.array([r[1] for r in rows], np.float64)
    p1 = np.array([r[2] for r in rows], np.float64)
    return kind, p0, p1


def _in_standardisation(rows):
    """mu_in = box centre / Gaussian mean; sigma_in = width/sqrt(12) / Gaussian sigma (E3)."""
    mu, sd = [], []
    for k, p0, p1 in rows:
        if k == PRIOR_UNIFORM:
            mu.append(0.5 * (p0 + p1)); sd.append((p1 - p0) / math.sqrt(12.0))
        else:
            mu.append(p0); sd.append(p1)
    return np.array(mu), np.array(sd)


def _std_normal_cdf(x: float) -> float:
    return 0.5 * (1.0 + math.erf(x / math.sqrt(2.0)))


def _u_of_theta(rows, theta):
    """hypercube image of a fiducial point; input bookkeeping only."""
    u = []
    for (k, p0, p1), t in zip(rows, theta):
        u.append((t - p0) / (p1 - p0) if k == PRIOR_UNIFORM else _std_normal_cdf((t - p0) / p1))
    return np.array(u, np.float64)


# ----------------------------------------------------------------------------------------
# c0: toy (BASELINE.json configs[0])
# ----------------------------------------------------------------------------------------
def toy(seed: int = 1000, D: int = 6, width: int = 128, n_out: int = 100, n_hidden: int = 4) -> Workload:
    rng = np.random.default_rng(seed)
    rows = [(PRIOR_UNIFORM, 0.0, 1.0)] * D
    kind, p0, p1 = _prior_arrays(rows)
    mu_in, sd_in = _in_standardisation(rows)
    emu = make_emulator(rng, D, n_hidden, width, n_out, OUT_LINEAR, mu_in, sd_in,
                        np.zeros(n_out), np.ones(n_out))
    th = Theory(kind=THEORY_EMULATOR, emu_in_idx=np.arange(D, dtype=np.int32),
                emu_in_const=np.zeros(D))
    return Workload("c0_toy", seed, D, kind, p0, p1, [emu], th, n_out,
                    np.full(D, 0.5), [f"x{i}" for i in range(D)],
                    notes="toy covariance C = A A^T + 0.1 I, A ~ N(0,1)/10")


def toy_identity(seed: int = 1000, D: int = 6, sigma: float = 0.04, rho_max: float = 0.6) -> Workload:
    """Identity theory: model = theta; correlated Gaussian with closed-form log Z (pin for NS)."""
    rng = np.random.default_rng(seed + 500)
    rows = [(PRIOR_UNIFORM, 0.0, 1.0)] * D
    kind, p0, p1 = _prior_arrays(rows)
    G = rng.standard_normal((D, 3 * D))
    R = G @ G.T
    dd = np.sqrt(np.diag(R))
    R = R / dd[:, None] / dd[None, :]
    off = R - np.eye(D)
    m = np.abs(off).max()
    if m > rho_max:
        off *= rho_max / m
    R = np.eye(D) + off
    C = (sigma ** 2) * R
    wl = Workload("c0_identity", seed, D, kind, p0, p1, [], Theory(kind=THEORY_IDENTITY), D,
                  np.full(D, 0.5), [f"x{i}" for i in range(D)])
    wl.data = np.full(D, 0.5)
    wl.chol = np.linalg.cholesky(C)
    return wl


def attach_toy_data(wl: Workload, model_fid: np.ndarray) -> Workload:
    """c0: d = model(theta_0) + L eps; C = A A^T + 0.1 I, A ~ N(0,1)/10."""
    rng = np.random.default_rng(wl.seed + 77)
    n = wl.n_data
    A = rng.standard_normal((n, n)) / 10.0
    C = A @ A.T + 0.1 * np.eye(n)
    L = np.linalg.cholesky(C)
    wl.chol = L
    wl.data = np.asarray(model_fid, np.float64) + L @ rng.standard_normal(n)
    return wl


def attach_data(wl: Workload, model_fid: np.ndarray, noise: bool = True) -> Workload:
    """c1..c4: C = S rho S, S = diag(f abs(d_i) + 1e-3 rms(d)), rho = normalise(G G^T/n + I)."""
    rng = np.random.default_rng(wl.seed + 77)
    n = wl.n_data
    d0 = np.asarray(model_fid, np.float64)
    assert d0.shape == (n,)
    s = wl.cov_frac * np.abs(d0) + 1e-3 * math.sqrt(float(np.mean(d0 ** 2)))
    G = rng.standard_normal((n, n))
    rho = G @ G.T / n + np.eye(n)
    dd = np.sqrt(np.diag(rho))
    rho = rho / dd[:, None] / dd[None, :]
    C = s[:, None] * rho * s[None, :]
    L = np.linalg.cholesky(C)
    eps = rng.standard_normal(n)
    wl.chol = L
    wl.data = d0 + (L @ eps if noise else 0.0)
    return wl


# ----------------------------------------------------------------------------------------
# c1: CMB-like (BASELINE.json configs[1]; readings C1-C4, E4)
# ----------------------------------------------------------------------------------------
def _contiguous_bins(lo: int, hi: int, n_bins: int):
    """n_bins contiguous near-equal-width bins covering integers lo..hi inclusive."""
    edges = np.floor(lo + (hi + 1 - lo) * np.arange(n_bins + 1) / n_bins + 1e-9).astype(np.int64)
    edges[-1] = hi + 1
    return edges


def cmb(seed: int = 1001, width: int = 512, n_hidden: int = 4, ell_max: int = 2508,
        n_bins=(215, 199, 199), ell_bin_lo: int = 30, ell_bin_hi=(2508, 1996, 1996)) -> Workload:
    rng = np.random.default_rng(seed)
    rows = [(PRIOR_UNIFORM, 0.01875, 0.02625),   # omega_b
            (PRIOR_UNIFORM, 0.05, 0.255),        # omega_cdm (L81)
            (PRIOR_UNIFORM, 0.64, 0.982),        # h         (L82)
            (PRIOR_UNIFORM, 0.01, 0.15),         # tau       (reading C4)
            (PRIOR_UNIFORM, 0.84, 1.1),          # n_s       (L83)
            (PRIOR_UNIFORM, 1.61, 3.91),         # ln10^10As (L84)
            (PRIOR_GAUSSIAN, 1.0, 0.0025)]       # A_cal     (reading C3)
    names = ["omega_b", "omega_cdm", "h", "tau", "n_s", "lnAs", "A_cal"]
    D = len(rows)
    kind, p0, p1 = _prior_arrays(rows)
    mu_in, sd_in = _in_standardisation(rows)
    n_out = ell_max - 1                       # ell = 2..ell_max
    ell = np.arange(2, ell_max + 1, dtype=np.float64)
    base = -9.0 - 2.0 * np.log10(np.maximum(ell, 100.0) / 100.0)
    emus = []
    for spec in ("TT", "TE", "EE"):
        if spec == "TE":
            emus.append(make_emulator(rng, D, n_hidden, width, n_out, OUT_LINEAR, mu_in, sd_in,
                                      np.zeros(n_out), np.full(n_out, 1e-11)))
        else:
            mu_out = base - (1.0 if spec == "EE" else 0.0)
            emus.append(make_emulator(rng, D, n_hidden, width, n_out, OUT_EXP10, mu_in, sd_in,
                                      mu_out, np.full(n_out, 0.1)))
    ptr, col, val = [0], [], []
    for s, (nb, hi) in enumerate(zip(n_bins, ell_bin_hi)):
        edges = _contiguous_bins(ell_bin_lo, min(hi, ell_max), nb)
        for b in range(nb):
            ls = np.arange(edges[b], edges[b + 1])
            col.extend((s * n_out + (ls - 2)).tolist())
            val.extend([1.0 / len(ls)] * len(ls))
            ptr.append(len(col))
    n_data = len(ptr) - 1
    th = Theory(kind=THEORY_CMB_BINNED, emu_in_idx=np.arange(D, dtype=np.int32),
                emu_in_const=np.zeros(D),
                bin_ptr=np.array(ptr, np.int32), bin_col=np.array(col, np.int32),
                bin_val=np.array(val, np.float32), cal_index=D - 1)
    theta_fid = [0.02242, 0.11933, 0.6766, 0.0544, 0.9665, 3.047, 1.0]
    return Workload("c1_cmb", seed, D, kind, p0, p1, emus, th, n_data,
                    _u_of_theta(rows, theta_fid), names)


def cmb_tt(seed: int = 1005, width: int = 512, n_hidden: int = 4, ell_max: int = 2508) -> Workload:
    """The paper's CMB run: 6 cosmological parameters on the Table-1 box (tau per reading
    C4), one TT emulator 6 -> 4 x 512 -> 2507 (l = 2..2508), cosmic-variance likelihood, no covariance.
    `chol` stays None; `data` = observed C_l (attach_cmb_tt_data)."""
    rng = np.random.default_rng(seed)
    rows = [(PRIOR_UNIFORM, 0.01875, 0.02625), (PRIOR_UNIFORM, 0.05, 0.255), (PRIOR_UNIFORM, 0.64, 0.982),
            (PRIOR_UNIFORM, 0.01, 0.15), (PRIOR_UNIFORM, 0.84, 1.1), (PRIOR_UNIFORM, 1.61, 3.91)]
    names = ["omega_b", "omega_cdm", "h", "tau", "n_s", "lnAs"]
    D = len(rows)
    kind, p0, p1 = _prior_arrays(rows)
    mu_in, sd_in = _in_standardisation(rows)
    n_out = ell_max - 1
    ell = np.arange(2, ell_max + 1, dtype=np.float64)
    mu_out = -9.0 - 2.0 * np.log10(np.maximum(ell, 100.0) / 100.0)
    # a cosmic-variance likelihood over 2507 multipoles is razor sharp: sigma_out = 0.01 keeps the synthetic
    # posterior a finite fraction of the prior box (random weights have no physical smoothness in l)
    emu = make_emulator(rng, D, n_hidden, width, n_out, OUT_EXP10, mu_in, sd_in, mu_out, np.full(n_out, 0.01))
    th = Theory(kind=THEORY_CMB_TT_CV, emu_in_idx=np.arange(D, dtype=np.int32), emu_in_const=np.zeros(D), ell_min=2)
    theta_fid = [0.02242, 0.11933, 0.6766, 0.0544, 0.9665, 3.047]
    return Workload("cmb_tt_cv", seed, D, kind, p0, p1, [emu], th, n_out, _u_of_theta(rows, theta_fid), names)


def attach_cmb_tt_data(wl: Workload, model_fid: np.ndarray, noise: bool = True) -> Workload:
    """observed spectrum: C_l(theta_0) x chi^2_{2l+1} / (2l+1) (a cosmic-variance draw), or noise-free."""
    rng = np.random.default_rng(wl.seed + 77)
    nu = 2.0 * (wl.theory.ell_min + np.arange(wl.n_data)) + 1.0
    c0 = np.asarray(model_fid, np.float64)
    wl.data = c0 * (rng.chisquare(nu) / nu if noise else 1.0)
    wl.chol = None
    return wl


# ----------------------------------------------------------------------------------------
# c2/c3/c4: cosmic shear (BASELINE.json configs[2..4]; readings S1-S21)
# ----------------------------------------------------------------------------------------
def shear(seed: int = 1002, w0wa: bool = False, fix_w0wa: bool = False, n_z_emu: int = 50,
          n_z: int = 50, width: int = 512, n_hidden: int = 4, n_k: int = 420, n_chi: int = 100,
          n_ell: int = 20, n_tomo: int = 5, name: Optional[str] = None, z_max: float = 2.0,
          n_ia_terms: int = 3, n_m_terms: int = 2, de_table1: bool = False) -> Workload:
    """theta layout (reading S2):
    [omega_b, omega_cdm, h, n_s, lnAs, c_min, (w0, wa,) eta_0, dz_0.., A_{i,0..2} (bin-major), m_{i,0..1}].
    `w0wa` adds w0, wa as sampled parameters; `fix_w0wa` builds the 9-input emulator of the
    w0wa model but pins w0 = -1, wa = 0 as constants (the LambdaCDM restriction of c4)."""
    rng = np.random.default_rng(seed)
    cosmo_rows = [(PRIOR_UNIFORM, 0.01875, 0.02625), (PRIOR_UNIFORM, 0.05, 0.255),
                  (PRIOR_UNIFORM, 0.64, 0.982), (PRIOR_UNIFORM, 0.84, 1.1),
                  (PRIOR_UNIFORM, 1.61, 3.91), (PRIOR_UNIFORM, 2.0, 4.0)]
    cosmo_names = ["omega_b", "omega_cdm", "h", "n_s", "lnAs", "c_min"]
    cosmo_fid = [0.02242, 0.11933, 0.6766, 0.9665, 3.047, 2.6]
    de_rows = [(PRIOR_UNIFORM, -3.0, 1.0), (PRIOR_UNIFORM, -3.0, 2.0)]   # reading S14 (BJ cfg 3)
    if de_table1:                                                       # the paper's own ranges (Table 1)
        de_rows = [(PRIOR_UNIFORM, -1.5, -0.5), (PRIOR_UNIFORM, -0.5, 0.5)]
    emu_rows = list(cosmo_rows) + (de_rows if (w0wa or fix_w0wa) else [])
    rows, names, fid = list(cosmo_rows), list(cosmo_names), list(cosmo_fid)
    if w0wa:
        rows += de_rows; names += ["w0", "wa"]; fid += [-1.0, 0.0]
    idx_eta0 = len(rows)
    rows.append((PRIOR_UNIFORM, 0.5, 1.0)); names.append("eta_0"); fid.append(0.7)
    idx_dz = len(rows)
    for i in range(n_tomo):
        rows.append((PRIOR_GAUSSIAN, 0.0, 0.01)); names.append(f"dz_{i}"); fid.append(0.0)
    idx_ia = len(rows)
    for i in range(n_tomo):
        for t in range(n_ia_terms):
            rows.append((PRIOR_UNIFORM, -6.0, 6.0)); names.append(f"A_{i}_{t}")
            fid.append(1.0 - 0.1 * (i + 1) if t == 0 else 0.0)
    idx_m = len(rows)
    for i in range(n_tomo):
        rows.append((PRIOR_GAUSSIAN, 0.01, 0.02)); names.append(f"m_{i}_0"); fid.append(0.01)
        if n_m_terms > 1:
            rows.append((PRIOR_GAUSSIAN, 0.0, 0.02)); names.append(f"m_{i}_1"); fid.append(0.0)
    D = len(rows)
    kind, p0, p1 = _prior_arrays(rows)
    mu_in, sd_in = _in_standardisation(emu_rows + [(PRIOR_UNIFORM, 0.0, z_max)])
    k_min, k_max = 1e-4, 50.0
    lk = np.linspace(math.log10(k_min), math.log10(k_max), n_k)
    mu_out = 4.3 - 1.2 * (lk + 1.7) ** 2 / (1.0 + 0.35 * np.abs(lk + 1.7))
    n_theta_in = len(emu_rows)
    emu = make_emulator(rng, n_theta_in + 1, n_hidden, width, n_k, OUT_EXP10, mu_in, sd_in,
                        mu_out, np.full(n_k, 0.15))
    emu_in_idx = np.arange(n_theta_in, dtype=np.int32)
    emu_in_const = np.zeros(n_theta_in)
    if fix_w0wa and not w0wa:
        emu_in_idx[6:8] = -1
        emu_in_const[6:8] = (-1.0, 0.0)
    ell = 100.0 * 30.0 ** ((np.arange(n_ell) + 0.5) / n_ell)
    nz_mean = 0.3 + 0.225 * np.arange(n_tomo) * (4.0 / max(n_tomo - 1, 1))
    th = Theory(kind=THEORY_SHEAR_LIMBER, emu_in_idx=emu_in_idx, emu_in_const=emu_in_const,
                n_z_emu=n_z_emu, n_z=n_z, n_chi=n_chi, n_k=n_k, n_ell=n_ell, n_tomo=n_tomo,
                z_interp=(Z_INTERP_NONE if n_z_emu == n_z else Z_INTERP_CUBIC),
                z_max=z_max, k_min=k_min, k_max=k_max, ell=ell, nz_mean=nz_mean, nz_sigma=0.1,
                idx_omega_b=0, idx_omega_cdm=1, idx_h=2,
                idx_w0=(6 if w0wa else -1), idx_wa=(7 if w0wa else -1),
                idx_eta0=idx_eta0, idx_dz=idx_dz, idx_ia=idx_ia, idx_m=idx_m,
                n_ia_terms=n_ia_terms, n_m_terms=n_m_terms)
    n_pairs = n_tomo * (n_tomo + 1) // 2
    if name is None:
        name = "shear_w0wa" if w0wa else ("shear_lcdm_restricted" if fix_w0wa else "shear_lcdm")
    return Workload(name, seed, D, kind, p0, p1, [emu], th, n_pairs * n_ell,
                    _u_of_theta(rows, fid), names)


def c2() -> Workload:
    return shear(seed=1002, name="c2_shear_lcdm_37d")


def c3a() -> Workload:
    return shear(seed=1003, w0wa=True, name="c3a_shear_w0wa_39d_50z")


def c3b() -> Workload:
    return shear(seed=1003, w0wa=True, n_z_emu=12, n_z=50, name="c3b_shear_w0wa_39d_12z_spline")


def c4_lcdm() -> Workload:
    """LambdaCDM restriction of c3a: same 9-input emulator weights, w0 = -1, wa = 0 pinned."""
    return shear(seed=1003, fix_w0wa=True, name="c4_shear_lcdm_37d_restricted")


def c5(interpolated: bool = True, w0wa: bool = True) -> Workload:
    """Paper-shape shear: 10 tomographic bins (55 spectra), one
    A_IA, m and D_z per bin (37/39-D), the priors of Table 1 including w0 in U(-1.5, -0.5) and wa in
    U(-0.5, 0.5) -- NOT BASELINE.json's wider cfg-3 ranges --, 1025 quadrature nodes evenly spaced in the scale factor
    down to z = 5.02; emulator at 1025 z nodes, or (`interpolated`, the paper's Shear (I)) on a 10x coarser grid of 103
    nodes followed by linear interpolation in z.  Deviations from the paper that remain: eta_0 is not an emulator input
    but acts through the synthetic baryon template of reading S21 (prior U(0.5, 1), Table 1), the n_i(z) are ten
    Gaussians (reading S25), weights, mock data and covariance are synthetic -- so evidences and evaluation counts of
    c5 runs describe a problem of the paper's shape, not the paper's problem."""
    nz = 103 if interpolated else 1025
    return shear(seed=1006, w0wa=w0wa, fix_w0wa=not w0wa, n_z_emu=nz, n_z=nz, n_chi=1025, n_tomo=10, z_max=5.02,
                 n_ia_terms=1, n_m_terms=1, de_table1=True,
                 name=("c5i" if interpolated else "c5") + "_shear_paper_shape_" + ("39d" if w0wa else "37d"))


def tiny_shear_paper(seed: int = 9) -> Workload:
    """Small workload with the paper-shape parameter layout (one A_IA and m per bin) and a quadrature grid
    longer than one chunk of the projection kernel."""
    return shear(seed=seed, w0wa=True, n_z_emu=17, n_z=17, width=48, n_hidden=2, n_k=37, n_chi=301, n_ell=7,
                 n_tomo=4, z_max=5.02, n_ia_terms=1, n_m_terms=1, name="tiny_shear_paper")


def tiny_shear(seed: int = 7, w0wa: bool = True, spline: bool = False) -> Workload:
    """Small ragged shear workload for fast parity tests (not a BASELINE config)."""
    return shear(seed=seed, w0wa=w0wa, n_z_emu=(5 if spline else 9), n_z=9, width=48, n_hidden=2,
                 n_k=37, n_chi=23, n_ell=6, n_tomo=3, name="tiny_shear" + ("_spline" if spline else ""))


def tiny_cmb(seed: int = 8) -> Workload:
    return cmb(seed=seed, width=40, n_hidden=2, ell_max=131, n_bins=(9, 7, 7), ell_bin_lo=30,
               ell_bin_hi=(131, 100, 100))


# ----------------------------------------------------------------------------------------
# test point sets in hypercube coordinates (S_prior, S_post)
# ----------------------------------------------------------------------------------------
def u_prior_set(wl: Workload, n: int, seed: int = 0) -> np.ndarray:
    rng = np.random.default_rng(wl.seed * 1000 + 11 + seed)
    return rng.random((n, wl.D))


def u_post_set(wl: Workload, n: int, seed: int = 0, scale: float = 0.005) -> np.ndarray:
    rng = np.random.default_rng(wl.seed * 1000 + 13 + seed)
    u = wl.u_fid[None, :] + scale * rng.standard_normal((n, wl.D))
    return np.clip(u, 1e-6, 1.0 - 1e-6)
