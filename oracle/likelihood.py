"""log L(theta) for a whole batch: emulator -> theory -> Gaussian chi^2 (the bulk likelihood
evaluation the paper calls the primary bottleneck; steps a2-a10)."""
import numpy as np

from . import cmb, cmb_tt, emulator, gaussian, prior, shear

IDENTITY, EMULATOR, CMB_BINNED, SHEAR_LIMBER, CMB_TT_CV = 0, 1, 2, 3, 4


def _emu_theta_inputs(th, theta):
    return np.array([[float(t[i]) if i >= 0 else float(c) for i, c in zip(th.emu_in_idx, th.emu_in_const)]
                     for t in theta], np.float64)


def emulate(wl, theta, which=0):
    """Emulated spectra (debug tap `nsgpu_emulate_batch`): [B, rows, n_out]; rows = n_z_emu for
    shear (one row per emulator redshift node), 1 otherwise. exp10 applied where out_kind = 1."""
    th, emu = wl.theory, wl.emulators[which]
    theta = np.asarray(theta, np.float64)
    if th.kind == SHEAR_LIMBER:
        z = shear.z_nodes_emulator(th)
        X = np.concatenate([shear.emulator_inputs(th, t, z) for t in theta], axis=0)
        return emulator.mlp_forward(emu, X).reshape(len(theta), len(z), emu.n_out)
    return emulator.mlp_forward(emu, _emu_theta_inputs(th, theta))[:, None, :]


def theory(wl, theta):
    """model vectors [B, n_data] (debug tap `nsgpu_theory_batch`)."""
    th = wl.theory
    theta = np.asarray(theta, np.float64)
    B = len(theta)
    if th.kind == IDENTITY:
        return theta.copy()
    if th.kind in (EMULATOR, CMB_TT_CV):
        return emulator.mlp_forward(wl.emulators[0], _emu_theta_inputs(th, theta))
    if th.kind == CMB_BINNED:
        X = _emu_theta_inputs(th, theta)
        spectra = [emulator.mlp_forward(e, X) for e in wl.emulators]
        return np.stack([cmb.model_vector(th, theta[b], [s[b] for s in spectra]) for b in range(B)])
    if th.kind == SHEAR_LIMBER:
        z = shear.z_nodes_emulator(th)
        X = np.concatenate([shear.emulator_inputs(th, t, z) for t in theta], axis=0)
        tables = emulator.mlp_raw(wl.emulators[0], X).reshape(B, len(z), th.n_k)      # log10 P(k, z_m)
        return np.stack([shear.model_vector(th, theta[b], tables[b]) for b in range(B)])
    raise ValueError(th.kind)


def loglike(wl, theta):
    """log L [B] in fp64; -inf outside the support of the uniform priors or for non-finite models."""
    theta = np.asarray(theta, np.float64)
    ok = prior.in_support(wl.prior_kind, wl.prior_p0, wl.prior_p1, theta)
    out = np.full(len(theta), -np.inf)
    if np.any(ok):
        model = theory(wl, theta[ok])
        if wl.theory.kind == CMB_TT_CV:      # per-multipole chi^2_{2l+1} likelihood, no covariance
            ll = cmb_tt.loglike_spectrum(cmb_tt.ells(wl.theory, wl.n_data), wl.data, model)
        else:
            ll = gaussian.loglike(wl.chol, model, wl.data)
        ll[~np.isfinite(ll)] = -np.inf
        out[ok] = ll
    return out


def loglike_u(wl, u):
    """log L as a function of hypercube coordinates (what the sampler sees)."""
    return loglike(wl, prior.transform(wl.prior_kind, wl.prior_p0, wl.prior_p1, u))
