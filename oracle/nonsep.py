"""Float64 CPU ORACLE of the NON-SEPARABLE weight model.

TEST INFRASTRUCTURE ONLY (same rules as `oracle/sps_model.py`; shares no code with the CUDA path).

PAPER.md:52 (section 2): "alternative SED models that relax the assumption of separability; for example ... models in
which the metallicity distribution function varies with stellar age in accord with the time evolution of the MZR", and
PAPER.md:378 (App. A.2): "variations in which stellar age is correlated with metallicity".  The paper gives no formula;
the reading (R26; the functional form itself is parity unpinned) is the lognormal MDF of A.2 with a median that
drifts linearly with log age,
    P_SSP(i, j) = a_i m_ij,   m_ij = Phi((g_{j+1} - mu_i)/sigma) - Phi((g_j - mu_i)/sigma),
    mu_i = logZ + gamma (log10 age_i/yr - 9),
with gamma (`dlogZ_dlogage`, dex per dex; negative = older stars are metal-poorer) a constant of the table, not a sampled
parameter, so the 13-parameter vector and Eq. (1), (4), (6) are unchanged; Eq. (2) is replaced by the full
[n_age, n_Z] array.  gamma = 0 is the separable model.
"""
from __future__ import annotations

import math

import numpy as np

from . import sps_model as M


def met_weights_by_age(logZ, sigma_logZ, log10_Z, log10_age_yr, gamma):
    """m [B,n_age,n_Z] and its partials with respect to logZ and sigma_logZ (R9 discretisation per age bin)."""
    la = np.asarray(log10_age_yr, float)
    out = [M.met_weights(np.asarray(logZ, float) + gamma * (la[i] - 9.0), sigma_logZ, log10_Z) for i in range(len(la))]
    return tuple(np.stack([o[k] for o in out], axis=1) for k in range(3))


def ssp_weights(theta, grid, gamma):
    """w [B,n_age,n_Z] = Mn a_i m_ij (Eq. 1 with the non-separable P_SSP) and dw/dtheta [B,n_age,n_Z,13]."""
    th = np.asarray(theta, float)
    W = M.weights(th, grid)
    m, dm_lz, dm_s = met_weights_by_age(th[:, M.I_LZ], th[:, M.I_SLZ], grid.log10_Z, grid.log10_age_yr, gamma)
    a, Mn = W["a"], W["Mn"]
    w = Mn[:, None, None] * a[:, :, None] * m
    dw = (W["JMn"][:, None, None, :] * (a[:, :, None] * m)[..., None]
          + Mn[:, None, None, None] * W["Ja"][:, :, None, :] * m[..., None])
    dw[..., M.I_LZ] += Mn[:, None, None] * a[:, :, None] * dm_lz
    dw[..., M.I_SLZ] += Mn[:, None, None] * a[:, :, None] * dm_s
    return w, dw, m


def photometry_exact(theta, grid, gamma, want_jac=True):
    """Eq. (4) with w_ij = Mn a_i m_ij."""
    th = np.asarray(theta, float)
    w, dw, _ = ssp_weights(th, grid, gamma)
    B = th.shape[0]
    L = np.asarray(grid.ssp, float)
    lam = np.asarray(grid.wave_A, float)
    dlam = M.trapezoid_weights(lam)
    n_band = M.n_bands(grid)
    flux = np.zeros((B, n_band)); J = np.zeros((B, n_band, M.NDIM))
    for r in range(B):
        S = w[r].reshape(-1) @ L
        z = th[r, M.I_Z]
        F, F_av, F_del, F_fl, _ = M.attenuation(lam, th[r, M.I_AV], th[r, M.I_DEL], th[r, M.I_FFL])
        T, dT = M.band_T(grid, lam * (1.0 + z))
        flux[r] = (T * (S * F * dlam)[None, :]).sum(1)
        if not want_jac:
            continue
        dS = dw[r].reshape(-1, M.NDIM).T @ L
        J[r] = np.einsum("bk,pk->bp", T * (F * dlam)[None, :], dS)
        J[r, :, M.I_AV] += (T * (S * F_av * dlam)[None, :]).sum(1)
        J[r, :, M.I_DEL] += (T * (S * F_del * dlam)[None, :]).sum(1)
        J[r, :, M.I_FFL] += (T * (S * F_fl * dlam)[None, :]).sum(1)
        J[r, :, M.I_Z] += (dT * (lam * S * F * dlam)[None, :]).sum(1)
    return flux, J


def photometry_approx(theta, grid, gamma, cssp, lam_eff_obs=None):
    """Eq. (6) with w_ij = Mn a_i m_ij."""
    th = np.asarray(theta, float)
    w, dw, _ = ssp_weights(th, grid, gamma)
    B = th.shape[0]
    if lam_eff_obs is None:
        lam_eff_obs = M.band_effective_wavelength(grid)
    n_band = M.n_bands(grid)
    n_age, n_Z = len(grid.log10_age_yr), len(grid.log10_Z)
    dz = (grid.z_max - grid.z_min) / (grid.n_z - 1)
    flux = np.zeros((B, n_band)); J = np.zeros((B, n_band, M.NDIM))
    for r in range(B):
        z = th[r, M.I_Z]
        t = int(min(max(math.floor((z - grid.z_min) / dz), 0), grid.n_z - 2))
        f = (z - (grid.z_min + t * dz)) / dz
        c = ((1.0 - f) * cssp[t] + f * cssp[t + 1]).reshape(n_age, n_Z, n_band)
        dc = ((cssp[t + 1] - cssp[t]) / dz).reshape(n_age, n_Z, n_band)
        lam_r = lam_eff_obs / (1.0 + z)
        F, F_av, F_del, F_fl, F_lam = M.attenuation(lam_r, th[r, M.I_AV], th[r, M.I_DEL], th[r, M.I_FFL])
        S = np.einsum("ij,ijb->b", w[r], c)
        flux[r] = F * S
        J[r] = F[:, None] * np.einsum("ijp,ijb->bp", dw[r], c)
        J[r, :, M.I_AV] += F_av * S
        J[r, :, M.I_DEL] += F_del * S
        J[r, :, M.I_FFL] += F_fl * S
        J[r, :, M.I_Z] += F * np.einsum("ij,ijb->b", w[r], dc) + S * F_lam * (-lam_r / (1.0 + z))
    return flux, J


def logp_and_grad(theta_unb, grid, gamma, prior, obs_flux, obs_sigma, path, cssp=None):
    thu = np.asarray(theta_unb, float)
    th, dth = M.bound(thu, prior)
    flux, J = photometry_exact(th, grid, gamma) if path == "exact" else photometry_approx(th, grid, gamma, cssp)
    r = (flux - obs_flux) / obs_sigma
    lp_prior, dlp = M.log_skew_normal(thu, prior)
    return -0.5 * (r * r).sum(1) + lp_prior.sum(1), np.einsum("rb,rbp->rp", -r / obs_sigma, J) * dth + dlp, flux
