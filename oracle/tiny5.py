"""Float64 CPU ORACLE of `SPS_MODEL_TINY5`: the 5-parameter model of BASELINE.json configs[0].

TEST INFRASTRUCTURE ONLY (same rules as `oracle/sps_model.py`; shares no code with the CUDA path).

This model is BASELINE.json's, not the paper's (reading R19): "5 params (logM*,
log tau delayed-exp SFH, logZ, dust tau_V, fixed z=0.5)".  Parameter order of a row:
    logM_star, log10 tau [Gyr], logZ, tau_V   (D = 4 sampled)   and   z   (data, not sampled)
  * SFH: SFR(t) proportional to (t/tau^2) exp(-t/tau), scaled so that the mass formed by t_obs is 10^logM_star;
    age bins (R5 edges) by the closed form  int t e^{-t/tau} dt = -tau (t + tau) e^{-t/tau};
  * MDF: the lognormal of PAPER.md:378 (R9) with fixed scatter sigma_logZ = 0.2;
  * dust: F_att(lambda) = exp(-tau_V (lambda / 5500 A)^-0.7)   (a power-law screen; no floor, no bump);
  * no burst; photometry by Eq. (4) (exact) or Eq. (6) (approximate) exactly as in the 13-parameter model.
Which dust law and which fixed scatter BASELINE.json means is not stated: parity unpinned (R19); everything else
is pinned in tests/test_oracle_tiny5.py.
"""
from __future__ import annotations

import math

import numpy as np

from . import sps_model as M

ND = 4
I_LOGM, I_LTAU, I_LZ, I_TAUV = range(4)
SIGMA_LOGZ = 0.2
DUST_SLOPE = -0.7


def gamma2_cdf(t, tau):
    """G(t) = int_0^t (s/tau^2) e^{-s/tau} ds = 1 - (1 + t/tau) e^{-t/tau}   (from -tau (t+tau) e^{-t/tau} / tau^2),
    and its partials dG/dt = (t/tau^2) e^{-t/tau},  dG/dtau = -(t^2/tau^3) e^{-t/tau}."""
    x = t / tau
    e = np.exp(-x)
    return 1.0 - (1.0 + x) * e, x / tau * e, -x * x / tau * e


def weights(theta, z, grid):
    """theta [B,4] bounded, z [B].  Returns dict a [B,n_age], m [B,n_Z], Mn [B] and the Jacobians
    Ja [B,n_age,4], Jm [B,n_Z,4], JMn [B,4] with respect to (logM, log10 tau, logZ, tau_V)."""
    th = np.asarray(theta, float); z = np.asarray(z, float)
    B = th.shape[0]
    t_obs, _ = M.cosmic_time(z, grid.H0, grid.Om)
    tau = 10.0 ** th[:, I_LTAU]
    A, _ = M.age_bin_edges_gyr(grid.log10_age_yr)
    t_hi = np.maximum(0.0, t_obs[:, None] - A[None, :-1])          # R5: bins older than t_obs clip to zero
    t_lo = np.maximum(0.0, t_obs[:, None] - A[None, 1:])           # the last upper edge is +inf
    G_hi, _, Gt_hi = gamma2_cdf(t_hi, tau[:, None])
    G_lo, _, Gt_lo = gamma2_cdf(t_lo, tau[:, None])
    G_obs, _, Gt_obs = gamma2_cdf(t_obs, tau)
    a = (G_hi - G_lo) / G_obs[:, None]                             # mass fraction formed in each age bin
    da_dtau = (Gt_hi - Gt_lo) / G_obs[:, None] - a * (Gt_obs / G_obs)[:, None]
    m, dm_lz, _ = M.met_weights(th[:, I_LZ], np.full(B, SIGMA_LOGZ), grid.log10_Z)
    Mn = 10.0 ** (th[:, I_LOGM] - grid.log10_mass_unit)            # total formed mass by t_obs, in mass units
    Ja = np.zeros((B, a.shape[1], ND)); Jm = np.zeros((B, m.shape[1], ND)); JMn = np.zeros((B, ND))
    Ja[:, :, I_LTAU] = da_dtau * (tau * math.log(10.0))[:, None]
    Jm[:, :, I_LZ] = dm_lz
    JMn[:, I_LOGM] = math.log(10.0) * Mn
    return dict(a=a, m=m, Mn=Mn, Ja=Ja, Jm=Jm, JMn=JMn, t_obs=t_obs)


def attenuation(lam_A, tau_V):
    """F_att = exp(-tau_V (lambda/5500)^-0.7) and dF/dtau_V."""
    r = (np.asarray(lam_A, float) / M.LAMBDA_V) ** DUST_SLOPE
    F = np.exp(-tau_V * r)
    return F, -r * F


def photometry_exact(theta, z, grid, want_jac=True):
    """Eq. (4) (R1, R3, R4) with this model's weights and dust.  flux [B,n_band], J [B,n_band,4]."""
    th = np.asarray(theta, float); z = np.asarray(z, float)
    W = weights(th, z, grid)
    B = th.shape[0]
    L = np.asarray(grid.ssp, float)
    lam = np.asarray(grid.wave_A, float)
    dlam = M.trapezoid_weights(lam)
    n_band = M.n_bands(grid)
    flux = np.zeros((B, n_band)); J = np.zeros((B, n_band, ND))
    for r in range(B):
        a, m, Mn = W["a"][r], W["m"][r], W["Mn"][r]
        w = Mn * np.outer(a, m).reshape(-1)
        S = w @ L
        F, F_tv = attenuation(lam, th[r, I_TAUV])
        T, _ = M.band_T(grid, lam * (1.0 + z[r]))
        flux[r] = (T * (S * F * dlam)[None, :]).sum(1)
        if not want_jac:
            continue
        dw = (W["JMn"][r][None, None, :] * np.outer(a, m)[:, :, None]
              + Mn * W["Ja"][r][:, None, :] * m[None, :, None]
              + Mn * a[:, None, None] * W["Jm"][r][None, :, :]).reshape(-1, ND)
        dS = dw.T @ L
        J[r] = np.einsum("bk,pk->bp", T * (F * dlam)[None, :], dS)
        J[r, :, I_TAUV] += (T * (S * F_tv * dlam)[None, :]).sum(1)
    return flux, J


def photometry_approx(theta, z, grid, cssp, lam_eff_obs=None):
    """Eq. (6) with this model's weights and dust; c_SSP interpolated linearly in z."""
    th = np.asarray(theta, float); z = np.asarray(z, float)
    W = weights(th, z, grid)
    B = th.shape[0]
    if lam_eff_obs is None:
        lam_eff_obs = M.band_effective_wavelength(grid)
    n_band = M.n_bands(grid)
    n_age, n_Z = len(grid.log10_age_yr), len(grid.log10_Z)
    dz = (grid.z_max - grid.z_min) / (grid.n_z - 1)
    flux = np.zeros((B, n_band)); J = np.zeros((B, n_band, ND))
    for r in range(B):
        t = int(min(max(math.floor((z[r] - grid.z_min) / dz), 0), grid.n_z - 2))
        f = (z[r] - (grid.z_min + t * dz)) / dz
        c = ((1.0 - f) * cssp[t] + f * cssp[t + 1]).reshape(n_age, n_Z, n_band)
        a, m, Mn = W["a"][r], W["m"][r], W["Mn"][r]
        F, F_tv = attenuation(lam_eff_obs / (1.0 + z[r]), th[r, I_TAUV])
        S = Mn * np.einsum("i,j,ijb->b", a, m, c)
        flux[r] = F * S
        dS = (W["JMn"][r][None, :] * np.einsum("i,j,ijb->b", a, m, c)[:, None]
              + Mn * np.einsum("ip,j,ijb->bp", W["Ja"][r], m, c)
              + Mn * np.einsum("i,jp,ijb->bp", a, W["Jm"][r], c))
        J[r] = F[:, None] * dS
        J[r, :, I_TAUV] += F_tv * S
    return flux, J


def logp_and_grad(theta_unb, z, grid, prior4, obs_flux, obs_sigma, path, cssp=None):
    """logP(theta~) = -1/2 sum_b ((flux_b - d_b)/sigma_b)^2 + sum_p log SN(theta~_p) over the D = 4 sampled
    parameters (R12), and its gradient.  prior4 [7,4]: rows y_lo, y_hi, k, x0, xi, omega, skew."""
    thu = np.asarray(theta_unb, float)
    th, dth = M.bound(thu, prior4)
    if path == "exact":
        flux, J = photometry_exact(th, z, grid)
    else:
        flux, J = photometry_approx(th, z, grid, cssp)
    r = (flux - obs_flux) / obs_sigma
    lp_prior, dlp = M.log_skew_normal(thu, prior4)
    logp = -0.5 * (r * r).sum(1) + lp_prior.sum(1)
    grad = np.einsum("rb,rbp->rp", -r / obs_sigma, J) * dth + dlp
    return logp, grad, flux
