"""Float64 CPU ORACLE of the SPS photometry log-likelihood and its gradient.

TEST INFRASTRUCTURE ONLY.  Only `tests/`, `__graft_entry__.smoke()` and the `cpu_baseline` /
`--impl reference` legs of `bench.py` may import this package.  It shares no code with the
CUDA path (`paper_2506_19919_b200/csrc`) and imports nothing from it; inputs arrive as arrays.

The method is a definition (a weighted sum, two quadratures), so the oracle follows the paper
step by step, in the paper's notation; numpy is used for elementwise maths and plain sums/matmuls,
with no blocking, fusion or reordering.  Every function cites the passage it follows
(`/root/reference/PAPER.md:<line>`).  Where the paper is silent the reading taken is listed in
DESIGN.md ("Readings") and referenced here as R#.

Parameter order (13): logM, tau, alpha, beta, F_burst, logT_peak, logT_max, logZ, sigma_logZ,
A_V, delta, F_floor, z  (z per BASELINE.json configs[1]).

Parity status: every function is pinned by `tests/test_oracle_*.py` except where a reading is
flagged "parity unpinned" below (the log base of A7 (R8), the Drude-bump strength (R10), the
numbers of the bounds/prior table (R13)).
"""
from __future__ import annotations

import math

import numpy as np
from numpy.polynomial.legendre import leggauss
from scipy.special import erf  # library primitive: the error function for the normal CDF

NDIM = 13
I_LOGM, I_TAU, I_ALPHA, I_BETA, I_FB, I_LTP, I_LTM, I_LZ, I_SLZ, I_AV, I_DEL, I_FFL, I_Z = range(13)

LAMBDA_V = 5500.0
GYR_PER_INV_H0 = 977.7922216807891   # (km/s/Mpc)^-1 in Gyr
_GL_X, _GL_W = leggauss(32)          # R6: 32-point Gauss-Legendre per age bin


# ----------------------------------------------------------------------------------------------
# a0  bounding sigmoid, Eq. (C1)
# ----------------------------------------------------------------------------------------------
def bound(theta_unb, prior):
    """theta = y_lo + (y_hi-y_lo)/(1+exp(-k(theta~ - x0)));  returns theta and d theta/d theta~."""
    y_lo, y_hi, k, x0 = prior[0], prior[1], prior[2], prior[3]
    x = k * (theta_unb - x0)
    # the same function, evaluated without overflow for saturated arguments (warmup reaches |x| ~ 20-90):
    # e = exp(-|x|) <= 1;  s = 1/(1+e) for x >= 0, e/(1+e) for x < 0;  s (1-s) = e/(1+e)^2 either way
    e = np.exp(-np.abs(x))
    s = np.where(x >= 0.0, 1.0, e) / (1.0 + e)
    return y_lo + (y_hi - y_lo) * s, (y_hi - y_lo) * k * e / ((1.0 + e) * (1.0 + e))


def unbound(theta, prior):
    """F_B^{-1}."""
    y_lo, y_hi, k, x0 = prior[0], prior[1], prior[2], prior[3]
    u = (theta - y_lo) / (y_hi - y_lo)
    return x0 + np.log(u / (1.0 - u)) / k


# ----------------------------------------------------------------------------------------------
# a1  age of the universe at z ("t_obs"; R11: flat LCDM closed form), Gyr
# ----------------------------------------------------------------------------------------------
def cosmic_time(z, H0, Om):
    OL = 1.0 - Om
    pref = 2.0 * GYR_PER_INV_H0 / (3.0 * H0 * math.sqrt(OL))
    t = pref * np.arcsinh(math.sqrt(OL / Om) * (1.0 + z) ** -1.5)
    Hz = H0 / GYR_PER_INV_H0 * np.sqrt(Om * (1.0 + z) ** 3 + OL)     # 1/Gyr
    return t, -1.0 / ((1.0 + z) * Hz)                                  # t, dt/dz


# ----------------------------------------------------------------------------------------------
# a2  smooth SFH: Eq. (A3)-(A5)
# ----------------------------------------------------------------------------------------------
def sfr_shape(t, tau, alpha, beta):
    """f(t) = [ (t/tau)^alpha + (t/tau)^-beta ]^-1  (Eq. A4 without M_formed), and its partials
    with respect to (t, tau, alpha, beta)."""
    x = t / tau
    xa = x ** alpha
    xb = x ** (-beta)
    f = 1.0 / (xa + xb)
    lx = np.log(x)
    q = f * f * (alpha * xa - beta * xb)
    return f, -q / t, q / tau, -f * f * xa * lx, f * f * xb * lx


def age_bin_edges_gyr(log10_age_yr):
    """R5: edges are midpoints of adjacent log10(age); first lower edge is age 0, last is +inf."""
    la = np.asarray(log10_age_yr, float)
    mid = 0.5 * (la[1:] + la[:-1])
    return np.concatenate([[0.0], 10.0 ** (mid - 9.0), [np.inf]]), np.concatenate([[-np.inf], mid, [np.inf]])


def smooth_age_weights(tau, alpha, beta, t_obs, log10_age_yr):
    """Mass formed in each age bin for M_formed = 1 (Eq. A5 numerators), by quadrature.

    Bin i holds stars of age in [A_i, A_{i+1}], i.e. formed at cosmic time
    t in [max(0,t_obs-A_{i+1}), max(0,t_obs-A_i)] (cosmic time runs opposite to age).
    R6: 32-point Gauss-Legendre in v = ln t per bin; the one bin that reaches t = 0 is cut at
    ln t_hi - 36 (the integrand falls as t^(beta+1), beta >= 0.2) and split into 12 panels.

    Inputs are 1-D arrays [B].  Returns dM [B,n_age] and its partials d/d(tau,alpha,beta,t_obs),
    each [B,n_age].
    """
    A, _ = age_bin_edges_gyr(log10_age_yr)
    tau = np.asarray(tau, float)[:, None]; alpha = np.asarray(alpha, float)[:, None]
    beta = np.asarray(beta, float)[:, None]; t_obs = np.asarray(t_obs, float)[:, None]
    t_hi = np.maximum(0.0, t_obs - A[None, :-1])
    t_lo = np.maximum(0.0, t_obs - A[None, 1:])
    B, n_age = t_hi.shape
    out = [np.zeros((B, n_age)) for _ in range(5)]   # dM, d/dtau, d/dalpha, d/dbeta, d/dt_obs

    def panel(lo, hi):
        """integral over v in [lo,hi] of f(e^v) e^v dv and the parameter partials; arrays [...]."""
        half = 0.5 * (hi - lo); mid = 0.5 * (hi + lo)
        v = mid[..., None] + half[..., None] * _GL_X
        t = np.exp(v)
        f, _, f_tau, f_al, f_be = sfr_shape(t, tau[..., None], alpha[..., None], beta[..., None])
        w = half[..., None] * _GL_W * t
        return [(w * g).sum(-1) for g in (f, f_tau, f_al, f_be)]

    reg = t_lo > 0.0
    lo = np.where(reg, np.log(np.where(reg, t_lo, 1.0)), 0.0)
    hi = np.where(reg, np.log(np.where(reg, t_hi, 1.0)), 0.0)
    vals = panel(lo, hi)
    for o, v in zip(out[:4], vals):
        o += np.where(reg, v, 0.0)
    # the bin that touches t = 0
    zero = (t_lo <= 0.0) & (t_hi > 0.0)
    t_c = np.where(zero, t_hi, 0.0).sum(1)                 # [B] exactly one such bin per row
    n_pan = 12
    edges = np.log(t_c)[:, None] - 36.0 + 3.0 * np.arange(n_pan + 1)[None, :]
    pv = panel(edges[:, :-1], edges[:, 1:])
    for o, v in zip(out[:4], pv):
        o += zero * v.sum(1)[:, None]
    # d/dt_obs: both limits move with t_obs (Leibniz); f(0) = 0 so clipped limits add nothing
    f_hi = np.where(t_hi > 0, sfr_shape(np.where(t_hi > 0, t_hi, 1.0), tau, alpha, beta)[0], 0.0)
    f_lo = np.where(t_lo > 0, sfr_shape(np.where(t_lo > 0, t_lo, 1.0), tau, alpha, beta)[0], 0.0)
    out[4] = f_hi - f_lo
    return out


# ----------------------------------------------------------------------------------------------
# a3  burst: Eq. (A6)-(A7)
# ----------------------------------------------------------------------------------------------
def triweight_pdf(x):
    """Eq. (A7)."""
    y = np.clip(x / 3.0, -1.0, 1.0)
    return 35.0 / 96.0 * (1.0 - y * y) ** 3


def triweight_cdf(x):
    """Integral of Eq. (A7) from -3 to x."""
    y = np.clip(x / 3.0, -1.0, 1.0)
    return 0.5 + 35.0 / 32.0 * (y - y ** 3 + 0.6 * y ** 5 - y ** 7 / 7.0)


def burst_age_weights(logT_peak, logT_max, log10_age_yr):
    """R7: P_burst,i = C_T(x(e_{i+1})) - C_T(x(e_i)), x = (log10 age - mu)/sigma, mu = log10 T_peak,
    sigma = (log10 T_max - log10 T_peak)/3 (R8: log is log10, ages in yr).
    Returns P [B,n_age], dP/dlogT_peak, dP/dlogT_max."""
    _, e = age_bin_edges_gyr(log10_age_yr)
    mu = np.asarray(logT_peak, float)[:, None]
    sg = (np.asarray(logT_max, float)[:, None] - mu) / 3.0
    with np.errstate(invalid="ignore"):
        x = (e[None, :] - mu) / sg
    x[:, 0] = -np.inf; x[:, -1] = np.inf
    C = triweight_cdf(x)
    pdf = triweight_pdf(x)
    xf = np.where(np.isfinite(x), x, 0.0)
    dC_dmu = pdf * (-1.0 / sg)
    dC_dsg = pdf * (-xf / sg)
    dC_dltp = dC_dmu - dC_dsg / 3.0
    dC_dltm = dC_dsg / 3.0
    return np.diff(C, axis=1), np.diff(dC_dltp, axis=1), np.diff(dC_dltm, axis=1)


# ----------------------------------------------------------------------------------------------
# a4  lognormal MDF  PAPER.md:378  (R9: normal-CDF differences over midpoints of the log10 Z grid)
# ----------------------------------------------------------------------------------------------
def met_weights(logZ, sigma_logZ, log10_Z):
    g = np.asarray(log10_Z, float)
    mid = 0.5 * (g[1:] + g[:-1])
    lz = np.asarray(logZ, float)[:, None]; s = np.asarray(sigma_logZ, float)[:, None]
    u = (mid[None, :] - lz) / s
    Phi = 0.5 * (1.0 + erf(u / math.sqrt(2.0)))
    phi = np.exp(-0.5 * u * u) / math.sqrt(2.0 * math.pi)
    one = np.ones_like(lz); zero = np.zeros_like(lz)
    Phi = np.concatenate([zero, Phi, one], 1)
    dlz = np.concatenate([zero, -phi / s, zero], 1)
    ds = np.concatenate([zero, -phi * u / s, zero], 1)
    return np.diff(Phi, axis=1), np.diff(dlz, axis=1), np.diff(ds, axis=1)


# ----------------------------------------------------------------------------------------------
# a0-a5 together: weights and their Jacobians with respect to the 13 bounded parameters
# ----------------------------------------------------------------------------------------------
def weights(theta, grid):
    """theta [B,13] bounded.  Returns dict with
       a [B,n_age]  (Eq. A6),  m [B,n_Z],  Mn [B] = M_star / mass_unit (Eq. A3),
       Ja [B,n_age,13], Jm [B,n_Z,13], JMn [B,13]  (partials w.r.t. theta)."""
    th = np.asarray(theta, float)
    B = th.shape[0]
    t_obs, dt_dz = cosmic_time(th[:, I_Z], grid.H0, grid.Om)
    dM, d_tau, d_al, d_be, d_to = smooth_age_weights(th[:, I_TAU], th[:, I_ALPHA], th[:, I_BETA], t_obs,
                                                     grid.log10_age_yr)
    Msum = dM.sum(1)                                   # Eq. (A3) for M_formed = 1
    Ps = dM / Msum[:, None]                            # Eq. (A5)
    def dPs(d):                                        # quotient rule
        return d / Msum[:, None] - dM * d.sum(1)[:, None] / Msum[:, None] ** 2
    Pb, dPb_ltp, dPb_ltm = burst_age_weights(th[:, I_LTP], th[:, I_LTM], grid.log10_age_yr)
    Fb = th[:, I_FB][:, None]
    a = (1.0 - Fb) * Ps + Fb * Pb                      # Eq. (A6)
    n_age = a.shape[1]
    Ja = np.zeros((B, n_age, NDIM))
    Ja[:, :, I_TAU] = (1.0 - Fb) * dPs(d_tau)
    Ja[:, :, I_ALPHA] = (1.0 - Fb) * dPs(d_al)
    Ja[:, :, I_BETA] = (1.0 - Fb) * dPs(d_be)
    Ja[:, :, I_Z] = (1.0 - Fb) * dPs(d_to) * dt_dz[:, None]
    Ja[:, :, I_FB] = Pb - Ps
    Ja[:, :, I_LTP] = Fb * dPb_ltp
    Ja[:, :, I_LTM] = Fb * dPb_ltm
    m, dm_lz, dm_s = met_weights(th[:, I_LZ], th[:, I_SLZ], grid.log10_Z)
    Jm = np.zeros((B, m.shape[1], NDIM))
    Jm[:, :, I_LZ] = dm_lz; Jm[:, :, I_SLZ] = dm_s
    Mf = 10.0 ** (th[:, I_LOGM] - grid.log10_mass_unit)   # R2: M_formed in mass_unit/Gyr
    Mn = Mf * Msum
    JMn = np.zeros((B, NDIM))
    JMn[:, I_LOGM] = math.log(10.0) * Mn
    JMn[:, I_TAU] = Mf * d_tau.sum(1)
    JMn[:, I_ALPHA] = Mf * d_al.sum(1)
    JMn[:, I_BETA] = Mf * d_be.sum(1)
    JMn[:, I_Z] = Mf * d_to.sum(1) * dt_dz
    return dict(a=a, m=m, Mn=Mn, Ja=Ja, Jm=Jm, JMn=JMn, t_obs=t_obs)


# ----------------------------------------------------------------------------------------------
# a8  dust: Eq. (A8)-(A9)  PAPER.md:386-392  (R10: Calzetti k0, Drude bump)
# ----------------------------------------------------------------------------------------------
_CALZ_SWITCH_INV_UM = 1.2809053864877329   # 1/lambda [1/um] where the two Calzetti branches cross (R10)


def calzetti_k0(lam_A):
    """Calzetti et al. (2000) k(lambda) with R_V = 4.05, lambda in Angstrom; each branch extended
    outward, the switch placed where the branches intersect (0.7807 um) so k0 is continuous;
    clamped at 0.  Returns k0 and dk0/dlambda [1/Angstrom]."""
    lam = np.asarray(lam_A, float)
    u = 1.0e4 / lam                       # 1/lambda in 1/um
    uv = 2.659 * (-2.156 + 1.509 * u - 0.198 * u * u + 0.011 * u ** 3) + 4.05
    duv = 2.659 * (1.509 - 0.396 * u + 0.033 * u * u)
    ir = 2.659 * (-1.857 + 1.040 * u) + 4.05
    dir_ = 2.659 * 1.040 * np.ones_like(u)
    k = np.where(u > _CALZ_SWITCH_INV_UM, uv, ir)
    dk_du = np.where(u > _CALZ_SWITCH_INV_UM, duv, dir_)
    pos = k > 0.0
    return np.where(pos, k, 0.0), np.where(pos, dk_du * (-u / lam), 0.0)


def drude(lam_A):
    """Lorentzian-like Drude profile of unit peak at 2175 A, width 350 A (R10).
    Returns profile and d/dlambda."""
    lam = np.asarray(lam_A, float)
    l0, w = 2175.0, 350.0
    n = (lam * w) ** 2
    d = (lam * lam - l0 * l0) ** 2 + n
    dn = 2.0 * lam * w * w
    dd = 4.0 * lam * (lam * lam - l0 * l0) + dn
    return n / d, (dn * d - n * dd) / (d * d)


def attenuation(lam_A, A_V, delta, F_floor):
    """F_att(lambda) of Eq. (A9) with A(lambda) of Eq. (A8); bump strength E_b = 0.85 - 1.9 delta (R10).
    lam_A broadcasts against the parameter arrays.
    Returns F, dF/dA_V, dF/ddelta, dF/dF_floor, dF/dlambda."""
    lam = np.asarray(lam_A, float)
    k0, dk0 = calzetti_k0(lam)
    dr, ddr = drude(lam)
    r = lam / LAMBDA_V
    pw = r ** delta
    Eb = 0.85 - 1.9 * delta
    br = k0 * pw + Eb * dr
    A = A_V / 4.05 * br
    pos = A > 0.0
    A = np.where(pos, A, 0.0)
    dA_dAV = np.where(pos, br / 4.05, 0.0)
    dA_ddel = np.where(pos, A_V / 4.05 * (k0 * pw * np.log(r) - 1.9 * dr), 0.0)
    dA_dlam = np.where(pos, A_V / 4.05 * (dk0 * pw + k0 * delta * pw / lam + Eb * ddr), 0.0)
    T = 10.0 ** (-0.4 * A)
    dF_dA = -(1.0 - F_floor) * 0.4 * math.log(10.0) * T
    F = F_floor + (1.0 - F_floor) * T
    return F, dF_dA * dA_dAV, dF_dA * dA_ddel, 1.0 - T + 0.0 * F, dF_dA * dA_dlam


# ----------------------------------------------------------------------------------------------
# filters and quadrature weights  (Eq. 3  PAPER.md:60-63;  R3, R4)
# ----------------------------------------------------------------------------------------------
def trapezoid_weights(wave_A):
    """R4: trapezoid rule on the SSP grid: dlam_k = (lam_{k+1}-lam_{k-1})/2, half-intervals at the ends."""
    w = np.asarray(wave_A, float)
    d = np.empty_like(w)
    d[1:-1] = 0.5 * (w[2:] - w[:-2])
    d[0] = 0.5 * (w[1] - w[0]); d[-1] = 0.5 * (w[-1] - w[-2])
    return d


def filter_T(lam_obs_A, mu_A, sigma_A):
    """Gaussian transmission (Fig. B.1), truncated at 5 sigma (R4).
    Returns T and dT/dlambda_obs."""
    x = (lam_obs_A - mu_A) / sigma_A
    T = np.where(np.abs(x) <= 5.0, np.exp(-0.5 * x * x), 0.0)
    return T, -T * x / sigma_A


def effective_wavelength(mu_A, sigma_A, n=20001):
    """Eq. (5) at z = 0 on the filter's own grid: int lam T / int T."""
    out = np.empty(len(mu_A))
    for b, (m, s) in enumerate(zip(mu_A, sigma_A)):
        lam = np.linspace(m - 5.0 * s, m + 5.0 * s, n)
        T, _ = filter_T(lam, m, s)
        out[b] = np.trapezoid(lam * T, lam) / np.trapezoid(T, lam)
    return out


def tabulated_T(lam_obs_A, wave_A, trans):
    """R4: a tabulated transmission curve (T(lambda) is a general curve; only App. B's test uses
    Gaussians) is linearly interpolated between its knots and is zero outside its support [wave[0], wave[-1]].
    Returns T and dT/dlambda_obs = the slope of the segment that holds lambda (R18: at a knot, the segment to its right)."""
    w = np.asarray(wave_A, float); t = np.asarray(trans, float)
    lam = np.asarray(lam_obs_A, float)
    seg = np.clip(np.searchsorted(w, lam, side="right") - 1, 0, len(w) - 2)
    slope = (t[1:] - t[:-1]) / (w[1:] - w[:-1])
    inside = (lam >= w[0]) & (lam <= w[-1])
    T = np.where(inside, t[seg] + (lam - w[seg]) * slope[seg], 0.0)
    return T, np.where(inside, slope[seg], 0.0)


def tabulated_effective_wavelength(wave_A, trans):
    """Eq. (5) at z = 0 for a tabulated curve: int lam T / int T of the piecewise-linear interpolant, each segment
    integrated exactly (T linear: trapezoid; lam T quadratic: Simpson)."""
    w = np.asarray(wave_A, float); t = np.asarray(trans, float)
    h = w[1:] - w[:-1]
    wm = 0.5 * (w[1:] + w[:-1]); tm = 0.5 * (t[1:] + t[:-1])
    den = (h * tm).sum()
    num = (h / 6.0 * (w[:-1] * t[:-1] + 4.0 * wm * tm + w[1:] * t[1:])).sum()
    return num / den


def _filter_tab(grid):
    return getattr(grid, "filt_tab", None)


def n_bands(grid):
    tab = _filter_tab(grid)
    return len(tab[2]) - 1 if tab is not None else len(grid.filt_mu_A)


def band_T(grid, lam_obs_A):
    """T_b(lambda_obs) and dT_b/dlambda_obs of every band of the grid at the observed wavelengths lam_obs_A [N]
    -> [n_band, N] each.  Gaussian filters (mu, sigma) or tabulated curves grid.filt_tab = (wave, trans, offsets):
    band b owns the knots offsets[b] .. offsets[b+1]-1."""
    lam = np.asarray(lam_obs_A, float)
    tab = _filter_tab(grid)
    if tab is None:
        return filter_T(lam[None, :], np.asarray(grid.filt_mu_A, float)[:, None], np.asarray(grid.filt_sigma_A, float)[:, None])
    wave, trans, off = tab
    out = [tabulated_T(lam, wave[off[b]:off[b + 1]], trans[off[b]:off[b + 1]]) for b in range(len(off) - 1)]
    return np.stack([o[0] for o in out]), np.stack([o[1] for o in out])


def band_effective_wavelength(grid):
    tab = _filter_tab(grid)
    if tab is None:
        return effective_wavelength(grid.filt_mu_A, grid.filt_sigma_A)
    wave, trans, off = tab
    return np.array([tabulated_effective_wavelength(wave[off[b]:off[b + 1]], trans[off[b]:off[b + 1]]) for b in range(len(off) - 1)])


# ----------------------------------------------------------------------------------------------
# a6  exact photometry, Eq. (4) with M_star restored (R1)
# ----------------------------------------------------------------------------------------------
def photometry_exact(theta, grid, want_jac=True):
    """flux_b = sum_k [ sum_ij w_ij L_ij(lam_k) ] F_att(lam_k) T_b(lam_k (1+z)) dlam_k.
    theta [B,13] bounded.  Returns flux [B,n_band] and J = d flux / d theta [B,n_band,13]."""
    th = np.asarray(theta, float)
    W = weights(th, grid)
    B = th.shape[0]
    L = np.asarray(grid.ssp, float)                      # [K, N]
    lam = np.asarray(grid.wave_A, float)
    dlam = trapezoid_weights(lam)
    n_band = n_bands(grid)
    flux = np.zeros((B, n_band)); J = np.zeros((B, n_band, NDIM))
    for r in range(B):
        a, m, Mn = W["a"][r], W["m"][r], W["Mn"][r]
        w = Mn * np.outer(a, m).reshape(-1)              # Eq. (2) and M_star:  w_ij
        S = w @ L                                        # Eq. (1) without dust  [N]
        z = th[r, I_Z]
        F, F_av, F_del, F_fl, _ = attenuation(lam, th[r, I_AV], th[r, I_DEL], th[r, I_FFL])
        T, dT = band_T(grid, lam * (1.0 + z))                                                          # [b,N]
        flux[r] = (T * (S * F * dlam)[None, :]).sum(1)
        if not want_jac:
            continue
        # d w / d theta_p  ->  d S / d theta_p
        dw = (W["JMn"][r][None, None, :] * np.outer(a, m)[:, :, None]
              + Mn * W["Ja"][r][:, None, :] * m[None, :, None]
              + Mn * a[:, None, None] * W["Jm"][r][None, :, :]).reshape(-1, NDIM)     # [K,13]
        dS = dw.T @ L                                                                # [13,N]
        J[r] = np.einsum("bk,pk->bp", T * (F * dlam)[None, :], dS)
        J[r, :, I_AV] += (T * (S * F_av * dlam)[None, :]).sum(1)
        J[r, :, I_DEL] += (T * (S * F_del * dlam)[None, :]).sum(1)
        J[r, :, I_FFL] += (T * (S * F_fl * dlam)[None, :]).sum(1)
        J[r, :, I_Z] += (dT * (lam * S * F * dlam)[None, :]).sum(1)
    return flux, J


# ----------------------------------------------------------------------------------------------
# a-setup  c_SSP table, Eq. (7)
# ----------------------------------------------------------------------------------------------
def z_grid(grid):
    return np.linspace(grid.z_min, grid.z_max, grid.n_z)


def cssp_table(grid, z_values=None):
    """c_SSP[t,i,j,b] = sum_k L_ij(lam_k) T_b(lam_k (1+z_t)) dlam_k    -> [n_z, n_age*n_Z, n_band]."""
    zs = z_grid(grid) if z_values is None else np.asarray(z_values, float)
    L = np.asarray(grid.ssp, float)
    lam = np.asarray(grid.wave_A, float)
    dlam = trapezoid_weights(lam)
    out = np.empty((len(zs), L.shape[0], n_bands(grid)))
    for t, z in enumerate(zs):
        T, _ = band_T(grid, lam * (1.0 + z))
        out[t] = L @ (T * dlam[None, :]).T
    return out


# ----------------------------------------------------------------------------------------------
# a7  approximate photometry, Eq. (6)
# ----------------------------------------------------------------------------------------------
def photometry_approx(theta, grid, cssp, lam_eff_obs=None):
    """flux_b = F_att(lam_eff,b/(1+z)) sum_ij w_ij c~_ijb(z),  c~ = linear interpolation in z of the
    c_SSP lookup table (R18: one-sided derivative of the cell holding z).
    Returns flux [B,n_band], J [B,n_band,13]."""
    th = np.asarray(theta, float)
    W = weights(th, grid)
    B = th.shape[0]
    if lam_eff_obs is None:
        lam_eff_obs = band_effective_wavelength(grid)
    n_band = n_bands(grid)
    n_age, n_Z = len(grid.log10_age_yr), len(grid.log10_Z)
    dz = (grid.z_max - grid.z_min) / (grid.n_z - 1)
    flux = np.zeros((B, n_band)); J = np.zeros((B, n_band, NDIM))
    for r in range(B):
        z = th[r, I_Z]
        t = int(min(max(math.floor((z - grid.z_min) / dz), 0), grid.n_z - 2))
        f = (z - (grid.z_min + t * dz)) / dz
        c = ((1.0 - f) * cssp[t] + f * cssp[t + 1]).reshape(n_age, n_Z, n_band)
        dc = ((cssp[t + 1] - cssp[t]) / dz).reshape(n_age, n_Z, n_band)
        a, m, Mn = W["a"][r], W["m"][r], W["Mn"][r]
        lam_r = lam_eff_obs / (1.0 + z)
        F, F_av, F_del, F_fl, F_lam = attenuation(lam_r, th[r, I_AV], th[r, I_DEL], th[r, I_FFL])
        S = Mn * np.einsum("i,j,ijb->b", a, m, c)
        flux[r] = F * S
        dS = (W["JMn"][r][None, :] * np.einsum("i,j,ijb->b", a, m, c)[:, None]
              + Mn * np.einsum("ip,j,ijb->bp", W["Ja"][r], m, c)
              + Mn * np.einsum("i,jp,ijb->bp", a, W["Jm"][r], c))
        J[r] = F[:, None] * dS
        J[r, :, I_AV] += F_av * S
        J[r, :, I_DEL] += F_del * S
        J[r, :, I_FFL] += F_fl * S
        J[r, :, I_Z] += F * Mn * np.einsum("i,j,ijb->b", a, m, dc) + S * F_lam * (-lam_r / (1.0 + z))
    return flux, J


# ----------------------------------------------------------------------------------------------
# a9  log-posterior: Gaussian likelihood in flux (R12) + skew-normal prior on theta~ (Eq. C2)
# ----------------------------------------------------------------------------------------------
def log_skew_normal(x_unb, prior):
    """log of Eq. (C2) and its derivative.  PAPER.md:438-442."""
    xi, om, s = prior[4], prior[5], prior[6]
    u = (x_unb - xi) / om
    from scipy.special import log_ndtr
    lp = math.log(2.0) - np.log(om) - 0.5 * math.log(2.0 * math.pi) - 0.5 * u * u + log_ndtr(s * u)
    ratio = np.exp(-0.5 * (s * u) ** 2 - log_ndtr(s * u)) / math.sqrt(2.0 * math.pi)   # phi/Phi
    return lp, (-u + s * ratio) / om


def logp_and_grad(theta_unb, grid, prior, obs_flux, obs_sigma, path, cssp=None):
    """logP(theta~) = -1/2 sum_b ((flux_b - d_b)/sigma_b)^2 + sum_p log SN(theta~_p)  (no Jacobian
    term: the prior is defined on theta~) and d logP / d theta~.
    theta_unb [B,13]; obs_* [B,n_band]; path in {'exact','approx'}."""
    thu = np.asarray(theta_unb, float)
    th, dth = bound(thu, prior)
    if path == "exact":
        flux, J = photometry_exact(th, grid)
    else:
        flux, J = photometry_approx(th, grid, cssp)
    r = (flux - obs_flux) / obs_sigma
    g_flux = -r / obs_sigma
    lp_prior, dlp = log_skew_normal(thu, prior)
    logp = -0.5 * (r * r).sum(1) + lp_prior.sum(1)
    grad = np.einsum("rb,rbp->rp", g_flux, J) * dth + dlp
    return logp, grad, flux
