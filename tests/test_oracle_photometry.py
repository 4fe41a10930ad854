"""Pins of the oracle's dust law, filters, exact/approximate photometry, likelihood and gradient.
CPU only.  See tests/test_oracle_model.py for conventions."""
import math

import numpy as np
import pytest
from scipy import stats

from oracle import sps_model as M
from paper_2506_19919_b200 import workloads as W


@pytest.fixture(scope="module")
def tiny():
    return W.make_grid("tiny")


@pytest.fixture(scope="module")
def prior():
    return W.make_prior().as_array()


@pytest.fixture(scope="module")
def cssp(tiny):
    return M.cssp_table(tiny)


def _theta(prior, n, seed, **fixed):
    th, _ = M.bound(W.draw_theta_unbounded(W.make_prior(), n, seed), prior)
    for k, v in fixed.items():
        th[:, W.PARAM_NAMES.index(k)] = v
    return th


# ---- A8-A9 dust (R10) -------------------------------------------------------------
def test_dust_normalisation_and_identities():
    k0, _ = M.calzetti_k0(np.array([5500.0]))
    assert abs(k0[0] - 4.05) < 0.01                                   # "A_V is the normalization at 5500 A"
    F = M.attenuation(np.array([5500.0]), 1.3, 0.0, 0.0)[0]
    assert abs(-2.5 * math.log10(F[0]) - 1.3) < 0.01 * 1.3            # A(lambda_V) = A_V
    lam = np.geomspace(300.0, 4e4, 200)
    assert np.all(M.attenuation(lam, 0.0, -0.4, 0.2)[0] == 1.0)       # A_V = 0  => identity
    assert np.allclose(M.attenuation(lam, 2.0, -0.4, 1.0)[0], 1.0)    # F_floor = 1 => identity (Eq. A9)
    F = M.attenuation(lam, 1.0, -0.3, 0.15)[0]
    assert np.all(F >= 0.15) and np.all(F <= 1.0)                     # floor = unobscured fraction
    # Calzetti branches: continuous at the switch, published values k(0.15um)~10.3? no: use Eq. itself at 0.3 um
    s = 1e4 / M._CALZ_SWITCH_INV_UM
    a, b = M.calzetti_k0(np.array([s * (1 - 1e-9), s * (1 + 1e-9)]))[0]
    assert abs(a - b) < 1e-6
    u = 1 / 0.3
    assert M.calzetti_k0(np.array([3000.0]))[0][0] == pytest.approx(2.659 * (-2.156 + 1.509 * u - 0.198 * u * u + 0.011 * u ** 3) + 4.05)
    assert M.calzetti_k0(np.array([12000.0]))[0][0] == pytest.approx(2.659 * (-1.857 + 1.040 / 1.2) + 4.05)
    d, _ = M.drude(np.array([2175.0, 2175.0 + 175.0 * 1.0]))
    assert d[0] == pytest.approx(1.0) and 0.4 < d[1] < 0.6            # unit peak, FWHM ~ 350 A


def test_dust_partials_finite_difference():
    lam = np.array([900.0, 2175.0, 4000.0, 7000.0, 9000.0, 20000.0])
    av, de, ff = 0.8, -0.35, 0.12
    F, dav, dde, dff, dlam = M.attenuation(lam, av, de, ff)
    h = 1e-6
    assert np.allclose(dav, (M.attenuation(lam, av + h, de, ff)[0] - M.attenuation(lam, av - h, de, ff)[0]) / (2 * h), rtol=1e-6)
    assert np.allclose(dde, (M.attenuation(lam, av, de + h, ff)[0] - M.attenuation(lam, av, de - h, ff)[0]) / (2 * h), rtol=1e-6, atol=1e-10)
    assert np.allclose(dff, (M.attenuation(lam, av, de, ff + h)[0] - M.attenuation(lam, av, de, ff - h)[0]) / (2 * h), rtol=1e-6)
    hl = 1e-3
    assert np.allclose(dlam, (M.attenuation(lam + hl, av, de, ff)[0] - M.attenuation(lam - hl, av, de, ff)[0]) / (2 * hl), rtol=1e-5, atol=1e-12)


# ---- Eq. 3, 5, 7 filters and quadrature (R3, R4) -----------------------------------------
def test_constant_spectrum_gives_filter_integral(tiny):
    g = W.make_grid("tiny"); g.ssp = np.ones_like(g.ssp)
    for z in (0.0, 0.7):
        c = M.cssp_table(g, [z])[0]
        ref = g.filt_sigma_A * math.sqrt(2 * math.pi) * math.erf(5 / math.sqrt(2)) / (1 + z)
        assert np.allclose(c, ref[None, :], rtol=2e-3)                # trapezoid on the 500-point grid
    assert M.trapezoid_weights(g.wave_A).sum() == pytest.approx(g.wave_A[-1] - g.wave_A[0])


def test_redshifted_filter_equals_blueshifted_curve(tiny):
    # T(lambda|z): the observed-frame curve read at lambda_rest (1+z)  ==  a curve with mu/(1+z), sigma/(1+z) at z=0
    z = 0.83
    g2 = W.make_grid("tiny"); g2.filt_mu_A = tiny.filt_mu_A / (1 + z); g2.filt_sigma_A = tiny.filt_sigma_A / (1 + z)
    assert np.allclose(M.cssp_table(tiny, [z])[0], M.cssp_table(g2, [0.0])[0], rtol=1e-12)


def test_effective_wavelength_of_symmetric_filter(tiny):
    assert np.allclose(M.effective_wavelength(tiny.filt_mu_A, tiny.filt_sigma_A), tiny.filt_mu_A, rtol=1e-9)  # Eq. 5


def test_delta_sfh_reproduces_single_ssp(tiny, prior):
    # a burst narrower than one age bin + a delta MDF + no dust  ==  M_star x one SSP's band flux (Eq. 1, 4)
    th = _theta(prior, 1, 3, F_burst=1.0, A_V=0.0, sigma_logZ=1e-4, z=0.5)
    i, j = 3, 2
    la = tiny.log10_age_yr
    th[0, M.I_LTP] = la[i]; th[0, M.I_LTM] = la[i] + 0.3 * (la[1] - la[0])
    th[0, M.I_LZ] = tiny.log10_Z[j]
    w = M.weights(th, tiny)
    assert w["a"][0, i] == pytest.approx(1.0) and w["m"][0, j] == pytest.approx(1.0)
    flux, _ = M.photometry_exact(th, tiny)
    lam = tiny.wave_A
    for b in range(tiny.n_band):
        T, _ = M.filter_T(lam * 1.5, tiny.filt_mu_A[b], tiny.filt_sigma_A[b])
        ref = w["Mn"][0] * np.trapezoid(tiny.ssp[i * tiny.n_Z + j].astype(float) * T, lam)
        assert flux[0, b] == pytest.approx(ref, rel=1e-10)


def test_flux_linear_in_mass(tiny, prior, cssp):
    th = _theta(prior, 2, 8)
    f0, J = M.photometry_approx(th, tiny, cssp)
    th2 = th.copy(); th2[:, 0] += 1.0
    assert np.allclose(M.photometry_approx(th2, tiny, cssp)[0], 10.0 * f0, rtol=1e-12)     # R1: flux ~ M_star
    assert np.allclose(J[:, :, 0], math.log(10.0) * f0, rtol=1e-12)


def test_zero_dust_approx_equals_exact_on_z_node(tiny, prior, cssp):
    zg = M.z_grid(tiny)
    th = _theta(prior, 3, 11, A_V=0.0)
    th[:, 12] = zg[[2, 5, 9]]
    fe, _ = M.photometry_exact(th, tiny)
    fa, _ = M.photometry_approx(th, tiny, cssp)
    assert np.allclose(fe, fa, rtol=1e-12)                                                  # Eq. 6 == Eq. 4 when F_att const


def test_approximation_accuracy_soft_band(tiny, prior):
    # <=0.1% in magnitude for lambda/FWHM 3.4..25.5 on MIST; on these smooth stand-in
    # spectra with lambda/FWHM = 6 filters and strong dust we only require it to stay small (|dm| < 0.06 mag; worst at the 2175 A bump).
    th = _theta(prior, 6, 21)
    zs = np.array([t[12] for t in th])
    c = M.cssp_table(tiny, zs)
    for r in range(len(th)):
        g = W.make_grid("tiny"); g.z_min = zs[r]; g.z_max = zs[r] + 1.0; g.n_z = 2
        cc = np.stack([c[r], c[r]])
        fa, _ = M.photometry_approx(th[r:r + 1], g, cc)
        fe, _ = M.photometry_exact(th[r:r + 1], tiny, want_jac=False)
        assert np.all(np.abs(2.5 * np.log10(fa / fe)) < 0.06)


# ---- C2 prior and the likelihood (R12) -------------------------------------------------
def test_skew_normal_matches_scipy(prior):
    x = np.random.default_rng(1).normal(0, 2, (20, 13)) * prior[5] + prior[4]
    lp, dlp = M.log_skew_normal(x, prior)
    ref = stats.skewnorm.logpdf(x, prior[6], loc=prior[4], scale=prior[5])
    assert np.allclose(lp, ref, rtol=1e-10, atol=1e-10)
    h = 1e-6
    fd = (M.log_skew_normal(x + h, prior)[0] - M.log_skew_normal(x - h, prior)[0]) / (2 * h)
    assert np.allclose(dlp, fd, rtol=1e-5, atol=1e-7)
    p0 = prior.copy(); p0[6] = 0.0
    assert np.allclose(M.log_skew_normal(x, p0)[0], stats.norm.logpdf(x, prior[4], prior[5]), atol=1e-12)  # s = 0


@pytest.mark.parametrize("path", ["approx", "exact"])
def test_gradient_matches_central_differences(tiny, prior, cssp, path):
    pr = W.make_prior()
    thu = W.draw_theta_unbounded(pr, 3, 77)
    th, _ = M.bound(thu, prior)
    zg = M.z_grid(tiny); dz = zg[1] - zg[0]
    # keep z away from a z-grid knot (R18) so the finite difference does not straddle a kink
    frac = ((th[:, 12] - zg[0]) / dz) % 1.0
    th[:, 12] += np.where(frac < 0.2, 0.3 * dz, np.where(frac > 0.8, -0.3 * dz, 0.0))
    thu = M.unbound(th, prior)
    truth = M.bound(W.draw_theta_unbounded(pr, 3, 78), prior)[0]
    truth[:, 12] = th[:, 12]
    f_true = (M.photometry_exact(truth, tiny, False)[0] if path == "exact" else M.photometry_approx(truth, tiny, cssp)[0])
    d, s = W.noisy_observations(f_true, 5, 0.05, 0.05)
    lp, g, flux = M.logp_and_grad(thu, tiny, prior, d, s, path, cssp)
    assert np.all(np.isfinite(g))
    for p in range(13):
        h = 1e-5
        tp = thu.copy(); tm = thu.copy(); tp[:, p] += h; tm[:, p] -= h
        fd = (M.logp_and_grad(tp, tiny, prior, d, s, path, cssp)[0] - M.logp_and_grad(tm, tiny, prior, d, s, path, cssp)[0]) / (2 * h)
        assert np.allclose(g[:, p], fd, rtol=2e-6, atol=2e-6 * np.abs(g).max()), (p, g[:, p], fd)
    # at flux == data the likelihood term vanishes with zero slope: only the prior is left
    lp0, g0, _ = M.logp_and_grad(thu, tiny, prior, flux, s, path, cssp)
    pl, pg = M.log_skew_normal(thu, prior)
    assert np.allclose(lp0, pl.sum(1)) and np.allclose(g0, pg)


# ---- tabulated filters (T(lambda) is a general transmission curve; R4: linear interpolation) ------------
def test_tabulated_curve_interpolation_and_support():
    w = np.array([4000.0, 4100.0, 4400.0, 5000.0]); t = np.array([0.0, 0.8, 1.0, 0.0])
    lam = np.array([3999.9, 4000.0, 4050.0, 4100.0, 4250.0, 4700.0, 5000.0, 5000.1])
    T, dT = M.tabulated_T(lam, w, t)
    assert np.allclose(T, [0.0, 0.0, 0.4, 0.8, 0.9, 0.5, 0.0, 0.0], atol=1e-15)          # hand-computed
    assert np.allclose(dT[[2, 4, 5]], [0.008, 0.2 / 300.0, -1.0 / 600.0]) and dT[0] == 0.0 and dT[-1] == 0.0
    assert np.allclose(T[1:-1], np.interp(lam[1:-1], w, t))                               # library routine
    # at an interior knot the slope is the one of the segment to its right (R18)
    assert M.tabulated_T(np.array([4100.0]), w, t)[1][0] == pytest.approx(0.2 / 300.0)


def test_tabulated_effective_wavelength_closed_forms():
    # a linear ramp rising from a to b: centroid (a + 2 b) / 3 exactly, whatever the knots (Eq. 5)
    a, b = 5000.0, 6200.0
    w = np.array([a, 5100.0, 5350.0, 6000.0, b]); t = (w - a) / (b - a)
    assert abs(M.tabulated_effective_wavelength(w, t) - (a + 2 * b) / 3) < 1e-9
    # a symmetric triangle: its centre; a top-hat built from two steep edges: its centre
    w = np.array([100.0, 150.0, 200.0]); t = np.array([0.0, 1.0, 0.0])
    assert abs(M.tabulated_effective_wavelength(w, t) - 150.0) < 1e-12
    # against adaptive quadrature of the interpolant for an asymmetric curve
    from scipy import integrate
    g = W.make_grid("tiny_tab")
    wave, trans, off = g.filt_tab
    for k in range(3):
        ww, tt = wave[off[k]:off[k + 1]], trans[off[k]:off[k + 1]]
        num = sum(integrate.quad(lambda x: x * np.interp(x, ww, tt), ww[i], ww[i + 1])[0] for i in range(len(ww) - 1))
        den = sum(integrate.quad(lambda x: np.interp(x, ww, tt), ww[i], ww[i + 1])[0] for i in range(len(ww) - 1))
        assert abs(M.band_effective_wavelength(g)[k] - num / den) < 1e-8


def test_tabulated_filters_in_photometry(prior):
    g = W.make_grid("tiny_tab")
    assert M.n_bands(g) == 3
    # (1) constant spectrum: flux_b = trapezoid sum of T_b over the SSP grid (R4), and close to the exact area
    g1 = __import__("dataclasses").replace(g, ssp=np.ones_like(g.ssp))
    th = _theta(prior, 2, 3, A_V=0.0, z=0.0)
    w = M.weights(th, g1)
    flux = M.photometry_exact(th, g1, want_jac=False)[0]
    lam = g.wave_A; dlam = M.trapezoid_weights(lam)
    wave, trans, off = g.filt_tab
    for b in range(3):
        Tb = np.interp(lam, wave[off[b]:off[b + 1]], trans[off[b]:off[b + 1]], left=0.0, right=0.0)
        assert np.allclose(flux[:, b], w["Mn"] * (Tb * dlam).sum(), rtol=1e-12)
    # (2) a curve tabulated from a Gaussian on a fine grid reproduces the Gaussian filter's photometry
    gg = W.make_grid("tiny")
    lam_f = [np.linspace(m - 5 * s, m + 5 * s, 4001) for m, s in zip(gg.filt_mu_A, gg.filt_sigma_A)]
    tab = (np.concatenate(lam_f), np.concatenate([np.exp(-0.5 * ((l - m) / s) ** 2) for l, m, s in zip(lam_f, gg.filt_mu_A, gg.filt_sigma_A)]),
           np.arange(4) * 4001)
    gt = __import__("dataclasses").replace(gg, filt_tab=tab)
    th = _theta(prior, 3, 4)
    f_g, J_g = M.photometry_exact(th, gg)
    f_t, J_t = M.photometry_exact(th, gt)
    assert np.allclose(f_t, f_g, rtol=2e-6) and np.allclose(J_t[:, :, :12], J_g[:, :, :12], rtol=1e-4, atol=1e-6 * np.abs(J_g).max())
    # d/dz sees the interpolant's piecewise-constant slope instead of the Gaussian's derivative: first order in the knot spacing
    assert np.allclose(J_t[:, :, 12], J_g[:, :, 12], rtol=5e-3, atol=1e-4 * np.abs(J_g).max())
    assert np.allclose(M.band_effective_wavelength(gt), M.band_effective_wavelength(gg), rtol=1e-6)
    # (3) gradient of the log-posterior against central differences, both paths (kinks of the interpolant: R18)
    cs = M.cssp_table(g)
    P = W.make_prior()
    thu = W.draw_theta_unbounded(P, 2, 8)
    d, s = W.noisy_observations(M.photometry_approx(M.bound(thu, prior)[0], g, cs)[0], 9, 0.05, 0.05)
    for path in ("exact", "approx"):
        lp, gr, _ = M.logp_and_grad(thu, g, prior, d, s, path, cs)
        for p in (0, 1, 9, 12):
            e = np.zeros(13); e[p] = 1e-6
            fd = (M.logp_and_grad(thu + e, g, prior, d, s, path, cs)[0] - M.logp_and_grad(thu - e, g, prior, d, s, path, cs)[0]) / 2e-6
            assert np.allclose(gr[:, p], fd, rtol=2e-4, atol=2e-5 * np.abs(gr).max()), (path, p, gr[:, p], fd)
