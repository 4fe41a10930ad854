"""Pins of the float64 oracle (`oracle/sps_model.py`) against what the paper and the mathematics
fix: closed forms, invariants, special cases that reduce to a library routine, finite differences.
CPU only.  Each test names the passage (PAPER.md:<line>) or DESIGN.md reading (R#) it pins."""
import math

import numpy as np
import pytest
from scipy import integrate, special, stats

from oracle import sps_model as M
from paper_2506_19919_b200 import workloads as W


@pytest.fixture(scope="module")
def tiny():
    return W.make_grid("tiny")


@pytest.fixture(scope="module")
def prior():
    return W.make_prior().as_array()


def _theta(prior, n, seed, **fixed):
    th, _ = M.bound(W.draw_theta_unbounded(W.make_prior(), n, seed), prior)
    for k, v in fixed.items():
        th[:, W.PARAM_NAMES.index(k)] = v
    return th


# ---- C1 bounding sigmoid -------------------------------------------------------
def test_bound_is_bijection_inside_bounds(prior):
    x = np.random.default_rng(0).normal(0, 2, (50, 13)) / prior[2] + prior[3]
    th, d = M.bound(x, prior)
    assert np.all(th > prior[0]) and np.all(th < prior[1])
    assert np.allclose(M.unbound(th, prior), x, atol=1e-9)
    h = 1e-6
    fd = (M.bound(x + h, prior)[0] - M.bound(x - h, prior)[0]) / (2 * h)
    assert np.allclose(d, fd, rtol=1e-6, atol=1e-9)
    # k = 4/(y_hi-y_lo): unit slope at the centre ("approximately linear")
    assert np.allclose(M.bound(prior[3][None, :], prior)[1], 1.0)


# ---- R11 cosmic time --------------------------------------------------------------------------------
@pytest.mark.parametrize("z", [0.0, 0.5, 2.9])
def test_cosmic_time_matches_integral(z):
    H0, Om = 67.74, 0.3089
    t, dt = M.cosmic_time(np.array([z]), H0, Om)
    f = lambda zz: M.GYR_PER_INV_H0 / H0 / ((1 + zz) * math.sqrt(Om * (1 + zz) ** 3 + 1 - Om))
    ref = integrate.quad(f, z, np.inf, epsabs=1e-12)[0]
    assert abs(t[0] - ref) < 1e-8
    assert abs(dt[0] + f(z)) < 1e-10


def test_cosmic_time_values():
    t, _ = M.cosmic_time(np.array([0.0, 0.5]), 67.74, 0.3089)
    assert abs(t[0] - 13.80) < 0.01 and abs(t[1] - 8.609) < 0.005   # Planck-15 textbook ages


# ---- A3-A5 smooth SFH (R2, R5, R6) -------------------------------------------------
LA_FULL = 5.0 + 0.05 * np.arange(107)


def test_sfh_closed_form_alpha_beta_one():
    # alpha=beta=1: int_0^t dt [x + 1/x]^-1 = (tau/2) ln(1 + (t/tau)^2)
    tau, t_obs = np.array([1.7, 0.4]), np.array([9.0, 3.0])
    dM = M.smooth_age_weights(tau, np.ones(2), np.ones(2), t_obs, LA_FULL)[0]
    assert np.allclose(dM.sum(1), 0.5 * tau * np.log1p((t_obs / tau) ** 2), rtol=1e-12)


def test_sfh_general_closed_form_hypergeometric():
    # int_0^t = tau x^(b+1)/(b+1) 2F1(1, c; 1+c; -x^(a+b)), c = (b+1)/(a+b), x = t/tau
    tau, al, be, t = 2.0, 2.5, 0.7, 1.9          # x < 1 keeps scipy's 2F1 inside its safe region
    dM = M.smooth_age_weights(*(np.array([v]) for v in (tau, al, be, t)), LA_FULL)[0]
    x = t / tau; c = (be + 1) / (al + be)
    ref = tau * x ** (be + 1) / (be + 1) * special.hyp2f1(1.0, c, 1.0 + c, -x ** (al + be))
    assert abs(dM.sum() - ref) < 1e-12 * ref


def test_sfh_bins_match_adaptive_quadrature():
    tau, al, be, t_obs = 3.1, 4.0, 0.3, 5.9
    dM = M.smooth_age_weights(*(np.array([v]) for v in (tau, al, be, t_obs)), LA_FULL)[0][0]
    A, _ = M.age_bin_edges_gyr(LA_FULL)
    f = lambda t: 1.0 / ((t / tau) ** al + (t / tau) ** -be)
    for i in (0, 30, 80, 95, 96, 97, 98, 106):
        lo, hi = max(0.0, t_obs - A[i + 1]), max(0.0, t_obs - A[i])
        ref = integrate.quad(f, lo, hi, epsabs=0, epsrel=1e-13)[0] if hi > lo else 0.0
        assert abs(dM[i] - ref) <= 1e-11 * max(ref, 1e-30), i
    assert np.all(dM[A[:-1] > t_obs] == 0.0)     # stars cannot be older than the universe


def test_constant_sfh_sums_to_formed_mass():
    # alpha = beta = 0  =>  SFR = M_formed/2 constant: each bin holds (its width in time)/2
    t_obs = np.array([7.3])
    dM = M.smooth_age_weights(np.array([2.0]), np.zeros(1), np.zeros(1), t_obs, LA_FULL)[0][0]
    A, _ = M.age_bin_edges_gyr(LA_FULL)
    width = np.maximum(0, t_obs - A[:-1]) - np.maximum(0, t_obs - A[1:])
    assert np.allclose(dM, 0.5 * width, rtol=1e-9, atol=1e-18)   # young bins: t_obs - age cancels ~1e-11
    assert abs(dM.sum() - 0.5 * t_obs[0]) < 1e-12


def test_sfh_partials_finite_difference():
    v = [np.array([2.3]), np.array([3.0]), np.array([1.2]), np.array([6.0])]
    out = M.smooth_age_weights(*v, LA_FULL)
    for p in range(4):
        h = 1e-6
        vp = [x.copy() for x in v]; vm = [x.copy() for x in v]
        vp[p] += h; vm[p] -= h
        fd = (M.smooth_age_weights(*vp, LA_FULL)[0] - M.smooth_age_weights(*vm, LA_FULL)[0]) / (2 * h)
        assert np.allclose(out[1 + p], fd, rtol=2e-6, atol=1e-9 * np.abs(fd).max()), p


# ---- A6-A7 burst --------------------------------------------------------------------
def test_triweight_closed_forms():
    assert M.triweight_pdf(np.array([0.0]))[0] == pytest.approx(35.0 / 96.0)       # Eq. A7 constant
    assert M.triweight_pdf(np.array([3.0, -3.0, 4.0])).max() == 0.0               # clipped at 3 sigma
    assert integrate.quad(lambda x: M.triweight_pdf(np.array([x]))[0], -3, 3)[0] == pytest.approx(1.0, abs=1e-12)
    assert integrate.quad(lambda x: x * x * M.triweight_pdf(np.array([x]))[0], -3, 3)[0] == pytest.approx(1.0, abs=1e-12)
    h = 1e-5                                                                      # "vanishing derivative at the clip"
    assert abs(M.triweight_pdf(np.array([3 - h]))[0]) / h < 1e-8
    xs = np.linspace(-3.5, 3.5, 29)
    for x in xs:
        ref = integrate.quad(lambda y: M.triweight_pdf(np.array([y]))[0], -3, min(max(x, -3), 3))[0]
        assert M.triweight_cdf(np.array([x]))[0] == pytest.approx(ref, abs=1e-12)


def test_burst_weights_properties():
    ltp, ltm = np.array([6.4, 7.0]), np.array([7.9, 8.5])
    P, dp, dm = M.burst_age_weights(ltp, ltm, LA_FULL)
    assert np.allclose(P.sum(1), 1.0, atol=1e-14) and np.all(P >= 0)
    _, e = M.age_bin_edges_gyr(LA_FULL)
    for r in range(2):       # "vanishes beyond the 3 sigma region": nothing older than T_max
        assert np.all(P[r][e[:-1] >= ltm[r]] == 0.0)
        assert np.all(P[r][e[1:] <= 2 * ltp[r] - ltm[r]] == 0.0)
    h = 1e-6
    fd = (M.burst_age_weights(ltp + h, ltm, LA_FULL)[0] - M.burst_age_weights(ltp - h, ltm, LA_FULL)[0]) / (2 * h)
    assert np.allclose(dp, fd, atol=1e-8)
    fd = (M.burst_age_weights(ltp, ltm + h, LA_FULL)[0] - M.burst_age_weights(ltp, ltm - h, LA_FULL)[0]) / (2 * h)
    assert np.allclose(dm, fd, atol=1e-8)


def test_fburst_zero_is_smooth_model(tiny, prior):
    th = _theta(prior, 3, 5, F_burst=0.0)
    w = M.weights(th, tiny)
    t_obs, _ = M.cosmic_time(th[:, 12], tiny.H0, tiny.Om)
    dM = M.smooth_age_weights(th[:, 1], th[:, 2], th[:, 3], t_obs, tiny.log10_age_yr)[0]
    assert np.allclose(w["a"], dM / dM.sum(1, keepdims=True), rtol=1e-14)
    assert np.allclose(w["a"].sum(1), 1.0, rtol=1e-13)


# ---- A.2 lognormal MDF (R9) -----------------------------------------------------------
def test_met_weights(tiny):
    lz, s = np.array([-0.4, 0.1]), np.array([0.3, 0.08])
    m, dlz, ds = M.met_weights(lz, s, tiny.log10_Z)
    assert np.allclose(m.sum(1), 1.0, atol=1e-15)
    g = tiny.log10_Z; mid = 0.5 * (g[1:] + g[:-1])
    for r in range(2):
        cdf = np.concatenate([[0], stats.norm.cdf(mid, lz[r], s[r]), [1]])
        assert np.allclose(m[r], np.diff(cdf), atol=1e-15)
    m0, _, _ = M.met_weights(np.array([-0.45]), np.array([1e-4]), g)          # sigma -> 0: one-hot at nearest Z
    assert m0[0].argmax() == np.abs(g + 0.45).argmin() and m0[0].max() == pytest.approx(1.0)
    h = 1e-6
    assert np.allclose(dlz, (M.met_weights(lz + h, s, g)[0] - M.met_weights(lz - h, s, g)[0]) / (2 * h), atol=1e-8)
    assert np.allclose(ds, (M.met_weights(lz, s + h, g)[0] - M.met_weights(lz, s - h, g)[0]) / (2 * h), atol=1e-8)


def test_bound_saturates_cleanly(prior):
    # HMC warmup reaches |k (theta~ - x0)| ~ 20-90 (Eq. C1): no overflow, theta inside [y_lo, y_hi], the
    # slope falls off as exp(-|x|), and the two branches agree with the textbook form where that one is finite
    import warnings
    x = np.array([-800.0, -90.0, -37.0, -20.0, -1.0, 0.0, 1.0, 20.0, 37.0, 90.0, 800.0])
    thu = prior[3][None, :] + x[:, None] / prior[2][None, :]
    with warnings.catch_warnings():
        warnings.simplefilter("error")
        th, d = M.bound(thu, prior)
    w = prior[1] - prior[0]
    assert np.all(np.isfinite(th)) and np.all(th >= prior[0]) and np.all(th <= prior[1] + 4e-16 * w) and np.all(d >= 0.0)
    ref = prior[0] + w / (1.0 + np.exp(-x[3:8]))[:, None]                  # Eq. (C1) as printed, |x| <= 20
    assert np.allclose(th[3:8], ref, rtol=1e-15)
    assert np.allclose(d[[1, 9]], (w * prior[2] * np.exp(-90.0))[None, :], rtol=1e-12)
    assert np.array_equal(th[0], prior[0]) and np.allclose(th[-1], prior[1], rtol=0, atol=4e-16 * w.max()) and np.all(d[[0, -1]] == 0.0)
    assert np.allclose(th[1] - prior[0], w * np.exp(-90.0), rtol=1e-12)     # lower tail keeps relative accuracy
