"""Pins of the SPS_MODEL_TINY5 oracle (`oracle/tiny5.py`; BASELINE.json configs[0], R19): closed forms,
invariants, limits and finite differences.  CPU only."""
import math

import numpy as np
import pytest
from scipy import integrate

from oracle import sps_model as M
from oracle import tiny5 as T5
from paper_2506_19919_b200 import workloads as W


@pytest.fixture(scope="module")
def tiny():
    return W.make_grid("tiny")


@pytest.fixture(scope="module")
def prior4():
    return W.make_prior(model="tiny5").as_array()


def _theta(prior4, n, seed):
    return M.bound(W.draw_theta_unbounded(W.make_prior(model="tiny5"), n, seed), prior4)[0]


def test_gamma2_cdf_is_the_integral_of_the_delayed_exponential():
    # int t e^{-t/tau} dt = -tau (t + tau) e^{-t/tau}
    for t, tau in ((0.3, 1.0), (4.0, 0.7), (8.6, 5.0)):
        ref = integrate.quad(lambda s: s / tau ** 2 * math.exp(-s / tau), 0.0, t, epsabs=1e-14)[0]
        G, dG_dt, dG_dtau = T5.gamma2_cdf(np.array(t), np.array(tau))
        assert abs(G - ref) < 1e-13
        assert abs(G - (1.0 - (-tau * (t + tau) * math.exp(-t / tau)) / (-tau * tau))) < 1e-15
        h = 1e-6
        assert abs(dG_dt - (T5.gamma2_cdf(np.array(t + h), np.array(tau))[0] - T5.gamma2_cdf(np.array(t - h), np.array(tau))[0]) / (2 * h)) < 1e-9
        assert abs(dG_dtau - (T5.gamma2_cdf(np.array(t), np.array(tau + h))[0] - T5.gamma2_cdf(np.array(t), np.array(tau - h))[0]) / (2 * h)) < 1e-9


def test_weights_sum_to_one_and_match_bin_quadrature(tiny, prior4):
    th = _theta(prior4, 6, 1)
    z = np.full(6, W.TINY5_Z)
    w = T5.weights(th, z, tiny)
    assert np.allclose(w["a"].sum(1), 1.0, atol=1e-13) and np.allclose(w["m"].sum(1), 1.0, atol=1e-13)
    assert np.all(w["a"] >= 0.0)
    assert np.allclose(w["Mn"], 10.0 ** (th[:, 0] - tiny.log10_mass_unit))       # formed mass by t_obs = 10^logM_star
    # every bin against adaptive quadrature of the SFR over the bin's span of cosmic time
    A, _ = M.age_bin_edges_gyr(tiny.log10_age_yr)
    r = 2
    tau = 10.0 ** th[r, 1]; t_obs = w["t_obs"][r]
    norm = integrate.quad(lambda s: s * math.exp(-s / tau), 0.0, t_obs, epsabs=1e-14)[0]
    for i in range(tiny.n_age):
        hi = max(0.0, t_obs - A[i]); lo = max(0.0, t_obs - A[i + 1])
        ref = integrate.quad(lambda s: s * math.exp(-s / tau), lo, hi, epsabs=1e-16)[0] / norm if hi > lo else 0.0
        assert abs(w["a"][r, i] - ref) < 1e-12, i


def test_long_timescale_limit_is_a_linear_ramp(tiny, prior4):
    # tau >> t_obs: SFR proportional to t, so a_i proportional to t_hi^2 - t_lo^2
    th = _theta(prior4, 1, 2); th[0, 1] = 4.0                 # t/tau < 1e-3: deviations from the ramp are O(t/tau)
    w = T5.weights(th, np.array([0.5]), tiny)
    A, _ = M.age_bin_edges_gyr(tiny.log10_age_yr)
    t_obs = w["t_obs"][0]
    hi = np.maximum(0.0, t_obs - A[:-1]); lo = np.maximum(0.0, t_obs - A[1:])
    assert np.allclose(w["a"][0], (hi ** 2 - lo ** 2) / t_obs ** 2, rtol=2e-3, atol=1e-12)


def test_dust_law():
    F, dF = T5.attenuation(np.array([5500.0, 2750.0, 11000.0]), 0.8)
    assert abs(F[0] - math.exp(-0.8)) < 1e-15                                   # (lambda/5500)^-0.7 = 1 at 5500 A
    assert abs(F[1] - math.exp(-0.8 * 2.0 ** 0.7)) < 1e-15 and abs(F[2] - math.exp(-0.8 * 2.0 ** -0.7)) < 1e-15
    assert np.all(T5.attenuation(np.array([3000.0, 9000.0]), 0.0)[0] == 1.0)   # zero dust is the identity
    h = 1e-6
    fd = (T5.attenuation(np.array([4000.0]), 0.8 + h)[0] - T5.attenuation(np.array([4000.0]), 0.8 - h)[0]) / (2 * h)
    assert abs(fd - T5.attenuation(np.array([4000.0]), 0.8)[1]) < 1e-9


def test_fixed_scatter_mdf_is_the_13_parameter_mdf_at_0p2(tiny, prior4):
    th = _theta(prior4, 4, 3)
    w = T5.weights(th, np.full(4, 0.5), tiny)
    ref = M.met_weights(th[:, 2], np.full(4, 0.2), tiny.log10_Z)[0]
    assert np.array_equal(w["m"], ref)


def test_zero_dust_approx_equals_exact_on_a_z_node(tiny, prior4):
    # Eq. 6 == Eq. 4 when F_att is constant
    th = _theta(prior4, 3, 4); th[:, 3] = 0.0
    zg = M.z_grid(tiny)
    z = np.full(3, zg[3])
    fe = T5.photometry_exact(th, z, tiny, want_jac=False)[0]
    fa = T5.photometry_approx(th, z, tiny, M.cssp_table(tiny))[0]
    assert np.allclose(fe, fa, rtol=1e-12)
    # flux linear in 10^logM (R1)
    th2 = th.copy(); th2[:, 0] += 0.3
    assert np.allclose(T5.photometry_exact(th2, z, tiny, False)[0], fe * 10 ** 0.3, rtol=1e-12)


@pytest.mark.parametrize("path", ["exact", "approx"])
def test_gradient_matches_central_differences(tiny, prior4, path):
    cssp = M.cssp_table(tiny)
    prior = W.make_prior(model="tiny5")
    thu = W.draw_theta_unbounded(prior, 3, 5)
    z = np.array([0.5, 0.5, 0.93])                              # inside a z cell (R18)
    th = M.bound(thu, prior4)[0]
    f0 = T5.photometry_approx(th, z, tiny, cssp)[0]
    d, s = W.noisy_observations(f0, 6, 0.05, 0.05)
    lp, g, _ = T5.logp_and_grad(thu, z, tiny, prior4, d, s, path, cssp)
    for p in range(4):
        h = 1e-5
        e = np.zeros(4); e[p] = h
        lp1 = T5.logp_and_grad(thu + e, z, tiny, prior4, d, s, path, cssp)[0]
        lp0 = T5.logp_and_grad(thu - e, z, tiny, prior4, d, s, path, cssp)[0]
        fd = (lp1 - lp0) / (2 * h)
        assert np.allclose(g[:, p], fd, rtol=2e-6, atol=1e-6 * np.abs(g).max()), (p, g[:, p], fd)
