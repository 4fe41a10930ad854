"""Pins of the convergence diagnostics (`oracle/diagnostics.py`: Gelman-Rubin R-hat; batch-means ESS,
DESIGN.md R24/R25) against hand-computed cases and textbook limits.  CPU only."""
import numpy as np

from oracle import diagnostics as D


def test_rhat_hand_computed_cases():
    # two chains d + (-1)^t and -d + (-1)^t, n = 4, d = 1: within-chain variance 4/3 each (W = 4/3), chain means +-1
    # (B/n = 2), so R^2 = ((3/4)(4/3) + 2) / (4/3) = 2.25
    alt = np.array([1.0, -1.0, 1.0, -1.0])
    x = np.stack([1.0 + alt, -1.0 + alt])
    assert abs(D.rhat(x) - 1.5) < 1e-14
    # identical chains: B = 0, R = sqrt((n-1)/n)
    y = np.stack([alt, alt, alt])
    assert abs(D.rhat(y) - np.sqrt(0.75)) < 1e-14
    # invariance under shift and scale; vectorised over trailing axes
    z = np.random.default_rng(0).normal(size=(4, 50, 3))
    assert np.allclose(D.rhat(z), D.rhat(7.0 - 3.0 * z)) and D.rhat(z).shape == (3,)


def test_rhat_of_independent_draws_is_one_and_of_separated_chains_is_large():
    rng = np.random.default_rng(1)
    x = rng.normal(size=(4, 4000))
    assert abs(D.rhat(x) - 1.0) < 5e-3
    # chain means separated by delta sd: R^2 -> (n-1)/n + var(means)/W
    sep = x + np.array([0.0, 1.0, 2.0, 3.0])[:, None]
    expect = np.sqrt(3999 / 4000 + np.var(sep.mean(1), ddof=1) / sep.var(1, ddof=1).mean())
    assert abs(D.rhat(sep) - expect) < 1e-12 and D.rhat(sep) > 1.5


def test_ess_of_white_noise_and_of_an_ar1_process():
    rng = np.random.default_rng(2)
    m, n = 8, 40000
    x = rng.normal(size=(m, n))
    assert abs(D.ess_batch_means(x) / (m * n) - 1.0) < 0.05
    # AR(1) with coefficient phi: ESS / N -> (1 - phi) / (1 + phi)   (textbook integrated autocorrelation time)
    for phi in (0.5, 0.8):
        y = np.empty((m, n)); y[:, 0] = x[:, 0]
        for t in range(1, n):
            y[:, t] = phi * y[:, t - 1] + np.sqrt(1 - phi * phi) * x[:, t]
        assert abs(D.ess_batch_means(y) / (m * n) / ((1 - phi) / (1 + phi)) - 1.0) < 0.08, phi
    # an antithetic chain (phi < 0) has ESS > N
    phi = -0.5
    y = np.empty((m, n)); y[:, 0] = x[:, 0]
    for t in range(1, n):
        y[:, t] = phi * y[:, t - 1] + np.sqrt(1 - phi * phi) * x[:, t]
    assert D.ess_batch_means(y) > 2.0 * m * n


def test_ess_hand_computed_case():
    # one chain, n = 9, L = 3: samples 0..8 -> batch means 1, 4, 7 (variance 9), tau2 = 27; s2 = 7.5; ESS = 9 * 7.5 / 27
    x = np.arange(9.0)[None, :]
    assert abs(D.ess_batch_means(x) - 2.5) < 1e-14
    # n = 11: the two trailing samples stay out of the batch means but enter the variance
    x = np.concatenate([np.arange(9.0), [100.0, -100.0]])[None, :]
    assert abs(D.ess_batch_means(x) - 11 * x.var(ddof=1) / 27.0) < 1e-10
