"""Float64 CPU ORACLE of the convergence diagnostics reported beside the posteriors.

TEST INFRASTRUCTURE ONLY (same rules as `oracle/sps_model.py`; shares no code with the CUDA path).

  * `rhat`: the Gelman-Rubin statistic the paper checks convergence with ("check for convergence
    according to the Gelman-Rubin statistic ... R < 1.2").  The paper does not print the formula; the
    reading (R24) is the original one of Gelman & Rubin (1992) without the sampling-variability correction:
    for m chains of n kept samples, W = mean of the within-chain variances (n-1 denominators), B/n = variance of the
    chain means (m-1 denominator), R = sqrt(((n-1)/n W + B/n) / W).
  * `ess_batch_means`: effective sample size by non-overlapping batch means (the paper names no estimator: R25).
    Batch length L = floor(sqrt(n)), nb = floor(n/L) batches per chain (a trailing remainder is left out of the batch
    means, not out of the variances); tau2_c = L * variance of chain c's batch means (nb-1 denominator) estimates the
    asymptotic variance, s2_c = variance of all n samples of chain c; ESS = m n * mean_c s2_c / mean_c tau2_c.
"""
from __future__ import annotations

import math

import numpy as np


def rhat(samples):
    """samples [m, n, ...] (chain, kept sample, parameter...) -> R-hat [...]."""
    x = np.asarray(samples, float)
    m, n = x.shape[0], x.shape[1]
    chain_mean = x.mean(1)
    W = x.var(1, ddof=1).mean(0)
    B_over_n = chain_mean.var(0, ddof=1)
    return np.sqrt(((n - 1.0) / n * W + B_over_n) / W)


def ess_batch_means(samples):
    """samples [m, n, ...] -> ESS [...] pooled over the m chains."""
    x = np.asarray(samples, float)
    m, n = x.shape[0], x.shape[1]
    L = int(math.floor(math.sqrt(n)))
    nb = n // L
    bm = x[:, :nb * L].reshape((m, nb, L) + x.shape[2:]).mean(2)          # [m, nb, ...]
    tau2 = L * bm.var(1, ddof=1)                                          # [m, ...]
    s2 = x.var(1, ddof=1)
    return m * n * s2.mean(0) / tau2.mean(0)
