"""Pins of the sampler oracle (`oracle/sampler.py`): RNG known answers, integrator order,
detailed-balance consequences on a Gaussian target, adaptation targets.  CPU only."""
import math

import numpy as np
import pytest

from oracle import sampler as S


# ---- R16 Philox4x32-10: known-answer vectors published with the generator (Random123 kat_vectors) --------
def test_philox_known_answers():
    assert S.philox4x32((0, 0, 0, 0), (0, 0)) == (0x6627e8d5, 0xe169c58d, 0xbc57ac4c, 0x9b00dbd8)
    assert S.philox4x32((0xffffffff,) * 4, (0xffffffff,) * 2) == (0x408f276d, 0x41c83b0e, 0xa20bc7c6, 0x6d5451fd)
    assert S.philox4x32((0x243f6a88, 0x85a308d3, 0x13198a2e, 0x03707344), (0xa4093822, 0x299f31d0)) == \
        (0xd16cfe09, 0x94fdcceb, 0x5001e420, 0x24126ea1)


def test_uniform_and_normal_streams():
    assert S.u01(0) == 2.0 ** -25 and S.u01(0xffffffff) == 1 - 2.0 ** -25
    assert np.float32(S.u01(0x12345678)) == S.u01(0x12345678)            # exact in fp32
    x = np.concatenate([S.normals(7, c, 3, S.P_MOMENTUM, 13) for c in range(3000)])
    assert abs(x.mean()) < 0.02 and abs(x.var() - 1) < 0.03
    assert abs((x ** 3).mean()) < 0.05 and abs((x ** 4).mean() - 3) < 0.15
    a = S.normals(7, 5, 3, S.P_MOMENTUM, 13); b = S.normals(7, 5, 3, S.P_MOMENTUM, 13)
    assert np.array_equal(a, b) and not np.array_equal(a, S.normals(7, 5, 4, S.P_MOMENTUM, 13))


def test_warmup_windows():
    assert S.warmup_windows(500) == ([100, 150, 250, 450], (75, 450))     # 75 | 25,50,100,200 | 50
    assert S.warmup_windows(100) == ([90], (15, 90))
    assert S.warmup_windows(10) == ([], (10, 10))
    ends, (lo, hi) = S.warmup_windows(1000)
    assert ends[-1] == hi == 950 and lo == 75 and all(b > a for a, b in zip(ends, ends[1:]))


def test_checkpoint_ranges_are_the_aligned_subtrees():
    # at an odd leaf n the slots [idx_min, idx_max] must be exactly the subtrees [n+1-2^k, n], k>=1, aligned
    for depth in range(1, 7):
        slot_start = {}
        for n in range(1 << depth):
            lo, hi = S._ckpt_range(n)
            if n % 2 == 0:
                slot_start[hi] = n
            else:
                spans = sorted(n - slot_start[i] + 1 for i in range(lo, hi + 1))
                expect = [2 ** k for k in range(1, depth + 1) if (n + 1) % (2 ** k) == 0]
                assert spans == expect, (depth, n, spans, expect)


# ---- Gaussian target ---------------------------------------------------------------------------------
def _gauss(D=4, seed=0):
    rng = np.random.default_rng(seed)
    A = rng.normal(size=(D, D))
    cov = A @ A.T / D + np.diag(rng.uniform(0.2, 2.0, D))
    prec = np.linalg.inv(cov)
    mu = rng.normal(size=D)

    def f(th):
        d = th - mu
        return -0.5 * np.einsum("bi,ij,bj->b", d, prec, d), -d @ prec
    return f, mu, cov


def test_leapfrog_second_order_and_reversible():
    f, mu, cov = _gauss()
    th0 = mu[None, :] + 0.5; p0 = np.array([[0.3, -1.0, 0.7, 0.2]])
    inv_m = np.array([[1.0, 0.5, 2.0, 1.0]])
    lp0, g0 = f(th0)
    H0 = S.hamiltonian(lp0, p0, inv_m)
    errs = []
    for eps, n in ((0.1, 10), (0.05, 20), (0.025, 40)):
        th, p, lp, g = S.leapfrog(th0, p0, g0, eps, inv_m, f, n)
        errs.append(abs(S.hamiltonian(lp, p, inv_m) - H0)[0])
    assert 3.5 < errs[0] / errs[1] < 4.5 and 3.5 < errs[1] / errs[2] < 4.5     # energy error ~ eps^2
    th, p, lp, g = S.leapfrog(th0, p0, g0, 0.1, inv_m, f, 10)
    thb, pb, _, _ = S.leapfrog(th, -p, g, 0.1, inv_m, f, 10)
    assert np.allclose(thb, th0, atol=1e-12) and np.allclose(-pb, p0, atol=1e-12)


@pytest.mark.parametrize("sampler", ["hmc", "nuts"])
def test_gaussian_target_mean_and_variance(sampler):
    f, mu, cov = _gauss()
    B = 8
    th0 = np.tile(mu, (B, 1)) + np.random.default_rng(3).normal(size=(B, 4))
    n_s = 3000 if sampler == "hmc" else 700
    out = S.run_chains(th0, f, seed=11, n_warmup=300, n_sample=n_s, eps0=0.1, sampler=sampler,
                       n_leapfrog=3, max_depth=6)   # short fixed trajectories: L*eps ~ 2 pi resonates
    x = out["samples"].reshape(-1, 4)
    sd = np.sqrt(np.diag(cov))
    assert np.all(np.abs(x.mean(0) - mu) < 0.08 * sd)
    assert np.all(np.abs(x.std(0) / sd - 1) < 0.08)
    c = np.cov(x.T)
    assert np.allclose(c / np.outer(sd, sd), cov / np.outer(sd, sd), atol=0.08)
    # adaptation: accept statistic near the 0.8 target, inverse mass near the marginal variances
    # (the averaged step size eps_bar used after warmup is a little smaller than the last iterate, so the
    #  sampling-phase accept rate sits somewhat above the 0.8 target, as in the reference schemes)
    assert 0.75 < out["accept"].mean() < 0.97
    assert np.all(np.abs(np.log(out["inv_mass"].mean(0) / np.diag(cov))) < 0.5)
    assert out["divergences"].sum() == 0


def test_hmc_and_nuts_agree():
    # the samplers "produce very similar contours" on the same target
    f, mu, cov = _gauss(D=3, seed=5)
    th0 = np.tile(mu, (6, 1))
    a = S.run_chains(th0, f, 1, 200, 3000, 0.1, "hmc", n_leapfrog=3)["samples"].reshape(-1, 3)
    b = S.run_chains(th0, f, 2, 200, 600, 0.1, "nuts", max_depth=6)["samples"].reshape(-1, 3)
    sd = np.sqrt(np.diag(cov))
    assert np.all(np.abs(a.mean(0) - b.mean(0)) < 0.1 * sd)
    assert np.all(np.abs(a.std(0) / b.std(0) - 1) < 0.1)


def test_gaussian_target_definition():
    # SPS_MODEL_GAUSS_TEST: log density of N(mu, P^-1) up to a constant (scipy), gradient by central differences
    from scipy import stats
    rng = np.random.default_rng(4)
    A = rng.normal(size=(5, 5)); cov = A @ A.T + np.eye(5); mu = rng.normal(size=5)
    f = S.gaussian_target(mu, np.linalg.inv(cov))
    x = rng.normal(size=(7, 5))
    lp, g = f(x)
    ref = stats.multivariate_normal(mu, cov).logpdf(x)
    assert np.allclose(lp - lp[0], ref - ref[0], atol=1e-12)
    for p in range(5):
        e = np.zeros(5); e[p] = 1e-6
        assert np.allclose(g[:, p], (f(x + e)[0] - f(x - e)[0]) / 2e-6, atol=1e-7)


def test_nuts_transition_leaves_a_gaussian_invariant():
    # Detailed balance of the multinomial / biased-progressive sampling (R15): with a LARGE fixed step (energy errors of
    # tens of per cent, so the leaf weights and the subtree acceptance matter) the chain started in the stationary
    # distribution N(0, 1) must stay there: variance, quartile and tail mass to ~1 %.  A dropped weight, a uniform instead
    # of the biased subtree choice, or a wrong U-turn sign all fail this.
    f1 = lambda q: (-0.5 * float(q[0] * q[0]), -q)
    n_chain, n_tr, eps = 64, 330, 1.3
    x0 = np.concatenate([S.normals(99, c, 0, S.P_INIT, 1) for c in range(n_chain)])
    xs = []
    for c in range(n_chain):
        q = np.array([x0[c]])
        lp, g = f1(q)
        for it in range(n_tr):
            q, lp, g, acc, n_leaf, div, depth = S.nuts_transition(q, lp, g, eps, np.ones(1), 6, f1, 5, c, it)
            xs.append(q[0])
    xs = np.array(xs)
    n_eff = xs.size / 1.5
    assert abs(xs.mean()) < 3.0 / np.sqrt(n_eff)
    assert abs(xs.var() - 1.0) < 3.0 * np.sqrt(2.0 / n_eff)
    assert abs((np.abs(xs) < 0.6744897501960817).mean() - 0.5) < 3.0 * 0.5 / np.sqrt(n_eff)       # inter-quartile mass
    assert abs((np.abs(xs) > 1.959963984540054).mean() - 0.05) < 3.0 * np.sqrt(0.05 * 0.95 / n_eff)  # tail mass
