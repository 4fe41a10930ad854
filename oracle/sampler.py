"""Float64 CPU ORACLE of the sampler: counter-based RNG, leapfrog, HMC, warmup, NUTS.

TEST INFRASTRUCTURE ONLY (see `oracle/sps_model.py` for the rules).  Shares no code with the
CUDA path.  The paper names the algorithms (HMC with a leapfrog integrator, PAPER.md:452-460;
an adaptation phase; NUTS) but gives none of their details;
the readings taken are R13-R17 in DESIGN.md and are restated in each docstring.

The target is any callable  logp_grad(theta [B,D]) -> (logp [B], grad [B,D]).
"""
from __future__ import annotations

import math

import numpy as np

# ----------------------------------------------------------------------------------------------
# R16  Philox4x32-10 (Salmon, Moraes, Dror & Shaw 2011), counter = (chain, transition, purpose, index)
# ----------------------------------------------------------------------------------------------
_M0, _M1 = 0xD2511F53, 0xCD9E8D57
_W0, _W1 = 0x9E3779B9, 0xBB67AE85
_MASK = 0xFFFFFFFF

P_MOMENTUM, P_ACCEPT, P_DIRECTION, P_LEAF, P_SUBTREE, P_INIT = 0, 1, 2, 3, 4, 5


def philox4x32(counter, key):
    """counter: 4 uint32, key: 2 uint32 -> 4 uint32 (10 rounds)."""
    c0, c1, c2, c3 = (int(c) & _MASK for c in counter)
    k0, k1 = (int(k) & _MASK for k in key)
    for _ in range(10):
        p0 = _M0 * c0
        p1 = _M1 * c2
        hi0, lo0 = p0 >> 32, p0 & _MASK
        hi1, lo1 = p1 >> 32, p1 & _MASK
        c0, c1, c2, c3 = (hi1 ^ c1 ^ k0) & _MASK, lo1, (hi0 ^ c3 ^ k1) & _MASK, lo0
        k0 = (k0 + _W0) & _MASK
        k1 = (k1 + _W1) & _MASK
    return c0, c1, c2, c3


def u01(word):
    """u = ((x >> 8) + 0.5) 2^-24: exact in fp32 and fp64, never 0 or 1."""
    return ((int(word) >> 8) + 0.5) * 2.0 ** -24


def seed_key(seed):
    return (seed & _MASK, (seed >> 32) & _MASK)


def uniform(seed, chain, transition, purpose, index):
    return u01(philox4x32((chain, transition, purpose, index), seed_key(seed))[0])


def normals(seed, chain, transition, purpose, n):
    """n standard normals: block q = counter index q gives 4 words -> 4 uniforms -> two Box-Muller
    pairs (n0,n1) from (u0,u1) and (n2,n3) from (u2,u3): r = sqrt(-2 ln u_a), angle = 2 pi u_b."""
    out = np.empty(4 * ((n + 3) // 4))
    for q in range((n + 3) // 4):
        w = philox4x32((chain, transition, purpose, q), seed_key(seed))
        u = [u01(x) for x in w]
        for h in range(2):
            r = math.sqrt(-2.0 * math.log(u[2 * h]))
            out[4 * q + 2 * h] = r * math.cos(2.0 * math.pi * u[2 * h + 1])
            out[4 * q + 2 * h + 1] = r * math.sin(2.0 * math.pi * u[2 * h + 1])
    return out[:n]


# ----------------------------------------------------------------------------------------------
# a11  leapfrog and the HMC transition (R-step 13)
# ----------------------------------------------------------------------------------------------
def leapfrog(theta, p, grad, eps, inv_mass, logp_grad, n_steps, record=False):
    """n_steps of  p += eps/2 grad;  theta += eps invM*p;  p += eps/2 grad(theta).
    eps [B] or scalar, inv_mass [B,D] (diagonal).  Returns theta, p, logp, grad (+ trajectory)."""
    eps = np.asarray(eps, float).reshape(-1, 1)
    traj = []
    logp = None
    for _ in range(n_steps):
        p = p + 0.5 * eps * grad
        theta = theta + eps * inv_mass * p
        logp, grad = logp_grad(theta)
        p = p + 0.5 * eps * grad
        if record:
            traj.append((theta.copy(), p.copy(), logp.copy()))
    return (theta, p, logp, grad, traj) if record else (theta, p, logp, grad)


def hamiltonian(logp, p, inv_mass):
    """H = -logP + 1/2 sum_i invM_i p_i^2."""
    return -logp + 0.5 * (inv_mass * p * p).sum(-1)


def hmc_transition(theta, logp, grad, eps, inv_mass, n_leapfrog, logp_grad, seed, chain_ids, transition):
    """One fixed-length HMC transition for B chains.  Draw order: D normals (purpose 0), then one
    uniform (purpose 1).  Accept iff u < exp(H0 - HL); a non-finite proposal is a rejection.
    Returns theta, logp, grad, accept_prob [B], accepted [B]."""
    B, D = theta.shape
    xi = np.stack([normals(seed, int(c), transition, P_MOMENTUM, D) for c in chain_ids])
    p0 = xi / np.sqrt(inv_mass)
    H0 = hamiltonian(logp, p0, inv_mass)
    th1, p1, lp1, g1 = leapfrog(theta, p0, grad, eps, inv_mass, logp_grad, n_leapfrog)
    H1 = hamiltonian(lp1, p1, inv_mass)
    dH = H1 - H0
    ok = np.isfinite(dH) & np.isfinite(th1).all(1) & np.isfinite(g1).all(1)
    acc_prob = np.where(ok, np.minimum(1.0, np.exp(np.minimum(0.0, -np.where(ok, dH, 0.0)))), 0.0)
    u = np.array([uniform(seed, int(c), transition, P_ACCEPT, 0) for c in chain_ids])
    accept = ok & (u < acc_prob)
    theta = np.where(accept[:, None], th1, theta)
    logp = np.where(accept, lp1, logp)
    grad = np.where(accept[:, None], g1, grad)
    return theta, logp, grad, acc_prob, accept


# ----------------------------------------------------------------------------------------------
# a12  warmup (R14): Stan-style windows, dual averaging, Welford diagonal mass
# ----------------------------------------------------------------------------------------------
def warmup_windows(n_warmup):
    """End indices (exclusive, in warmup-iteration units) of the slow windows, and the slow-phase
    bounds (start, end).  500 -> 75 | 25,50,100,200 | 50.   <20 -> no mass adaptation."""
    W = n_warmup
    if W < 20:
        return [], (W, W)
    if W >= 150:
        init, term, base = 75, 50, 25
    else:
        init, term = int(0.15 * W), int(0.1 * W)
        base = W - init - term
    ends = []
    start, size, stop = init, base, W - term
    while start < stop:
        end = start + size
        if end + 2 * size > stop:
            end = stop
        ends.append(end)
        start = end
        size *= 2
    return ends, (init, stop)


class DualAveraging:
    """Hoffman & Gelman (2014) Alg. 5: gamma=0.05, t0=10, kappa=0.75, mu=log(10 eps)."""

    def __init__(self, eps, target):
        self.target = target
        self.restart(eps)

    def restart(self, eps):
        self.mu = np.log(10.0 * eps)
        self.hbar = np.zeros_like(eps)
        self.log_eps_bar = np.zeros_like(eps)
        self.m = 0

    def update(self, accept_stat):
        self.m += 1
        m = self.m
        self.hbar = (1.0 - 1.0 / (m + 10.0)) * self.hbar + (self.target - accept_stat) / (m + 10.0)
        log_eps = self.mu - math.sqrt(m) / 0.05 * self.hbar
        eta = m ** -0.75
        self.log_eps_bar = eta * log_eps + (1.0 - eta) * self.log_eps_bar
        return np.exp(log_eps)


def run_chains(theta0, logp_grad, seed, n_warmup, n_sample, eps0, sampler="hmc", n_leapfrog=16,
               max_depth=8, target_accept=0.8, chain_ids=None):
    """Warmup + sampling for B chains in lock-step.  Returns dict(samples [B,n_sample,D],
    accept [B] (mean accept statistic over sampling), eps [B], inv_mass [B,D], n_leapfrog_total [B],
    divergences [B] (sampling phase only))."""
    theta = np.array(theta0, float)
    B, D = theta.shape
    chain_ids = np.arange(B) if chain_ids is None else np.asarray(chain_ids)
    logp, grad = logp_grad(theta)
    eps = np.full(B, float(eps0))
    inv_mass = np.ones((B, D))
    ends, (slow_lo, slow_hi) = warmup_windows(n_warmup)
    da = DualAveraging(eps, target_accept)
    wn = 0; wmean = np.zeros((B, D)); wm2 = np.zeros((B, D))
    samples = np.empty((B, n_sample, D))
    acc_sum = np.zeros(B); nlf = np.zeros(B, int); ndiv = np.zeros(B, int)
    for it in range(n_warmup + n_sample):
        if sampler == "hmc":
            theta, logp, grad, acc, _ = hmc_transition(theta, logp, grad, eps, inv_mass, n_leapfrog, logp_grad,
                                                       seed, chain_ids, it)
            nlf += n_leapfrog
        else:
            acc = np.empty(B)
            for c in range(B):
                f1 = lambda q: tuple(x[0] for x in logp_grad(q[None, :]))
                th_c, lp_c, g_c, acc[c], n_c, div_c, _ = nuts_transition(
                    theta[c], logp[c], grad[c], eps[c], inv_mass[c], max_depth, f1, seed, int(chain_ids[c]), it)
                theta[c], logp[c], grad[c] = th_c, lp_c, g_c
                nlf[c] += n_c; ndiv[c] += div_c if it >= n_warmup else 0
        if it < n_warmup:
            eps = da.update(acc)
            if slow_lo <= it < slow_hi:
                wn += 1
                d = theta - wmean
                wmean += d / wn
                wm2 += d * (theta - wmean)
                if it + 1 in ends:
                    var = wm2 / (wn - 1)
                    inv_mass = (wn / (wn + 5.0)) * var + 1e-3 * (5.0 / (wn + 5.0))
                    wn = 0; wmean[:] = 0; wm2[:] = 0
                    da.restart(eps)
            if it + 1 == n_warmup:
                eps = np.exp(da.log_eps_bar)
        else:
            samples[:, it - n_warmup] = theta
            acc_sum += acc
    return dict(samples=samples, accept=acc_sum / max(n_sample, 1), eps=eps, inv_mass=inv_mass,
                n_leapfrog_total=nlf, divergences=ndiv)


# ----------------------------------------------------------------------------------------------
# a13  NUTS (R15): multinomial, iterative doubling with O(depth) checkpoints
# ----------------------------------------------------------------------------------------------
def _ckpt_range(n):
    """For leaf index n (0-based) in a subtree: slot range [idx_min, idx_max] of the checkpoints
    that close a power-of-two-aligned subtree at this leaf (n odd), or the slot to fill (n even)."""
    idx_max = bin(n >> 1).count("1")
    trailing = 0
    k = n
    while k & 1:
        trailing += 1
        k >>= 1
    return idx_max - trailing + 1, idx_max


def _uturn(rho, p_a, p_b, inv_mass):
    """Generalised criterion: continue only while rho.(invM p_a) > 0 and rho.(invM p_b) > 0."""
    return (np.dot(rho, inv_mass * p_a) <= 0.0) or (np.dot(rho, inv_mass * p_b) <= 0.0)


def nuts_transition(theta, logp, grad, eps, inv_mass, max_depth, logp_grad1, seed, chain, transition):
    """One multinomial-NUTS transition for ONE chain (theta [D]).  logp_grad1(theta [D]) -> (logp, grad [D]).
    Per doubling `depth`: direction forward iff uniform(purpose 2, index depth) < 1/2; the new subtree
    of 2^depth leaves is built leaf by leaf; leaf weight w = exp(H0 - H); inside the subtree the
    proposal is replaced by the new leaf with probability w / W_subtree (uniform(purpose 3,
    index depth*65536 + n)); the subtree's proposal replaces the tree's with probability
    min(1, W_subtree / W_tree) (uniform(purpose 4, index depth)); a subtree that diverges
    (H - H0 > 1000 or non-finite) or contains a U-turn on any aligned sub-subtree ends the transition and
    is discarded; after a merge the whole tree is tested.  Accept statistic: mean over leaves of
    min(1, exp(H0 - H)).  Returns theta, logp, grad, accept_stat, n_leapfrog, diverged, depth."""
    D = theta.shape[0]
    p0 = normals(seed, chain, transition, P_MOMENTUM, D) / np.sqrt(inv_mass)
    H0 = -logp + 0.5 * np.dot(inv_mass * p0, p0)
    left = (theta.copy(), p0.copy(), grad.copy())
    right = (theta.copy(), p0.copy(), grad.copy())
    prop = (theta.copy(), logp, grad.copy())
    rho = p0.copy()
    W = 1.0
    acc_sum, n_leaf, diverged, depth = 0.0, 0, 0, 0
    while depth < max_depth:
        fwd = uniform(seed, chain, transition, P_DIRECTION, depth) < 0.5
        q, p, g = right if fwd else left
        step = eps if fwd else -eps
        W_sub, rho_sub, prop_sub, bad = 0.0, np.zeros(D), None, False
        p_ck = np.zeros((max_depth + 1, D)); rho_ck = np.zeros((max_depth + 1, D))
        for n in range(1 << depth):
            p = p + 0.5 * step * g
            q = q + step * inv_mass * p
            lp, g = logp_grad1(q)
            p = p + 0.5 * step * g
            dH = -lp + 0.5 * np.dot(inv_mass * p, p) - H0
            if not (np.isfinite(dH) and np.isfinite(g).all()):
                dH = np.inf
            w = math.exp(-dH) if dH < 700 else 0.0
            acc_sum += min(1.0, w); n_leaf += 1
            if dH > 1000.0:
                diverged, bad = 1, True
                break
            W_sub += w
            rho_sub = rho_sub + p
            if uniform(seed, chain, transition, P_LEAF, depth * 65536 + n) * W_sub < w:
                prop_sub = (q.copy(), lp, g.copy())
            i_min, i_max = _ckpt_range(n)
            if n % 2 == 0:
                p_ck[i_max] = p; rho_ck[i_max] = rho_sub
            else:
                for i in range(i_max, i_min - 1, -1):
                    if _uturn(rho_sub - rho_ck[i] + p_ck[i], p_ck[i], p, inv_mass):
                        bad = True
                        break
                if bad:
                    break
        if bad:
            break
        if prop_sub is not None and uniform(seed, chain, transition, P_SUBTREE, depth) < min(1.0, W_sub / W):
            prop = prop_sub
        W += W_sub
        rho = rho + rho_sub
        if fwd:
            right = (q, p, g)
        else:
            left = (q, p, g)
        depth += 1
        if _uturn(rho, left[1], right[1], inv_mass):
            break
    return prop[0], prop[1], prop[2], acc_sum / max(n_leaf, 1), n_leaf, diverged, depth


def gaussian_target(mu, prec):
    """SPS_MODEL_GAUSS_TEST: logP(theta) = -1/2 (theta-mu)^T P (theta-mu), grad = -P (theta-mu), the
    correlated Gaussian on which north_star asks HMC and NUTS to recover the mean and the variance."""
    mu = np.asarray(mu, float); prec = np.asarray(prec, float)

    def f(th):
        d = np.asarray(th, float) - mu
        return -0.5 * np.einsum("bi,ij,bj->b", d, prec, d), -d @ prec.T
    return f


def init_chains(prior, seed, chain_ids, D):
    """R17: theta~_0 = xi + 0.1 omega N(0,1) from the chain's own stream (transition 0, purpose 5)."""
    xi, om = prior[4], prior[5]
    return np.stack([xi + 0.1 * om * normals(seed, int(c), 0, P_INIT, D) for c in chain_ids])
