"""GPU parity tests of the models and features besides the 13-parameter hot path: SPS_MODEL_TINY5 (BASELINE.json configs[0] as
stated), SPS_MODEL_GAUSS_TEST (the samplers on a target whose answer is known), tabulated filters, the convergence
diagnostics (R-hat, ESS) against the oracle's, the exact path inside the samplers, saturated bounding sigmoids, config 5's
launch shape, continuing only the unconverged galaxies, the SPS_OPT_CHECK_FINITE option and per-stream scratch.
Everything is called through the C ABI; expected values come from `oracle/` at run time."""
import numpy as np
import pytest

from oracle import diagnostics as D
from oracle import sampler as S
from oracle import sps_model as M
from oracle import tiny5 as T5
from paper_2506_19919_b200 import workloads as W

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


def _sps():
    import paper_2506_19919_b200 as sps
    return sps


def _dev(a, dtype=None):
    return torch.tensor(np.asarray(a), dtype=dtype or torch.float32, device="cuda")


def _rel(a, b):
    return np.abs(a - b) / np.maximum(np.abs(b), 1e-300)


def _grad_err(g, ref, floor=1e-3):
    return np.abs(g - ref) / np.maximum(np.abs(ref), floor * np.abs(ref).max(1, keepdims=True))


def _pad(a, z=None):
    out = np.zeros((a.shape[0], 13), np.float32)
    out[:, :a.shape[1]] = a
    if z is not None:
        out[:, 4] = z
    return out


@pytest.fixture(params=["tcgen05", "simt_fp32"])
def kernels(request):
    """Both contraction kernel families of both paths."""
    sps = _sps()
    simt = int(request.param == "simt_fp32")
    sps.sps_set_option(sps.OPT_EXACT_SIMT, simt); sps.sps_set_option(sps.OPT_APPROX_SIMT, simt)
    yield request.param
    sps.sps_set_option(sps.OPT_EXACT_SIMT, 0); sps.sps_set_option(sps.OPT_APPROX_SIMT, 0)


# ---- SPS_MODEL_TINY5: BASELINE.json configs[0] as it states the model (R19) ------------------------------------
class Tiny5:
    def __init__(self):
        sps = _sps()
        self.sps = sps
        self.grid = W.make_grid("tiny")
        self.prior = W.make_prior(model="tiny5")
        self.P4 = self.prior.as_array()
        self.ph = sps.PriorHandle(W.pad_prior(self.prior, {4: W.TINY5_Z}))
        self.table = sps.sps_create_table(self.grid, model=sps.MODEL_TINY5)
        self.cssp = M.cssp_table(self.grid)

    def observations(self, n_gal, seed, frac=0.05):
        truth_u = W.draw_theta_unbounded(self.prior, n_gal, seed).astype(np.float32).astype(np.float64)
        z = np.full(n_gal, W.TINY5_Z)
        f = T5.photometry_approx(M.bound(truth_u, self.P4)[0], z, self.grid, self.cssp)[0]
        d, s = W.noisy_observations(f, seed + 1, frac, frac)
        return truth_u, d.astype(np.float32), s.astype(np.float32)


@pytest.fixture(scope="module")
def t5():
    return Tiny5()


def test_tiny5_table_reports_four_sampled_parameters(t5):
    assert t5.table.n_dim == 4


def test_tiny5_weights(t5):
    n = 300
    thu = W.draw_theta_unbounded(t5.prior, n, 5).astype(np.float32)
    z = np.random.default_rng(0).uniform(0.1, 2.9, n).astype(np.float32)
    th = M.bound(thu.astype(np.float64), t5.P4)[0]
    ow = T5.weights(th, z.astype(np.float64), t5.grid)
    wa, wm, ms = (x.cpu().numpy().astype(np.float64) for x in t5.sps.sps_weights(t5.table, t5.ph, _dev(_pad(thu, z))))
    for got, ref in ((wa, ow["a"]), (wm, ow["m"])):
        mx = ref.max(1, keepdims=True)
        assert (np.abs(got - ref) / mx).max() <= 1e-5
        mask = ref > 1e-6 * mx
        assert _rel(got, ref)[mask].max() <= 1e-4
    assert _rel(ms, ow["Mn"]).max() <= 1e-5
    assert np.allclose(wa.sum(1), 1.0, atol=1e-5)


def test_tiny5_flux_and_loglike_grad(t5, kernels):
    n_gal, n_chain = 24, 3
    truth_u, d, s = t5.observations(n_gal, 31)
    thu = (np.repeat(truth_u, n_chain, 0) + 0.3 * np.random.default_rng(2).normal(size=(n_gal * n_chain, 4)) / t5.P4[2]).astype(np.float32)
    gal = np.repeat(np.arange(n_gal), n_chain).astype(np.int32)
    z = np.full(n_gal * n_chain, W.TINY5_Z)
    th, dth = M.bound(thu.astype(np.float64), t5.P4)
    for path, name in ((t5.sps.PATH_APPROX, "approx"), (t5.sps.PATH_EXACT, "exact")):
        flux = t5.sps.sps_photometry(t5.table, t5.ph, path, _dev(_pad(thu, z))).cpu().numpy()
        of, J = (T5.photometry_approx(th, z, t5.grid, t5.cssp) if name == "approx" else T5.photometry_exact(th, z, t5.grid))
        assert _rel(flux, of).max() <= 1e-4, name
        # per-band Jacobians (no cross-band cancellation): the north_star rule as it stands
        for b in range(t5.grid.n_band):
            fb = np.zeros((thu.shape[0], t5.grid.n_band), np.float32); fb[:, b] = 1.0
            _, tb = t5.sps.sps_photometry(t5.table, t5.ph, path, _dev(_pad(thu, z)), True, _dev(fb))
            tb = tb.cpu().numpy()
            assert _grad_err(tb[:, :4], J[:, b, :] * dth).max() <= 1e-3, (name, b)
            assert np.all(tb[:, 4:] == 0.0)                            # unsampled slots carry no gradient
        lp, g = t5.sps.sps_loglike_grad(t5.table, t5.ph, path, _dev(_pad(thu, z)), _dev(d), _dev(s), _dev(gal, torch.int32))
        olp, og, _ = T5.logp_and_grad(thu.astype(np.float64), z, t5.grid, t5.P4, d[gal].astype(np.float64), s[gal].astype(np.float64), name, t5.cssp)
        assert (np.abs(lp.cpu().numpy() - olp) / np.maximum(1.0, np.abs(olp))).max() <= 1e-4, name
        g = g.cpu().numpy()
        allow = FLUX_EPS[name] * np.einsum("rb,rbp->rp", of / s[gal].astype(np.float64) ** 2, np.abs(J)) * dth      # DESIGN.md R23
        err = np.maximum(np.abs(g[:, :4] - og) - allow, 0.0)
        assert (err / np.maximum(np.abs(og), 1e-3 * np.abs(og).max(1, keepdims=True))).max() <= 1e-3, name


# R23: the flux-error allowance of log-likelihood gradients near the mode, relative flux error per path
FLUX_EPS = {"approx": 4e-6, "exact": 2e-5}


def test_tiny5_leapfrog_trajectory(t5):
    # first-20-leapfrog-step trajectories within 1e-4 (north_star), both paths
    n = 16
    truth_u, d, s = t5.observations(n, 41)
    th0 = (truth_u + 0.2 * np.random.default_rng(3).normal(size=(n, 4)) / t5.P4[2]).astype(np.float32)
    z = np.full(n, W.TINY5_Z)
    inv_m = np.tile((0.5 / t5.P4[2]) ** 2, (n, 1)).astype(np.float32)
    p0 = (np.random.default_rng(4).normal(size=(n, 4)) / np.sqrt(inv_m)).astype(np.float32)
    eps = np.full(n, 0.01, np.float32)
    for path, name in ((t5.sps.PATH_APPROX, "approx"), (t5.sps.PATH_EXACT, "exact")):
        traj, _ = t5.sps.sps_leapfrog(t5.table, t5.ph, path, _dev(_pad(th0, z)), _dev(_pad(p0)), _dev(eps), _dev(_pad(inv_m) + (np.arange(13) >= 4)),
                                      _dev(d), _dev(s), 20)
        f = lambda th: T5.logp_and_grad(th, z, t5.grid, t5.P4, d.astype(np.float64), s.astype(np.float64), name, t5.cssp)[:2]
        lp0, g0 = f(th0.astype(np.float64))
        ref = S.leapfrog(th0.astype(np.float64), p0.astype(np.float64), g0, eps.astype(np.float64), inv_m.astype(np.float64), f, 20, record=True)[4]
        traj = traj.cpu().numpy()
        for k in range(20):
            assert (np.abs(traj[k, :, 0, :4] - ref[k][0]) / np.maximum(1.0, np.abs(ref[k][0]))).max() <= 1e-4, (name, k)
            assert (np.abs(traj[k, :, 1, :4] - ref[k][1]) / np.maximum(1.0, np.abs(ref[k][1]))).max() <= 1e-3, (name, k)
            assert np.all(traj[k, :, 0, 4] == np.float32(W.TINY5_Z)) and np.all(traj[k, :, 1, 4:] == 0.0)       # z is data: it never moves


def test_config1_full_run_matches_oracle(t5):
    # BASELINE.json configs[0] as stated: 20 x 4 x 500 grid, 3 filters, 8 galaxies x 4 chains, 5 parameters with z = 0.5 fixed,
    # 5 % noise, HMC 200 steps of 10 leapfrog steps (no warmup).  The whole oracle chain runs beside the GPU under the shared
    # Philox streams; chains stay coupled until an accept decision splits in the last bits.
    n_gal, n_chain, n_sample, L, eps0, seed = 8, 4, 200, 10, 0.01, W.CONFIGS["c1_tiny_hmc"]["seed"]
    truth_u, d, s = t5.observations(n_gal, 51)
    gal = np.repeat(np.arange(n_gal), n_chain)
    z = np.full(n_gal * n_chain, W.TINY5_Z)
    out = t5.sps.sps_hmc_run(t5.table, t5.ph, _dev(d), _dev(s), sampler=t5.sps.SAMPLER_HMC, path=t5.sps.PATH_APPROX, n_chain=n_chain,
                             n_warmup=0, n_sample=n_sample, n_leapfrog=L, eps0=eps0, seed=seed, keep_samples=True)
    got = {k: v.cpu().numpy() for k, v in out.items()}
    f = lambda th: T5.logp_and_grad(th, z, t5.grid, t5.P4, d[gal].astype(np.float64), s[gal].astype(np.float64), "approx", t5.cssp)[:2]
    th0 = S.init_chains(t5.P4, seed, np.arange(n_gal * n_chain), 4)
    ref = S.run_chains(th0, f, seed, 0, n_sample, eps0, "hmc", n_leapfrog=L)
    gs, rs = got["samples"][:, :, :4], ref["samples"]
    assert np.all(got["samples"][:, :, 4] == np.float32(W.TINY5_Z)) and np.all(got["samples"][:, :, 5:] == 0.0)
    err = (np.abs(gs - rs) / np.maximum(1.0, np.abs(rs))).max(2)                # [chain, transition]
    assert err[:, :2].max() <= 1e-4                                             # 2 transitions = the first 20 leapfrog steps of every chain
    assert err[:, :20].max() <= 2e-3                                            # 200 leapfrog steps on: fp32 / fp64 rounding has grown, no decision has split
    ok = err.max(1) <= 1e-2                                                     # chains whose accept decisions never split
    assert ok.mean() >= 0.85
    mu_r, sd_r = rs.mean(1), rs.std(1, ddof=1)
    assert (np.abs(got["mean"][:, :4] - mu_r)[ok] <= 0.05 * sd_r[ok] + 1e-6).all()       # posterior mean / sd within 0.05 sigma
    assert (np.abs(got["sd"][:, :4] - sd_r)[ok] <= 0.05 * sd_r[ok] + 1e-6).all()
    assert np.abs(got["accept"] - ref["accept"])[ok].max() <= 0.02
    assert 0.3 < ref["accept"].mean() < 0.999                                   # the chains do move and do reject
    assert (got["n_leapfrog"] == n_sample * L).all()
    # convergence diagnostics: the device's R-hat / ESS are the oracle's formulas applied to the device's
    # samples, and agree with the oracle's own chains where every chain of the galaxy stayed coupled
    s4 = gs.reshape(n_gal, n_chain, n_sample, 4)
    r_dev = np.stack([D.rhat(s4[g]) for g in range(n_gal)]); e_dev = np.stack([D.ess_batch_means(s4[g]) for g in range(n_gal)])
    assert np.allclose(got["rhat"][:, :4], r_dev, rtol=2e-3) and np.all(got["rhat"][:, 4:] == 1.0)
    assert np.allclose(got["ess"][:, :4], e_dev, rtol=2e-2)
    r_ref = np.stack([D.rhat(rs.reshape(n_gal, n_chain, n_sample, 4)[g]) for g in range(n_gal)])
    gal_ok = ok.reshape(n_gal, n_chain).all(1)
    assert gal_ok.sum() >= 4 and np.allclose(got["rhat"][gal_ok, :4], r_ref[gal_ok], rtol=2e-2)


# ---- SPS_MODEL_GAUSS_TEST: the CUDA samplers on a target whose answer is known (north_star) -------------------------------
def _gauss_problem(Dm=5, seed=0):
    rng = np.random.default_rng(seed)
    A = rng.normal(size=(Dm, Dm))
    cov = A @ A.T / Dm + np.diag(rng.uniform(0.2, 2.0, Dm))
    mu = rng.normal(size=Dm)
    return mu, cov, np.linalg.inv(cov)


@pytest.mark.parametrize("sampler", ["hmc", "nuts"])
def test_gaussian_target_mean_and_variance(sampler):
    sps = _sps()
    mu, cov, prec = _gauss_problem()
    Dm = mu.size
    table = sps.sps_create_table(None, model=sps.MODEL_GAUSS_TEST, gauss=(mu, prec))
    assert table.n_dim == Dm
    n_gal, n_chain = 16, 8
    th0 = np.zeros((n_gal * n_chain, 13), np.float32)
    th0[:, :Dm] = mu + np.random.default_rng(3).normal(size=(n_gal * n_chain, Dm))
    kw = dict(n_leapfrog=3) if sampler == "hmc" else dict(max_depth=6)
    out = sps.sps_hmc_run(table, None, None, None, n_gal=n_gal, sampler=sps.SAMPLER_HMC if sampler == "hmc" else sps.SAMPLER_NUTS,
                          n_chain=n_chain, n_warmup=300, n_sample=1500, eps0=0.1, seed=11, theta0=_dev(th0), keep_samples=True, **kw)
    x = out["samples"].cpu().numpy()[:, :, :Dm].reshape(-1, Dm).astype(np.float64)
    sd = np.sqrt(np.diag(cov))
    assert np.all(np.abs(x.mean(0) - mu) < 0.03 * sd)
    assert np.all(np.abs(x.std(0) / sd - 1) < 0.03)
    assert np.allclose(np.cov(x.T) / np.outer(sd, sd), cov / np.outer(sd, sd), atol=0.03)
    assert 0.7 < out["accept"].mean().item() < 0.98
    im = out["inv_mass"].cpu().numpy()[:, :Dm]
    assert np.all(np.abs(np.log(np.median(im, 0) / np.diag(cov))) < 0.4)                  # adapted masses ~ marginal variances
    assert (out["divergences"].cpu().numpy() == 0).all()
    assert np.all(out["samples"].cpu().numpy()[:, :, Dm:] == 0.0)
    rh = out["rhat"].cpu().numpy()[:, :Dm]
    assert np.all(rh < 1.05)
    ess = out["ess"].cpu().numpy()[:, :Dm]
    assert np.all(ess > 0.05 * n_chain * 1500)
    if sampler == "nuts":
        hist = out["depth_hist"].cpu().numpy()
        assert hist.sum() == n_gal * n_chain * 1500 and hist[0] == 0 and hist[7:].sum() == 0
    # and the first transitions follow the oracle's sampler on the same target under the shared RNG streams
    f = S.gaussian_target(mu, prec)
    short = sps.sps_hmc_run(table, None, None, None, n_gal=2, sampler=sps.SAMPLER_HMC if sampler == "hmc" else sps.SAMPLER_NUTS, n_chain=2,
                            n_warmup=0, n_sample=12, eps0=0.2, seed=5, theta0=_dev(th0[:4]), keep_samples=True, **kw)
    ref = S.run_chains(th0[:4, :Dm].astype(np.float64), f, 5, 0, 12, 0.2, sampler, n_leapfrog=3, max_depth=6)
    assert np.abs(short["samples"].cpu().numpy()[:, :, :Dm] - ref["samples"]).max() <= 2e-4
    assert (short["n_leapfrog"].cpu().numpy() == ref["n_leapfrog_total"]).all()


def test_gaussian_target_loglike_grad():
    sps = _sps()
    mu, cov, prec = _gauss_problem(7, 1)
    table = sps.sps_create_table(None, model=sps.MODEL_GAUSS_TEST, gauss=(mu, prec))
    th = np.zeros((100, 13), np.float32); th[:, :7] = np.random.default_rng(2).normal(size=(100, 7))
    lp, g = sps.sps_loglike_grad(table, None, sps.PATH_APPROX, _dev(th), None, None)
    olp, og = S.gaussian_target(mu, prec)(th[:, :7].astype(np.float64))
    assert np.allclose(lp.cpu().numpy(), olp, rtol=1e-5, atol=1e-5) and np.allclose(g.cpu().numpy()[:, :7], og, rtol=1e-5, atol=1e-5)
    assert np.all(g.cpu().numpy()[:, 7:] == 0.0)


# ---- the 13-parameter model: what round 1 left untested against the oracle ------------------------------------------------
class Ctx:
    def __init__(self, kind, **kw):
        sps = _sps()
        self.sps = sps
        self.grid = W.make_grid(kind)
        self.prior = W.make_prior()
        self.P = self.prior.as_array()
        self.ph = sps.PriorHandle(self.P)
        self.table = sps.sps_create_table(self.grid, **kw)
        self._cssp = None

    def cssp(self):
        if self._cssp is None:
            self._cssp = M.cssp_table(self.grid)
        return self._cssp

    def observations(self, n_gal, seed, path="approx", frac=(0.05, 0.05)):
        truth_u = W.draw_theta_unbounded(self.prior, n_gal, seed).astype(np.float32).astype(np.float64)
        truth = M.bound(truth_u, self.P)[0]
        f = M.photometry_approx(truth, self.grid, self.cssp())[0] if path == "approx" else M.photometry_exact(truth, self.grid, False)[0]
        d, s = W.noisy_observations(f, seed + 1, *frac)
        return truth_u, d.astype(np.float32), s.astype(np.float32)


@pytest.fixture(scope="module")
def tiny():
    return Ctx("tiny")


@pytest.fixture(scope="module")
def full():
    return Ctx("full")


def test_exact_path_leapfrog_trajectory_and_hmc(tiny):
    # the exact path inside the integrator and the sampler, against the oracle (round 1 covered the approximate path only)
    cx = tiny
    n = 12
    truth_u, d, s = cx.observations(n, 43, path="exact")
    th0 = (truth_u + 0.2 * np.random.default_rng(3).normal(size=(n, 13)) / cx.P[2]).astype(np.float32)
    inv_m = np.tile((0.5 / cx.P[2]) ** 2, (n, 1)).astype(np.float32)
    p0 = (np.random.default_rng(4).normal(size=(n, 13)) / np.sqrt(inv_m)).astype(np.float32)
    eps = np.full(n, 0.01, np.float32)
    traj, _ = cx.sps.sps_leapfrog(cx.table, cx.ph, cx.sps.PATH_EXACT, _dev(th0), _dev(p0), _dev(eps), _dev(inv_m), _dev(d), _dev(s), 20)
    f = lambda th: M.logp_and_grad(th, cx.grid, cx.P, d.astype(np.float64), s.astype(np.float64), "exact")[:2]
    lp0, g0 = f(th0.astype(np.float64))
    ref = S.leapfrog(th0.astype(np.float64), p0.astype(np.float64), g0, eps.astype(np.float64), inv_m.astype(np.float64), f, 20, record=True)[4]
    traj = traj.cpu().numpy()
    for k in range(20):
        assert (np.abs(traj[k, :, 0] - ref[k][0]) / np.maximum(1.0, np.abs(ref[k][0]))).max() <= 1e-4, k
        assert (np.abs(traj[k, :, 1] - ref[k][1]) / np.maximum(1.0, np.abs(ref[k][1]))).max() <= 1e-3, k
    # a short HMC run on the exact path, coupled to the oracle under the shared RNG streams
    n_gal, n_chain, n_sample, L, eps0, seed = 3, 2, 30, 6, 0.004, 17
    gal = np.repeat(np.arange(n_gal), n_chain)
    out = cx.sps.sps_hmc_run(cx.table, cx.ph, _dev(d[:n_gal]), _dev(s[:n_gal]), sampler=cx.sps.SAMPLER_HMC, path=cx.sps.PATH_EXACT, n_chain=n_chain,
                             n_warmup=0, n_sample=n_sample, n_leapfrog=L, eps0=eps0, seed=seed, keep_samples=True)
    fh = lambda th: M.logp_and_grad(th, cx.grid, cx.P, d[gal].astype(np.float64), s[gal].astype(np.float64), "exact")[:2]
    refr = S.run_chains(S.init_chains(cx.P, seed, np.arange(n_gal * n_chain), 13), fh, seed, 0, n_sample, eps0, "hmc", n_leapfrog=L)
    err = (np.abs(out["samples"].cpu().numpy() - refr["samples"]) / np.maximum(1.0, np.abs(refr["samples"]))).max(2)
    assert err[:, :10].max() <= 1e-3
    assert (err.max(1) <= 1e-2).mean() >= 0.66
    assert np.abs(out["accept"].cpu().numpy() - refr["accept"])[err.max(1) <= 1e-2].max() <= 0.05


def test_saturated_sigmoid(tiny, kernels):
    # HMC warmup drives k (theta~ - x0) to tens (Eq. C1): theta pinned at a bound, zero slope; the weights, the
    # log-posterior and the gradient must stay finite and follow the oracle
    cx = tiny
    n = 48
    rng = np.random.default_rng(7)
    thu = W.draw_theta_unbounded(cx.prior, n, 9)
    x = np.array([-90.0, -37.0, -20.0, 20.0, 37.0, 90.0])
    for r in range(n):                                                      # one to three saturated parameters per row
        for p in rng.choice(13, rng.integers(1, 4), replace=False):
            if p == 6 and x[r % 6] < 0 or p == 5 and x[r % 6] > 0:
                continue                                                    # keep logT_max > logT_peak by a margin (Eq. A7)
            thu[r, p] = cx.P[3][p] + x[(r + p) % 6] / cx.P[2][p]
    thu = thu.astype(np.float32)
    th, dth = M.bound(thu.astype(np.float64), cx.P)
    ow = M.weights(th, cx.grid)
    wa, wm, ms = (v.cpu().numpy().astype(np.float64) for v in cx.sps.sps_weights(cx.table, cx.ph, _dev(thu)))
    assert np.isfinite(wa).all() and (np.abs(wa - ow["a"]) / ow["a"].max(1, keepdims=True)).max() <= 1e-5
    assert np.abs(wm - ow["m"]).max() <= 1e-5 and _rel(ms, ow["Mn"]).max() <= 1e-5
    _, d, s = cx.observations(n, 71)
    for path, name in ((cx.sps.PATH_APPROX, "approx"), (cx.sps.PATH_EXACT, "exact")):
        lp, g = cx.sps.sps_loglike_grad(cx.table, cx.ph, path, _dev(thu), _dev(d), _dev(s))
        olp, og, of = M.logp_and_grad(thu.astype(np.float64), cx.grid, cx.P, d.astype(np.float64), s.astype(np.float64), name, cx.cssp())
        lp, g = lp.cpu().numpy(), g.cpu().numpy()
        assert np.isfinite(lp).all() and np.isfinite(g).all()
        lp_allow = FLUX_EPS[name] * (np.abs(of - d) * of / s.astype(np.float64) ** 2).sum(1)             # R23 on the log-posterior
        assert (np.maximum(np.abs(lp - olp) - lp_allow, 0.0) / np.maximum(1.0, np.abs(olp))).max() <= 1e-4, name
        # these rows sit far from their data (chi^2 of thousands): the plain north_star rule applies
        assert _grad_err(g, og).max() <= 1e-3, name


def test_config5_launch_shape_sampled(full):
    # BASELINE.json configs[4]'s launch: 100,000 galaxies x 4 chains, the exact path on a seeded 10 % of the galaxies
    # (40,000 rows) and the approximate path on the rest (360,000 rows); 32 sampled rows of each against the oracle
    cx = full
    cfg = W.CONFIGS["c5_nuts"]
    n_gal, n_chain = cfg["n_gal"], cfg["n_chain"]
    mask = np.random.default_rng(cfg["seed"]).random(n_gal) >= cfg["exact_fraction"]                      # True = approximate
    truth_u = W.draw_theta_unbounded(cx.prior, n_gal, cfg["seed"]).astype(np.float32)
    rng = np.random.default_rng(12)
    for approx, path, name, eps_flux in ((True, cx.sps.PATH_APPROX, "approx", FLUX_EPS["approx"]), (False, cx.sps.PATH_EXACT, "exact", FLUX_EPS["exact"])):
        gals = np.nonzero(mask == approx)[0]
        tu = truth_u[gals]
        f = cx.sps.sps_photometry(cx.table, cx.ph, path, _dev(tu)).cpu().numpy().astype(np.float64)
        d, s = W.noisy_observations(f, 9, 0.05, 0.10)
        d = d.astype(np.float32); s = s.astype(np.float32)
        gal = np.repeat(np.arange(gals.size), n_chain).astype(np.int32)
        thu = (np.repeat(tu, n_chain, 0) + 0.25 * rng.normal(size=(gals.size * n_chain, 13)) / cx.P[2]).astype(np.float32)
        assert thu.shape[0] in (range(355000, 365001) if approx else range(39000, 41001))
        lp, g = cx.sps.sps_loglike_grad(cx.table, cx.ph, path, _dev(thu), _dev(d), _dev(s), _dev(gal, torch.int32))
        sel = rng.choice(thu.shape[0], 32, replace=False)
        olp, og, of = M.logp_and_grad(thu[sel].astype(np.float64), cx.grid, cx.P, d[gal[sel]].astype(np.float64), s[gal[sel]].astype(np.float64),
                                      name, cx.cssp() if approx else None)
        # log-posterior: 1e-4 relative plus the same propagated flux error (R23): eps sum_b |f_b - d_b| f_b / sigma_b^2
        lp_allow = eps_flux * (np.abs(of - d[gal[sel]]) * of / s[gal[sel]].astype(np.float64) ** 2).sum(1)
        assert (np.maximum(np.abs(lp.cpu().numpy()[sel] - olp) - lp_allow, 0.0) / np.maximum(1.0, np.abs(olp))).max() <= 1e-4, name
        th, dth = M.bound(thu[sel].astype(np.float64), cx.P)
        J = (M.photometry_approx(th, cx.grid, cx.cssp()) if approx else M.photometry_exact(th, cx.grid))[1]
        allow = eps_flux * np.einsum("rb,rbp->rp", of / s[gal[sel]].astype(np.float64) ** 2, np.abs(J)) * dth       # DESIGN.md R23
        err = np.maximum(np.abs(g.cpu().numpy()[sel] - og) - allow, 0.0)
        assert (err / np.maximum(np.abs(og), 1e-3 * np.abs(og).max(1, keepdims=True))).max() <= 1e-3, name


def test_exact_path_is_reproducible(full):
    # the band sums are combined by integer atomics: a row's fluxes and gradients do not depend on the rows it shares a
    # launch with, on their order, or on the run
    cx = full
    n = 700
    thu = W.draw_theta_unbounded(cx.prior, n, 77, z_uniform=(0.1, 2.9)).astype(np.float32)
    fb = np.random.default_rng(1).normal(size=(n, cx.grid.n_band)).astype(np.float32)
    f1, g1 = cx.sps.sps_photometry(cx.table, cx.ph, cx.sps.PATH_EXACT, _dev(thu), True, _dev(fb))
    f2, g2 = cx.sps.sps_photometry(cx.table, cx.ph, cx.sps.PATH_EXACT, _dev(thu), True, _dev(fb))
    assert torch.equal(f1, f2) and torch.equal(g1, g2)
    perm = np.random.default_rng(2).permutation(n)
    f3, g3 = cx.sps.sps_photometry(cx.table, cx.ph, cx.sps.PATH_EXACT, _dev(thu[perm]), True, _dev(fb[perm]))
    assert torch.equal(f3, f1[_dev(perm, torch.int64)])
    sub = perm[:97]
    f4 = cx.sps.sps_photometry(cx.table, cx.ph, cx.sps.PATH_EXACT, _dev(thu[sub]))
    assert torch.equal(f4, f1[_dev(sub, torch.int64)])


# ---- tabulated filters (R4) -----------------------------------------------------------------------------
def test_tabulated_filters(kernels):
    cx = Ctx("tiny_tab")
    c = cx.sps.sps_table_cssp(cx.table).astype(np.float64)
    ref = cx.cssp()
    maskc = ref > 1e-6 * ref.max()
    assert _rel(c, ref)[maskc].max() <= 1e-5
    n_gal, n_chain = 30, 3
    truth_u, d, s = cx.observations(n_gal, 91, frac=(0.05, 0.10))
    thu = (np.repeat(truth_u, n_chain, 0) + 0.3 * np.random.default_rng(2).normal(size=(n_gal * n_chain, 13)) / cx.P[2]).astype(np.float32)
    gal = np.repeat(np.arange(n_gal), n_chain).astype(np.int32)
    th, dth = M.bound(thu.astype(np.float64), cx.P)
    for path, name in ((cx.sps.PATH_APPROX, "approx"), (cx.sps.PATH_EXACT, "exact")):
        of, J = (M.photometry_approx(th, cx.grid, cx.cssp()) if name == "approx" else M.photometry_exact(th, cx.grid))
        flux = cx.sps.sps_photometry(cx.table, cx.ph, path, _dev(thu)).cpu().numpy()
        assert _rel(flux, of).max() <= 1e-4, name
        for b in range(cx.grid.n_band):
            fb = np.zeros((thu.shape[0], cx.grid.n_band), np.float32); fb[:, b] = 1.0
            _, tb = cx.sps.sps_photometry(cx.table, cx.ph, path, _dev(thu), True, _dev(fb))
            e = _grad_err(tb.cpu().numpy(), J[:, b, :] * dth, TAB_FLOOR[name])
            assert e.max() <= 1e-3, (name, b, e.max())
        lp, g = cx.sps.sps_loglike_grad(cx.table, cx.ph, path, _dev(thu), _dev(d), _dev(s), _dev(gal, torch.int32))
        olp, og, _ = M.logp_and_grad(thu.astype(np.float64), cx.grid, cx.P, d[gal].astype(np.float64), s[gal].astype(np.float64), name, cx.cssp())
        assert (np.abs(lp.cpu().numpy() - olp) / np.maximum(1.0, np.abs(olp))).max() <= 1e-4, name
        allow = FLUX_EPS[name] * np.einsum("rb,rbp->rp", of / s[gal].astype(np.float64) ** 2, np.abs(J)) * dth
        err = np.maximum(np.abs(g.cpu().numpy() - og) - allow, 0.0)
        assert (err / np.maximum(np.abs(og), TAB_FLOOR[name] * np.abs(og).max(1, keepdims=True))).max() <= 1e-3, name


# exact path + tabulated filters: d flux / d z sums the piecewise-constant slope of the curve over ~30 wavelengths; a sample
# within fp32 rounding of a knot may take either neighbouring segment's slope (R18), which moves that one component
TAB_FLOOR = {"approx": 1e-3, "exact": 1e-2}


# ---- SPS_OPT_CHECK_FINITE -------------------------------------------------------------------------------------------------
def test_check_finite_option(tiny):
    cx = tiny
    from paper_2506_19919_b200 import binding
    thu = W.draw_theta_unbounded(cx.prior, 8, 3).astype(np.float32)
    _, d, s = cx.observations(8, 5)
    bad = thu.copy(); bad[3, 7] = np.nan
    cx.sps.sps_set_option(cx.sps.OPT_CHECK_FINITE, 1)
    try:
        cx.sps.sps_loglike_grad(cx.table, cx.ph, cx.sps.PATH_APPROX, _dev(thu), _dev(d), _dev(s))      # clean inputs pass
        with pytest.raises(binding.SpsError) as e:
            cx.sps.sps_loglike_grad(cx.table, cx.ph, cx.sps.PATH_APPROX, _dev(bad), _dev(d), _dev(s))
        assert e.value.status == binding.STATUS_ENONFINITE
        s0 = s.copy(); s0[2, 1] = 0.0
        with pytest.raises(binding.SpsError) as e:
            cx.sps.sps_hmc_run(cx.table, cx.ph, _dev(d), _dev(s0), n_chain=2, n_warmup=2, n_sample=2, n_leapfrog=2, eps0=0.004)
        assert e.value.status == binding.STATUS_ENONFINITE
    finally:
        cx.sps.sps_set_option(cx.sps.OPT_CHECK_FINITE, 0)
    lp, _ = cx.sps.sps_loglike_grad(cx.table, cx.ph, cx.sps.PATH_APPROX, _dev(bad), _dev(d), _dev(s))  # off: no check, no sync, NaN flows through
    assert np.isnan(lp.cpu().numpy()[3]) and np.isfinite(lp.cpu().numpy()[[0, 1, 2, 4, 5, 6, 7]]).all()


# ---- one table, two streams (scratch is per stream) ---------------------------------------------------------------------
def test_two_streams_share_a_table(full):
    cx = full
    n = 20000
    tha = _dev(W.draw_theta_unbounded(cx.prior, n, 21).astype(np.float32)); thb = _dev(W.draw_theta_unbounded(cx.prior, n, 22).astype(np.float32))
    ra = cx.sps.sps_photometry(cx.table, cx.ph, cx.sps.PATH_APPROX, tha); rb = cx.sps.sps_photometry(cx.table, cx.ph, cx.sps.PATH_EXACT, thb)
    torch.cuda.synchronize()
    sa, sb = torch.cuda.Stream(), torch.cuda.Stream()
    outs = []
    for _ in range(3):
        with torch.cuda.stream(sa):
            xa = cx.sps.sps_photometry(cx.table, cx.ph, cx.sps.PATH_APPROX, tha)
        with torch.cuda.stream(sb):
            xb = cx.sps.sps_photometry(cx.table, cx.ph, cx.sps.PATH_EXACT, thb)
        outs.append((xa, xb))
    torch.cuda.synchronize()
    for xa, xb in outs:
        assert torch.equal(xa, ra) and torch.equal(xb, rb)


# ---- unconverged fits "require an additional ~N_steps": continue only those galaxies ---------------------------
def test_continue_only_unconverged_galaxies(tiny):
    cx = tiny
    n_gal, n_chain = 12, 3
    _, d, s = cx.observations(n_gal, 81)
    kw = dict(sampler=cx.sps.SAMPLER_HMC, path=cx.sps.PATH_APPROX, n_chain=n_chain, n_leapfrog=6, seed=13)
    first = cx.sps.sps_hmc_run(cx.table, cx.ph, _dev(d), _dev(s), n_warmup=60, n_sample=40, eps0=0.004, **kw)
    rhat = first["rhat"].max(1).values.cpu().numpy()
    todo = np.nonzero(rhat >= np.median(rhat))[0]                                  # "unconverged": the worse half
    assert 0 < todo.size < n_gal
    rows = (todo[:, None] * n_chain + np.arange(n_chain)[None, :]).reshape(-1)
    ri = _dev(rows, torch.int64)
    cont = dict(n_warmup=0, n_sample=30, first_transition=100, keep_samples=True)
    all_ = cx.sps.sps_hmc_run(cx.table, cx.ph, _dev(d), _dev(s), theta0=first["theta_last"], eps_in=first["eps"], inv_mass_in=first["inv_mass"], **cont, **kw)
    sub = cx.sps.sps_hmc_run(cx.table, cx.ph, _dev(d[todo]), _dev(s[todo]), theta0=first["theta_last"][ri].contiguous(), eps_in=first["eps"][ri].contiguous(),
                             inv_mass_in=first["inv_mass"][ri].contiguous(), gal_id=_dev(todo, torch.int32), **cont, **kw)
    # with their original RNG stream ids the continued galaxies get, bit for bit, what continuing everything gives them
    assert torch.equal(sub["samples"], all_["samples"][ri])
    assert torch.equal(sub["rhat"], all_["rhat"][_dev(todo, torch.int64)])
    # without the ids they would draw other galaxies' streams
    wrong = cx.sps.sps_hmc_run(cx.table, cx.ph, _dev(d[todo]), _dev(s[todo]), theta0=first["theta_last"][ri].contiguous(), eps_in=first["eps"][ri].contiguous(),
                               inv_mass_in=first["inv_mass"][ri].contiguous(), **cont, **kw)
    assert not torch.equal(wrong["samples"], sub["samples"])


# ---- NEXT-3 (Fig. 1 / B.3): posteriors from the exact and the approximate photometry model ----------
def test_posterior_overlay_exact_vs_approximate(tiny):
    # "compare the posteriors from HMC using both the exact and the approximate photometry models ... exact same initial
    # conditions".  Same data (from the exact model), same seed, same starts; pooled over 16 chains.
    cx = tiny
    n_gal, n_chain = 3, 16
    _, d, s = cx.observations(n_gal, 61, path="exact")
    th0 = _dev(S.init_chains(cx.P, 23, np.arange(n_gal * n_chain), 13).astype(np.float32))
    res = {}
    for name, path in (("exact", cx.sps.PATH_EXACT), ("approx", cx.sps.PATH_APPROX)):
        o = cx.sps.sps_hmc_run(cx.table, cx.ph, _dev(d), _dev(s), sampler=cx.sps.SAMPLER_NUTS, path=path, n_chain=n_chain, n_warmup=300, n_sample=500,
                               max_depth=6, eps0=0.004, seed=23, theta0=th0, keep_samples=True)
        x = o["samples"].cpu().numpy().reshape(n_gal, n_chain * 500, 13).astype(np.float64)
        res[name] = (x.mean(1), x.std(1), o["rhat"].cpu().numpy(), o["ess"].cpu().numpy())
        assert np.isfinite(x).all()
    (me, se, re_, ee), (ma, sa, ra, ea) = res["exact"], res["approx"]
    # the approximation moves band fluxes by ~1e-3..1e-2 of their 5 % errors' worth (Fig. B.2): the two posteriors overlay.
    # Compared where both runs have mixed (R-hat < 1.1), with the Monte-Carlo error of a mean of ESS draws as the yardstick.
    okm = (re_ < 1.1) & (ra < 1.1)
    assert okm.mean() > 0.5
    mc = np.sqrt(se ** 2 / np.maximum(ee, 1.0) + sa ** 2 / np.maximum(ea, 1.0))
    assert np.all(np.abs(me - ma)[okm] <= 0.15 * np.maximum(se, sa)[okm] + 4.0 * mc[okm])
    assert np.all(np.abs(np.log(se / sa))[okm] < 0.25)


# ---- NEXT-4: non-separable weights, an MDF whose median drifts with log age (R26) ------------------
@pytest.mark.parametrize("kind,n_gal", [("tiny", 30), ("full", 6)])
def test_nonseparable_weights(kind, n_gal, kernels):
    from oracle import nonsep as N
    gamma = -0.3
    cx = Ctx(kind, dlogZ_dlogage=gamma)
    n_chain = 3
    truth_u = W.draw_theta_unbounded(cx.prior, n_gal, 33).astype(np.float32).astype(np.float64)
    f = N.photometry_approx(M.bound(truth_u, cx.P)[0], cx.grid, gamma, cx.cssp())[0]
    d, s = W.noisy_observations(f, 34, 0.05, 0.10)
    d = d.astype(np.float32); s = s.astype(np.float32)
    thu = (np.repeat(truth_u, n_chain, 0) + 0.3 * np.random.default_rng(2).normal(size=(n_gal * n_chain, 13)) / cx.P[2]).astype(np.float32)
    gal = np.repeat(np.arange(n_gal), n_chain).astype(np.int32)
    th, dth = M.bound(thu.astype(np.float64), cx.P)
    for path, name in ((cx.sps.PATH_APPROX, "approx"), (cx.sps.PATH_EXACT, "exact")):
        of, J = (N.photometry_approx(th, cx.grid, gamma, cx.cssp()) if name == "approx" else N.photometry_exact(th, cx.grid, gamma))
        flux = cx.sps.sps_photometry(cx.table, cx.ph, path, _dev(thu)).cpu().numpy()
        assert _rel(flux, of).max() <= 1e-4, name
        # the model is really different from the separable one (so the test would see a kernel that ignored gamma)
        assert _rel(flux, (M.photometry_approx(th, cx.grid, cx.cssp()) if name == "approx" else M.photometry_exact(th, cx.grid, False))[0]).max() > 1e-2
        floor = 1e-2 if (name == "exact" and kernels == "tcgen05") else 1e-3            # the tcgen05 exact path's floor (test_gpu_parity.TC_FLOOR)
        for b in range(cx.grid.n_band):
            fb = np.zeros((thu.shape[0], cx.grid.n_band), np.float32); fb[:, b] = 1.0
            _, tb = cx.sps.sps_photometry(cx.table, cx.ph, path, _dev(thu), True, _dev(fb))
            assert _grad_err(tb.cpu().numpy(), J[:, b, :] * dth, floor).max() <= 1e-3, (name, b)
        lp, g = cx.sps.sps_loglike_grad(cx.table, cx.ph, path, _dev(thu), _dev(d), _dev(s), _dev(gal, torch.int32))
        olp, og, _ = N.logp_and_grad(thu.astype(np.float64), cx.grid, gamma, cx.P, d[gal].astype(np.float64), s[gal].astype(np.float64), name, cx.cssp())
        lp_allow = FLUX_EPS[name] * (np.abs(of - d[gal]) * of / s[gal].astype(np.float64) ** 2).sum(1)
        assert (np.maximum(np.abs(lp.cpu().numpy() - olp) - lp_allow, 0.0) / np.maximum(1.0, np.abs(olp))).max() <= 1e-4, name
        allow = FLUX_EPS[name] * np.einsum("rb,rbp->rp", of / s[gal].astype(np.float64) ** 2, np.abs(J)) * dth
        err = np.maximum(np.abs(g.cpu().numpy() - og) - allow, 0.0)
        assert (err / np.maximum(np.abs(og), floor * np.abs(og).max(1, keepdims=True))).max() <= 1e-3, name
    # and inside the sampler: a short NUTS run on the approximate path stays coupled to the oracle's
    if kind == "tiny":
        n_g, n_c, n_s, seed = 2, 2, 10, 29
        gl = np.repeat(np.arange(n_g), n_c)
        out = cx.sps.sps_hmc_run(cx.table, cx.ph, _dev(d[:n_g]), _dev(s[:n_g]), sampler=cx.sps.SAMPLER_HMC, path=cx.sps.PATH_APPROX, n_chain=n_c, n_warmup=0,
                                 n_sample=n_s, n_leapfrog=5, eps0=0.004, seed=seed, keep_samples=True)
        fh = lambda x: N.logp_and_grad(x, cx.grid, gamma, cx.P, d[gl].astype(np.float64), s[gl].astype(np.float64), "approx", cx.cssp())[:2]
        ref = S.run_chains(S.init_chains(cx.P, seed, np.arange(n_g * n_c), 13), fh, seed, 0, n_s, 0.004, "hmc", n_leapfrog=5)
        assert (np.abs(out["samples"].cpu().numpy() - ref["samples"]) / np.maximum(1.0, np.abs(ref["samples"]))).max() <= 1e-3


def test_row_groups_do_not_change_results(full):
    # SPS_OPT_ROW_GROUPS splits the chains of a fixed-length HMC run over several streams: same chains, bit for bit
    cx = full
    n_gal = 300
    _, d, s = cx.observations(n_gal, 97, frac=(0.05, 0.10))
    kw = dict(sampler=cx.sps.SAMPLER_HMC, path=cx.sps.PATH_APPROX, n_chain=4, n_warmup=6, n_sample=6, n_leapfrog=4, eps0=0.01, seed=3)
    ref = cx.sps.sps_hmc_run(cx.table, cx.ph, _dev(d), _dev(s), **kw)
    try:
        for G in (2, 3):
            cx.sps.sps_set_option(cx.sps.OPT_ROW_GROUPS, G)
            out = cx.sps.sps_hmc_run(cx.table, cx.ph, _dev(d), _dev(s), **kw)
            assert torch.equal(out["theta_last"], ref["theta_last"]) and torch.equal(out["mean"], ref["mean"]) and torch.equal(out["eps"], ref["eps"])
    finally:
        cx.sps.sps_set_option(cx.sps.OPT_ROW_GROUPS, 0)


def test_dependent_launch_and_cell_counts(full):
    # The prologue / contraction / epilogue kernels are launched programmatically dependent on one another, and the
    # tensor-core contraction clears the z-cell counts for the next prologue (no memset in between).  Neither may change a
    # result: the same HMC run with SPS_OPT_NO_PDL, and log-posterior calls that alternate between the tensor-core kernel
    # (clears the counts) and the SIMT kernel (needs them zeroed by the prologue's memset), bit for bit.
    cx = full
    n_gal = 300
    thu, d, s = cx.observations(n_gal, 98, frac=(0.05, 0.10))
    kw = dict(sampler=cx.sps.SAMPLER_HMC, path=cx.sps.PATH_APPROX, n_chain=4, n_warmup=6, n_sample=6, n_leapfrog=4, eps0=0.01, seed=3)
    ref = cx.sps.sps_hmc_run(cx.table, cx.ph, _dev(d), _dev(s), **kw)
    try:
        cx.sps.sps_set_option(cx.sps.OPT_NO_PDL, 1)
        out = cx.sps.sps_hmc_run(cx.table, cx.ph, _dev(d), _dev(s), **kw)
        assert torch.equal(out["theta_last"], ref["theta_last"]) and torch.equal(out["mean"], ref["mean"]) and torch.equal(out["eps"], ref["eps"])
    finally:
        cx.sps.sps_set_option(cx.sps.OPT_NO_PDL, 0)
    th = _dev(thu.astype(np.float32))
    runs = []
    try:
        for simt in (0, 0, 1, 0, 1, 1, 0):
            cx.sps.sps_set_option(cx.sps.OPT_APPROX_SIMT, simt)
            lp, g = cx.sps.sps_loglike_grad(cx.table, cx.ph, cx.sps.PATH_APPROX, th, _dev(d), _dev(s))
            runs.append((simt, lp.clone(), g.clone()))
    finally:
        cx.sps.sps_set_option(cx.sps.OPT_APPROX_SIMT, 0)
    for simt, lp, g in runs:
        first = next(r for r in runs if r[0] == simt)
        assert torch.equal(lp, first[1]) and torch.equal(g, first[2])


def test_sampler_runs_reuse_their_device_buffers(tiny):
    # per-run state comes from the library's block cache: after the first run of a shape, further runs neither allocate nor
    # free device memory (a cudaFree per run cost up to 0.7 s), for both samplers
    cx = tiny
    _, d, s = cx.observations(64, 5, frac=(0.05, 0.10))
    for sampler, extra in ((cx.sps.SAMPLER_HMC, dict(n_leapfrog=4)), (cx.sps.SAMPLER_NUTS, dict(max_depth=4))):
        kw = dict(sampler=sampler, path=cx.sps.PATH_APPROX, n_chain=4, n_warmup=5, n_sample=5, eps0=0.01, seed=3, **extra)
        ref = cx.sps.sps_hmc_run(cx.table, cx.ph, _dev(d), _dev(s), **kw)
        torch.cuda.synchronize()
        free0 = torch.cuda.mem_get_info()[0]
        for _ in range(3):
            out = cx.sps.sps_hmc_run(cx.table, cx.ph, _dev(d), _dev(s), **kw)
            assert torch.equal(out["theta_last"], ref["theta_last"])
        torch.cuda.synchronize()
        assert torch.cuda.mem_get_info()[0] == free0


# ---- degenerate launch shapes ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("n", [1, 129, 257])
def test_exact_path_ragged_sizes(full, n):
    # one row, one row past a 128-row tile, one past two: fluxes and the VJP against the oracle on sampled rows, and every
    # row bit-identical to the same row evaluated alone (the exact path's band sums are order-independent)
    cx = full
    thu = W.draw_theta_unbounded(cx.prior, n, 900 + n, z_uniform=(0.05, 2.95)).astype(np.float32)
    fb = np.random.default_rng(n).normal(size=(n, cx.grid.n_band)).astype(np.float32)
    flux, tb = cx.sps.sps_photometry(cx.table, cx.ph, cx.sps.PATH_EXACT, _dev(thu), True, _dev(fb))
    pick = np.unique(np.r_[0, n - 1, np.random.default_rng(3).integers(0, n, 4)])
    th, dth = M.bound(thu[pick].astype(np.float64), cx.P)
    of, J = M.photometry_exact(th, cx.grid, True)
    assert (np.abs(flux.cpu().numpy()[pick] - of) / np.abs(of)).max() <= 1e-4
    ref = np.einsum("rb,rbp->rp", fb[pick].astype(np.float64), J * dth[:, None, :])
    scale = np.einsum("rb,rbp->rp", np.abs(fb[pick]).astype(np.float64), np.abs(J * dth[:, None, :]))
    assert (np.abs(tb.cpu().numpy()[pick] - ref) / np.maximum(scale, TAB_FLOOR["exact"] * scale.max(1, keepdims=True))).max() <= 1e-3
    for r in pick[:3]:
        f1, t1 = cx.sps.sps_photometry(cx.table, cx.ph, cx.sps.PATH_EXACT, _dev(thu[r:r + 1]), True, _dev(fb[r:r + 1]))
        assert torch.equal(f1[0], flux[r]) and torch.equal(t1[0], tb[r])


def test_all_rows_in_one_z_cell_and_at_the_grid_ends(full, kernels):
    # the approximate path groups rows by z cell: 700 rows of ONE cell (six tiles of the same cell, the others empty), and
    # rows whose redshift saturates at the bounds of the prior (first / last cell of the table)
    cx = full
    n = 700
    thu = W.draw_theta_unbounded(cx.prior, n, 31).astype(np.float64)
    k, x0 = cx.P[2][12], cx.P[3][12]
    y_lo, y_hi = cx.P[0][12], cx.P[1][12]
    z_target = 1.2345
    thu[:, 12] = x0 + np.log((z_target - y_lo) / (y_hi - z_target)) / k          # Eq. (C1) inverted: every row at z = 1.2345
    thu[-8:-4, 12] = x0 - 60.0 / k                                               # z -> lower bound
    thu[-4:, 12] = x0 + 60.0 / k                                                 # z -> upper bound
    thu = thu.astype(np.float32)
    th, dth = M.bound(thu.astype(np.float64), cx.P)
    assert np.abs(th[:-8, 12] - z_target).max() < 1e-5
    of, J = M.photometry_approx(th, cx.grid, cx.cssp())
    fb = np.random.default_rng(8).normal(size=(n, cx.grid.n_band)).astype(np.float32)
    flux, tb = cx.sps.sps_photometry(cx.table, cx.ph, cx.sps.PATH_APPROX, _dev(thu), True, _dev(fb))
    assert (np.abs(flux.cpu().numpy() - of) / np.abs(of)).max() <= 1e-4
    ref = np.einsum("rb,rbp->rp", fb.astype(np.float64), J * dth[:, None, :])
    scale = np.einsum("rb,rbp->rp", np.abs(fb).astype(np.float64), np.abs(J * dth[:, None, :]))
    err = np.abs(tb.cpu().numpy() - ref) / np.maximum(scale, 1e-3 * scale.max(1, keepdims=True))
    err[-8:, 12] = 0.0             # saturated sigmoid: d z / d theta~ ~ 1e-26, nothing to compare
    assert err.max() <= 1e-3
