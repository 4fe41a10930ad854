"""Pins of the non-separable weight model (`oracle/nonsep.py`; R26).  CPU only."""
import numpy as np
import pytest

from oracle import nonsep as N
from oracle import sps_model as M
from paper_2506_19919_b200 import workloads as W


@pytest.fixture(scope="module")
def setup():
    g = W.make_grid("tiny"); P = W.make_prior()
    return g, P, P.as_array(), M.cssp_table(g)


def test_gamma_zero_is_the_separable_model(setup):
    g, P, prior, cssp = setup
    th = M.bound(W.draw_theta_unbounded(P, 4, 1), prior)[0]
    for fn_n, fn_s in ((lambda: N.photometry_exact(th, g, 0.0), lambda: M.photometry_exact(th, g)),
                       (lambda: N.photometry_approx(th, g, 0.0, cssp), lambda: M.photometry_approx(th, g, cssp))):
        (f1, J1), (f0, J0) = fn_n(), fn_s()
        assert np.allclose(f1, f0, rtol=1e-13) and np.allclose(J1, J0, rtol=1e-10, atol=1e-14 * np.abs(J0).max())


def test_rows_sum_to_one_and_the_median_drifts(setup):
    g, P, prior, _ = setup
    th = M.bound(W.draw_theta_unbounded(P, 3, 2), prior)[0]
    w, _, m = N.ssp_weights(th, g, -0.3)
    assert np.allclose(m.sum(2), 1.0, atol=1e-13)                       # every age bin's MDF is normalised
    Wd = M.weights(th, g)
    assert np.allclose(w.sum(2), Wd["Mn"][:, None] * Wd["a"], rtol=1e-12)   # summing over Z gives back M* a_i
    mean_Z = (m * g.log10_Z[None, None, :]).sum(2)
    assert np.all(np.diff(mean_Z, axis=1) <= 1e-12)                     # gamma < 0: older stars are metal-poorer
    # the bin whose age is 1e9 yr would have exactly the separable MDF: check through a grid that contains it
    la = np.array([8.0, 9.0, 10.0])
    mm = N.met_weights_by_age(th[:, 7], th[:, 8], g.log10_Z, la, -0.3)[0]
    assert np.allclose(mm[:, 1], M.met_weights(th[:, 7], th[:, 8], g.log10_Z)[0], atol=1e-15)
    assert np.allclose(mm[:, 0], M.met_weights(th[:, 7] + 0.3, th[:, 8], g.log10_Z)[0], atol=1e-15)


@pytest.mark.parametrize("path", ["exact", "approx"])
def test_gradient_matches_central_differences(setup, path):
    g, P, prior, cssp = setup
    thu = W.draw_theta_unbounded(P, 2, 3)
    d, s = W.noisy_observations(N.photometry_approx(M.bound(thu, prior)[0], g, -0.25, cssp)[0], 4, 0.05, 0.05)
    lp, gr, _ = N.logp_and_grad(thu, g, -0.25, prior, d, s, path, cssp)
    for p in range(13):
        e = np.zeros(13); e[p] = 1e-6
        fd = (N.logp_and_grad(thu + e, g, -0.25, prior, d, s, path, cssp)[0] - N.logp_and_grad(thu - e, g, -0.25, prior, d, s, path, cssp)[0]) / 2e-6
        assert np.allclose(gr[:, p], fd, rtol=5e-5, atol=1e-6 * np.abs(gr).max()), (p, gr[:, p], fd)
