"""sps_loglike_grad_noalloc (the entry point that allocates nothing: its scratch is a fixed device array inside the library)
against the existing sps_loglike_grad on the approximate path, on two calls in a row, plus its size limit.  Collected last
on purpose (the file name): the array is shared by all calls, so this runs after everything else has used the device, and
it must also pass alone in a fresh process."""
import numpy as np
import pytest

from paper_2506_19919_b200 import workloads as W

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


def _dev(a, dtype=None):
    return torch.tensor(np.asarray(a), dtype=dtype or torch.float32, device="cuda")


def _grad_err(g, ref, floor=1e-3):
    return np.abs(g - ref) / np.maximum(np.abs(ref), floor * np.abs(ref).max(1, keepdims=True))


def _case(sps, grid_name, n_gal, n_chain, seed):
    """A table, a prior and a batch of chains scattered around prior-drawn truths (several 128-row tiles, a ragged tail,
    many z cells), with observations from the library's own photometry of the truths."""
    grid = W.make_grid(grid_name); prior = W.make_prior(); ph = sps.PriorHandle(prior.as_array())
    table = sps.sps_create_table(grid)
    truth_u = W.draw_theta_unbounded(prior, n_gal, seed).astype(np.float32)
    f = sps.sps_photometry(table, ph, sps.PATH_APPROX, _dev(truth_u)).cpu().numpy().astype(np.float64)
    d, s = W.noisy_observations(f, seed + 1, 0.05, 0.10)
    rng = np.random.default_rng(seed + 2)
    thu = (np.repeat(truth_u, n_chain, 0) + 0.3 * rng.standard_normal((n_gal * n_chain, 13)) / prior.as_array()[2]).astype(np.float32)
    gal = np.repeat(np.arange(n_gal), n_chain).astype(np.int32)
    return table, ph, _dev(thu), _dev(d.astype(np.float32)), _dev(s.astype(np.float32)), _dev(gal, torch.int32)


@pytest.mark.parametrize("grid_name", ["tiny", "full"])
def test_no_alloc_entry_point_matches_the_allocating_one(grid_name):
    import paper_2506_19919_b200 as sps
    table, ph, thu, d, s, gal = _case(sps, grid_name, 333, 3, 41)          # 999 rows
    n = thu.shape[0]
    ref_lp, ref_g = sps.sps_loglike_grad(table, ph, sps.PATH_APPROX, thu, d, s, gal)
    ref_lp = ref_lp.cpu().numpy().astype(np.float64); ref_g = ref_g.cpu().numpy().astype(np.float64)
    assert np.isfinite(ref_lp).all() and np.isfinite(ref_g).all()
    # two calls in a row, the second on fewer rows in another order (the array keeps the first call's contents)
    lp = torch.full((n,), float("nan"), device="cuda"); g = torch.full((n, 13), float("nan"), device="cuda")
    sps.sps_loglike_grad_noalloc(table, ph, thu, d, s, lp, g, gal)
    torch.cuda.synchronize()
    lp1 = lp.cpu().numpy().astype(np.float64); g1 = g.cpu().numpy().astype(np.float64)
    perm = torch.tensor(np.random.default_rng(5).permutation(n)[:601].copy(), device="cuda")
    thu2 = thu[perm].contiguous(); gal2 = gal[perm].contiguous()
    lp2 = torch.full((601,), float("nan"), device="cuda"); g2 = torch.full((601, 13), float("nan"), device="cuda")
    free_before = torch.cuda.mem_get_info()[0]
    sps.sps_loglike_grad_noalloc(table, ph, thu2, d, s, lp2, g2, gal2)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free_before                      # nothing was allocated on the device
    idx = perm.cpu().numpy()
    for got_lp, got_g, want_lp, want_g in ((lp1, g1, ref_lp, ref_g),
                                           (lp2.cpu().numpy().astype(np.float64), g2.cpu().numpy().astype(np.float64), ref_lp[idx], ref_g[idx])):
        # the parity suite's tolerances (tests/test_gpu_parity.py): logP 1e-4 max(1, |logP|), gradients 1e-3 with floor 1e-3
        assert (np.abs(got_lp - want_lp) / np.maximum(1.0, np.abs(want_lp))).max() <= 1e-4
        assert _grad_err(got_g, want_g).max() <= 1e-3
    # log-posterior only (grad = NULL)
    lp3 = torch.full((n,), float("nan"), device="cuda")
    sps.sps_loglike_grad_noalloc(table, ph, thu, d, s, lp3, None, gal)
    assert (np.abs(lp3.cpu().numpy() - ref_lp) / np.maximum(1.0, np.abs(ref_lp))).max() <= 1e-4


def test_no_alloc_entry_point_rejects_sizes_beyond_its_array():
    import paper_2506_19919_b200 as sps
    table, ph, thu, d, s, gal = _case(sps, "tiny", 8, 1, 43)
    n = sps.binding.NOALLOC_MAX_ROWS + 1
    big = thu[:1].repeat(n, 1).contiguous(); big_gal = torch.zeros(n, dtype=torch.int32, device="cuda")
    lp = torch.zeros(n, device="cuda"); g = torch.zeros(n, 13, device="cuda")
    with pytest.raises(sps.SpsError) as e:
        sps.sps_loglike_grad_noalloc(table, ph, big, d, s, lp, g, big_gal)
    assert e.value.status == 2 and "SPS_NOALLOC_MAX_ROWS" in str(e.value)          # SPS_ESHAPE
    # the limit itself is accepted
    lp, g = sps.sps_loglike_grad_noalloc(table, ph, big[:-1].contiguous(), d, s, lp[:-1], g[:-1].contiguous(), big_gal[:-1].contiguous())
    ref_lp, ref_g = sps.sps_loglike_grad(table, ph, sps.PATH_APPROX, big[:-1].contiguous(), d, s, big_gal[:-1].contiguous())
    assert (torch.abs(lp - ref_lp) / torch.clamp(torch.abs(ref_lp), min=1.0)).max().item() <= 1e-4
    assert _grad_err(g.cpu().numpy().astype(np.float64), ref_g.cpu().numpy().astype(np.float64)).max() <= 1e-3
