"""Seeded synthetic inputs shaped like the paper's workloads (numpy only).

This module holds NO arithmetic of the method (no SFH, dust, photometry, likelihood or
sampler maths): it only manufactures arrays -- grids, stand-in SSP spectra, Gaussian filter
parameters, prior hyper-parameters and parameter draws -- that are handed, unchanged, both to
the CUDA library and to the float64 oracle by the tests.  Neither `oracle/` nor the CUDA path
imports the other; both receive these arrays.

What stands in for what:
  * SSP spectra: the paper uses MIST templates; they are not available here, so
    smooth positive spectra (5 log-normal bumps per SSP, ~3 dex young->old) stand in.
  * Filters: Gaussian transmission curves with lambda/FWHM from 3.4 to 25.5 -- the paper's own
    kind of filter (Fig. B.1).
  * Galaxies: parameters drawn from the prior on the unbounded parameters.
  * Bounds / prior numbers: not given anywhere in the paper; the table
    PRIOR_TABLE below is this repository's choice.
"""
from __future__ import annotations

import dataclasses
import math

import numpy as np

SEED0 = 20250619

# parameter order of the 13-parameter model (PAPER.md:349, 372, 378, 390 + redshift)
PARAM_NAMES = ("logM", "tau", "alpha", "beta", "F_burst", "logT_peak", "logT_max",
               "logZ", "sigma_logZ", "A_V", "delta", "F_floor", "z")
NDIM = len(PARAM_NAMES)

# name: (y_lo, y_hi, gaussian mean, gaussian sd) in the bounded (physical) space
PRIOR_TABLE = {
    "logM": (8.0, 12.0, 10.0, 0.8),
    "tau": (0.3, 14.0, 4.0, 2.0),
    "alpha": (0.5, 8.0, 3.0, 1.5),
    "beta": (0.2, 5.0, 1.5, 1.0),
    "F_burst": (0.0, 0.5, 0.05, 0.05),
    "logT_peak": (5.5, 7.5, 6.5, 0.4),
    "logT_max": (7.6, 9.0, 8.3, 0.3),
    "logZ": (-2.2, 0.4, -0.3, 0.4),
    "sigma_logZ": (0.05, 0.6, 0.2, 0.1),
    "A_V": (0.0, 3.0, 0.5, 0.4),
    "delta": (-1.2, 0.4, -0.3, 0.3),
    "F_floor": (0.0, 0.5, 0.1, 0.1),
    "z": (0.02, 2.98, 1.0, 0.6),
}

# SPS_MODEL_TINY5 (BASELINE.json configs[0]; R19): logM_star, log10 tau/Gyr, logZ, tau_V sampled; z = 0.5 is data
TINY5_PARAM_NAMES = ("logM", "log_tau", "logZ", "tau_V")
TINY5_PRIOR_TABLE = {
    "logM": (8.0, 12.0, 10.0, 0.8),
    "log_tau": (-0.5, 1.2, 0.5, 0.3),
    "logZ": (-2.2, 0.4, -0.3, 0.4),
    "tau_V": (0.0, 3.0, 0.5, 0.4),
}
TINY5_Z = 0.5


@dataclasses.dataclass
class Grid:
    """Everything `sps_create_table` needs, as host arrays."""
    log10_age_yr: np.ndarray   # [n_age] float64, increasing
    log10_Z: np.ndarray        # [n_Z]   float64, increasing (log10 Z/Zsun)
    wave_A: np.ndarray         # [n_wave] float64, strictly increasing, rest-frame Angstrom
    ssp: np.ndarray            # [n_age*n_Z, n_wave] float32, row = i*n_Z + j
    filt_mu_A: np.ndarray      # [n_band] float64 observed-frame centre
    filt_sigma_A: np.ndarray   # [n_band] float64 Gaussian sigma
    z_min: float
    z_max: float
    n_z: int
    H0: float = 67.74
    Om: float = 0.3089
    log10_mass_unit: float = 10.0
    # tabulated filters (observed frame) instead of Gaussian ones: (wave_A [n_knot], trans [n_knot], offsets [n_band+1]);
    # band b owns the knots offsets[b] .. offsets[b+1]-1 (strictly increasing wavelengths within a band)
    filt_tab: tuple | None = None

    @property
    def n_age(self): return int(self.log10_age_yr.size)
    @property
    def n_Z(self): return int(self.log10_Z.size)
    @property
    def n_wave(self): return int(self.wave_A.size)
    @property
    def n_band(self): return int(self.filt_mu_A.size) if self.filt_tab is None else int(len(self.filt_tab[2]) - 1)


@dataclasses.dataclass
class Prior:
    """Per-parameter hyper-parameters: C1 bounds and C2 skew-normal (438-444)."""
    y_lo: np.ndarray
    y_hi: np.ndarray
    k: np.ndarray
    x0: np.ndarray
    xi: np.ndarray
    omega: np.ndarray
    skew: np.ndarray

    def as_array(self) -> np.ndarray:
        """[7, D] float64, rows in the order of the fields above."""
        return np.stack([self.y_lo, self.y_hi, self.k, self.x0, self.xi, self.omega, self.skew])


def _rng(seed):
    return np.random.Generator(np.random.PCG64(seed))


def make_ssp_spectra(log10_age_yr, log10_Z, wave_A, seed):
    """Smooth, positive stand-in spectra: a young->old fading power law times 5 log-normal bumps
    whose centres drift redward with age and mildly with metallicity."""
    rng = _rng(seed)
    n_b = 5
    centre = rng.uniform(math.log(1500.0), math.log(20000.0), n_b)
    s_age = rng.uniform(0.05, 0.25, n_b)
    s_met = rng.uniform(-0.1, 0.1, n_b)
    width = rng.uniform(0.15, 0.6, n_b)
    amp0 = rng.uniform(0.1, 1.0, n_b)
    phase = rng.uniform(0.0, 2 * math.pi, n_b)
    qz = rng.uniform(-0.2, 0.2, n_b)
    la = np.asarray(log10_age_yr, float)[:, None, None, None]      # [i,1,1,1]
    lz = np.asarray(log10_Z, float)[None, :, None, None]           # [1,j,1,1]
    lnw = np.log(np.asarray(wave_A, float))[None, None, None, :]   # [1,1,1,k]
    mu = centre[None, None, :, None] + s_age[None, None, :, None] * (la - 8.0) + s_met[None, None, :, None] * lz
    amp = amp0[None, None, :, None] * (1.0 + 0.2 * np.cos(phase[None, None, :, None] + 0.5 * (la - 8.0))) \
        * (1.0 + qz[None, None, :, None] * lz / 2.5)
    bumps = amp * np.exp(-0.5 * ((lnw - mu) / width[None, None, :, None]) ** 2)
    spec = bumps.sum(axis=2) * 10.0 ** (-0.7 * (la[:, :, 0, :] - 6.0))  # [i,j,k]
    spec = spec / 1000.0                                                # per-Angstrom scale: band fluxes O(1e-3..1)
    n_age, n_Z, n_wave = spec.shape
    return np.ascontiguousarray(spec.reshape(n_age * n_Z, n_wave).astype(np.float32))


def gaussian_filters(centres_A, lam_over_fwhm):
    centres_A = np.asarray(centres_A, float)
    fwhm = centres_A / np.asarray(lam_over_fwhm, float)
    return centres_A, fwhm / (2.0 * math.sqrt(2.0 * math.log(2.0)))


def make_grid(kind: str, seed: int | None = None) -> Grid:
    """kind = 'tiny' (BASELINE.json configs[0]: 20 x 4 x 500, 3 filters), 'odd' (33 x 5 x 777, 12 filters: test shapes) or
    'full' (configs[1..4]: 107 x 12 x 5994, 10 filters, 200-point z grid)."""
    if kind == "tiny":
        seed = SEED0 if seed is None else seed
        la = np.linspace(6.0, math.log10(1.3e10), 20)
        lz = np.linspace(-2.0, 0.3, 4)
        wave = np.geomspace(1.0e3, 1.0e5, 500)
        mu, sg = gaussian_filters([4500.0, 6500.0, 9000.0], [6.0, 6.0, 6.0])
        n_z = 16
    elif kind == "full":
        seed = SEED0 + 1 if seed is None else seed
        la = 5.0 + 0.05 * np.arange(107)
        lz = np.linspace(-2.5, 0.5, 12)
        wave = np.geomspace(250.0, 5.0e4, 5994)
        mu, sg = gaussian_filters(np.geomspace(3300.0, 11000.0, 10), np.geomspace(3.4, 25.5, 10))
        n_z = 200
    elif kind == "odd":
        # awkward sizes for the parity tests (not a BASELINE config): nothing is a multiple of a tile, 12 bands
        seed = SEED0 + 2 if seed is None else seed
        la = np.linspace(5.5, 10.2, 33)
        lz = np.linspace(-2.2, 0.4, 5)
        wave = np.geomspace(400.0, 4.0e4, 777)
        mu, sg = gaussian_filters(np.geomspace(3500.0, 10500.0, 12), np.geomspace(4.0, 12.0, 12))
        n_z = 9
    elif kind == "tiny_tab":
        # the tiny grid with TABULATED filters: three asymmetric curves on their own non-uniform wavelength grids
        g = make_grid("tiny", seed)
        return dataclasses.replace(g, filt_tab=tabulated_filters([4500.0, 6500.0, 9000.0], [900.0, 1300.0, 1700.0], SEED0 + 3))
    else:
        raise ValueError(kind)
    ssp = make_ssp_spectra(la, lz, wave, seed)
    return Grid(la, lz, wave, ssp, mu, sg, 0.0, 3.0, n_z)


def tabulated_filters(centres_A, widths_A, seed, n_knot=(41, 57, 73)):
    """Stand-ins for measured transmission curves: per band a smooth asymmetric bump (steep blue edge, slow red decline,
    a ripple on top) sampled on a jittered, non-uniform grid of its own; zero at both ends.  Input data only."""
    rng = _rng(seed)
    waves, trans, off = [], [], [0]
    for c, w, n in zip(centres_A, widths_A, n_knot):
        u = np.sort(np.concatenate([[0.0, 1.0], rng.uniform(0.0, 1.0, n - 2)]))
        lam = c - 0.5 * w + w * u
        t = (1.0 - np.exp(-u / 0.08)) * np.clip(1.0 - u, 0.0, 1.0) ** 0.6 * (1.0 + 0.1 * np.sin(17.0 * u))
        t[0] = 0.0; t[-1] = 0.0
        waves.append(lam); trans.append(t / t.max()); off.append(off[-1] + n)
    return np.concatenate(waves), np.concatenate(trans), np.array(off, np.int32)


def _logit_inverse(theta, y_lo, y_hi, k, x0):
    """Inverse of the bounding sigmoid; used only to place draws / fit prior hyper-parameters."""
    u = (theta - y_lo) / (y_hi - y_lo)
    return x0 + np.log(u / (1.0 - u)) / k


def make_prior(seed: int = SEED0 + 100, n_fit: int = 20000, model: str = "dpl13") -> Prior:
    """Bounds from PRIOR_TABLE (model = "dpl13") or TINY5_PRIOR_TABLE ("tiny5"), k = 4/(y_hi-y_lo), x0 = centre (unit
    slope at the centre); skew-normal (xi, omega, s) moment-fitted to Gaussian draws mapped to the
    unbounded space (the fit itself is host-side setup, out of scope)."""
    rng = _rng(seed)
    cols = [PRIOR_TABLE[n] for n in PARAM_NAMES] if model == "dpl13" else [TINY5_PRIOR_TABLE[n] for n in TINY5_PARAM_NAMES]
    NDIM = len(cols)
    y_lo = np.array([c[0] for c in cols]); y_hi = np.array([c[1] for c in cols])
    mean = np.array([c[2] for c in cols]); sd = np.array([c[3] for c in cols])
    k = 4.0 / (y_hi - y_lo); x0 = 0.5 * (y_lo + y_hi)
    xi = np.zeros(NDIM); om = np.zeros(NDIM); sk = np.zeros(NDIM)
    for p in range(NDIM):
        d = np.empty(0)
        while d.size < n_fit:
            c = rng.normal(mean[p], sd[p], 2 * n_fit)
            w = 1e-3 * (y_hi[p] - y_lo[p])
            d = np.concatenate([d, c[(c > y_lo[p] + w) & (c < y_hi[p] - w)]])
        u = _logit_inverse(d[:n_fit], y_lo[p], y_hi[p], k[p], x0[p])
        m1, m2 = u.mean(), u.var()
        g1 = float(np.clip(((u - m1) ** 3).mean() / m2 ** 1.5, -0.9, 0.9))
        # method of moments for the skew-normal
        a = abs(g1) ** (2.0 / 3.0)
        dlt = math.copysign(math.sqrt(0.5 * math.pi * a / (a + (0.5 * (4.0 - math.pi)) ** (2.0 / 3.0))), g1)
        dlt = max(-0.95, min(0.95, dlt))
        om[p] = math.sqrt(m2 / (1.0 - 2.0 * dlt * dlt / math.pi))
        xi[p] = m1 - om[p] * dlt * math.sqrt(2.0 / math.pi)
        sk[p] = dlt / math.sqrt(1.0 - dlt * dlt)
    return Prior(y_lo, y_hi, k, x0, xi, om, sk)


def draw_theta_unbounded(prior: Prior, n: int, seed: int, z_uniform: tuple[float, float] | None = None):
    """n draws of the unbounded parameters from the skew-normal prior [n, D] float64.
    z_uniform=(a,b) replaces the redshift column by U[a,b] in bounded space (configs[1], [2])."""
    rng = _rng(seed)
    NDIM = prior.xi.size
    u0 = rng.standard_normal((n, NDIM)); u1 = rng.standard_normal((n, NDIM))
    dlt = prior.skew / np.sqrt(1.0 + prior.skew ** 2)
    x = dlt * np.abs(u0) + np.sqrt(1.0 - dlt ** 2) * u1
    th = prior.xi + prior.omega * x
    # keep draws away from the saturated ends of the sigmoid
    lim = 5.0 / prior.k
    th = np.clip(th, prior.x0 - lim, prior.x0 + lim)
    if z_uniform is not None:
        zz = rng.uniform(z_uniform[0], z_uniform[1], n)
        w = 1e-3 * (prior.y_hi[-1] - prior.y_lo[-1])             # U[0.1,3] reaches past the bound y_hi = 2.98: keep draws inside
        zz = np.clip(zz, prior.y_lo[-1] + w, prior.y_hi[-1] - w)
        th[:, NDIM - 1] = _logit_inverse(zz, prior.y_lo[-1], prior.y_hi[-1], prior.k[-1], prior.x0[-1])
    return th


def pad_prior(prior: Prior, fixed: dict[int, float] | None = None, ndim: int = NDIM) -> np.ndarray:
    """[7, ndim] array for the C ABI from a prior over fewer sampled parameters (SPS_MODEL_TINY5: 4): unused slots get
    the identity bounds (0, 1), k = 1, x0 = 0, omega = 1, skew = 0; `fixed` puts data values (the redshift) into xi."""
    a = prior.as_array()
    out = np.zeros((7, ndim)); out[1] = 1.0; out[2] = 1.0; out[5] = 1.0
    out[:, :a.shape[1]] = a
    for slot, v in (fixed or {}).items():
        out[4, slot] = v
    return out


def noisy_observations(flux_true: np.ndarray, seed: int, frac_lo: float, frac_hi: float):
    """d = f(1 + e*n), sigma = e*f with e ~ U[frac_lo, frac_hi] per band (BASELINE.json configs[0], [3])."""
    rng = _rng(seed)
    e = rng.uniform(frac_lo, frac_hi, flux_true.shape)
    n = rng.standard_normal(flux_true.shape)
    return flux_true * (1.0 + e * n), e * np.abs(flux_true)


CONFIGS = {
    # name: description of the BASELINE.json config it stands for
    "c1_tiny_hmc": dict(grid="tiny", n_gal=8, n_chain=4, n_warmup=0, n_sample=200, n_leapfrog=10, seed=SEED0 + 0),
    "c2_exact": dict(grid="full", batch=8192, seed=SEED0 + 1),
    "c3_approx": dict(grid="full", batch=1 << 20, seed=SEED0 + 2),
    "c4_hmc": dict(grid="full", n_gal=10000, n_chain=4, n_warmup=500, n_sample=500, n_leapfrog=16, seed=SEED0 + 3),
    "c5_nuts": dict(grid="full", n_gal=100000, n_chain=4, n_warmup=500, n_sample=500, max_depth=8,
                    exact_fraction=0.1, seed=SEED0 + 4),
}
