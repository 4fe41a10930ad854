"""Thin ctypes binding of libsps_b200.so (include/sps.h).  Argument marshalling only: every step of
the hot path runs in the CUDA kernels behind the C ABI.  torch is used for device memory and streams.

There is no CPU fallback: if the shared library is missing or cannot be loaded, every call raises.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libsps_b200.so")
NDIM = 13
PATH_EXACT, PATH_APPROX = 0, 1
SAMPLER_HMC, SAMPLER_NUTS = 0, 1
EXACT_BF16X3, EXACT_TF32X3 = 0, 1
MODEL_TINY5, MODEL_DPL13, MODEL_GAUSS_TEST = 0, 1, 2
OPT_CHECK_FINITE, OPT_EXACT_SIMT, OPT_APPROX_SIMT, OPT_NO_TC_SETUP, OPT_NO_GRAPH, OPT_ROW_GROUPS, OPT_NO_PDL = 0, 1, 2, 3, 4, 5, 6
STATUS_ENONFINITE = 6

EXPORTS = ("sps_create_table", "sps_destroy_table", "sps_table_cssp", "sps_weights", "sps_photometry",
           "sps_loglike_grad", "sps_leapfrog", "sps_hmc_run", "sps_philox_words", "sps_profile", "sps_profile_read", "sps_launch_count",
           "sps_last_error", "sps_version", "sps_exact_last_work", "sps_exact_work_since", "sps_loglike_grad_noalloc", "sps_model_ndim", "sps_set_option", "sps_measure_peak")


class SpsError(RuntimeError):
    pass


class _TableDesc(C.Structure):
    _fields_ = [("n_age", C.c_int32), ("n_Z", C.c_int32), ("n_wave", C.c_int32), ("n_band", C.c_int32), ("n_z", C.c_int32),
                ("log10_age_yr", C.POINTER(C.c_double)), ("log10_Z", C.POINTER(C.c_double)), ("wave_A", C.POINTER(C.c_double)),
                ("ssp", C.POINTER(C.c_float)), ("filt_mu_A", C.POINTER(C.c_double)), ("filt_sigma_A", C.POINTER(C.c_double)),
                ("z_min", C.c_double), ("z_max", C.c_double), ("H0", C.c_double), ("Om", C.c_double),
                ("log10_mass_unit", C.c_double), ("exact_precision", C.c_int32), ("model", C.c_int32),
                ("filt_wave_A", C.POINTER(C.c_double)), ("filt_trans", C.POINTER(C.c_double)), ("filt_offsets", C.POINTER(C.c_int32)),
                ("dlogZ_dlogage", C.c_double), ("gauss_ndim", C.c_int32), ("gauss_mu", C.POINTER(C.c_double)),
                ("gauss_prec", C.POINTER(C.c_double))]


class _Prior(C.Structure):
    _fields_ = [(n, C.POINTER(C.c_double)) for n in ("y_lo", "y_hi", "k", "x0", "xi", "omega", "skew")]


class _HmcConfig(C.Structure):
    _fields_ = [("sampler", C.c_int32), ("path", C.c_int32), ("n_chain", C.c_int32), ("n_warmup", C.c_int32),
                ("n_sample", C.c_int32), ("n_leapfrog", C.c_int32), ("max_depth", C.c_int32), ("eps0", C.c_float),
                ("target_accept", C.c_float), ("seed", C.c_uint64),
                ("first_transition", C.c_uint32), ("eps_in", C.c_void_p), ("inv_mass_in", C.c_void_p), ("gal_id", C.c_void_p)]


class _HmcSummary(C.Structure):
    _fields_ = [(n, C.c_void_p) for n in ("mean", "sd", "accept", "eps", "inv_mass", "n_leapfrog", "divergences", "rhat", "theta_last",
                                          "ess", "depth_hist")]


_lib = None


def lib():
    """Load the shared library (once).  Raises loudly when it is missing: no fallback exists."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise SpsError(f"{LIB_PATH} is missing: build it with `python -m paper_2506_19919_b200.build` "
                           "(there is no CPU fallback)")
        L = C.CDLL(LIB_PATH)
        L.sps_last_error.restype = C.c_char_p
        L.sps_version.restype = C.c_char_p
        L.sps_launch_count.restype = C.c_int64
        L.sps_model_ndim.restype = C.c_int32
        _lib = L
    return _lib


def _check(status: int, what: str):
    if status != 0:
        e = SpsError(f"{what} failed with status {status}: {lib().sps_last_error().decode()}")
        e.status = status
        raise e


def _dptr(t):
    if t is None:
        return C.c_void_p(0)
    import torch
    assert isinstance(t, torch.Tensor) and t.is_cuda and t.is_contiguous(), "need a contiguous CUDA tensor"
    return C.c_void_p(t.data_ptr())


def _stream():
    import torch
    return C.c_void_p(torch.cuda.current_stream().cuda_stream)


def _f64(a):
    return np.ascontiguousarray(np.asarray(a, dtype=np.float64))


class PriorHandle:
    """Holds the host arrays of an sps_prior alive."""

    def __init__(self, prior_array):
        a = _f64(prior_array)
        assert a.shape == (7, NDIM)
        self._rows = [np.ascontiguousarray(a[i]) for i in range(7)]
        self.c = _Prior(*[r.ctypes.data_as(C.POINTER(C.c_double)) for r in self._rows])

    def ref(self):
        return C.byref(self.c)


class Table:
    """Owner of an sps_table handle.  model = MODEL_DPL13 (the paper's 13-parameter model), MODEL_TINY5 (BASELINE.json
    configs[0]) or MODEL_GAUSS_TEST (grid = None, gauss = (mu [D], precision [D, D]))."""

    def __init__(self, grid, exact_precision=0, model=MODEL_DPL13, gauss=None, dlogZ_dlogage=0.0):
        dp = lambda a: a.ctypes.data_as(C.POINTER(C.c_double))
        d = _TableDesc()
        d.model = int(model); d.exact_precision = int(exact_precision); d.dlogZ_dlogage = float(dlogZ_dlogage)
        keep = []
        if model == MODEL_GAUSS_TEST:
            mu, prec = _f64(gauss[0]), _f64(gauss[1])
            assert prec.shape == (mu.size, mu.size)
            keep += [mu, prec]
            d.gauss_ndim = mu.size; d.gauss_mu = dp(mu); d.gauss_prec = dp(prec)
            self.n_age = self.n_Z = self.n_wave = self.n_band = self.n_z = 0
        else:
            self.n_age, self.n_Z, self.n_wave, self.n_band, self.n_z = grid.n_age, grid.n_Z, grid.n_wave, grid.n_band, grid.n_z
            keep += [_f64(grid.log10_age_yr), _f64(grid.log10_Z), _f64(grid.wave_A), np.ascontiguousarray(grid.ssp, dtype=np.float32)]
            assert keep[3].shape == (self.n_age * self.n_Z, self.n_wave)
            d.n_age, d.n_Z, d.n_wave, d.n_band, d.n_z = self.n_age, self.n_Z, self.n_wave, self.n_band, self.n_z
            d.log10_age_yr, d.log10_Z, d.wave_A = dp(keep[0]), dp(keep[1]), dp(keep[2])
            d.ssp = keep[3].ctypes.data_as(C.POINTER(C.c_float))
            tab = getattr(grid, "filt_tab", None)
            if tab is None:
                mu, sg = _f64(grid.filt_mu_A), _f64(grid.filt_sigma_A)
                keep += [mu, sg]
                d.filt_mu_A, d.filt_sigma_A = dp(mu), dp(sg)
            else:
                fw, ft, fo = _f64(tab[0]), _f64(tab[1]), np.ascontiguousarray(tab[2], dtype=np.int32)
                keep += [fw, ft, fo]
                d.filt_wave_A, d.filt_trans, d.filt_offsets = dp(fw), dp(ft), fo.ctypes.data_as(C.POINTER(C.c_int32))
            d.z_min, d.z_max, d.H0, d.Om = float(grid.z_min), float(grid.z_max), float(grid.H0), float(grid.Om)
            d.log10_mass_unit = float(grid.log10_mass_unit)
        h = C.c_void_p()
        _check(lib().sps_create_table(C.byref(d), C.byref(h)), "sps_create_table")
        self.handle = h
        self.n_dim = int(lib().sps_model_ndim(h))

    def close(self):
        if getattr(self, "handle", None):
            lib().sps_destroy_table(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def sps_create_table(grid, exact_precision=EXACT_BF16X3, model=MODEL_DPL13, gauss=None, dlogZ_dlogage=0.0) -> Table:
    return Table(grid, exact_precision, model, gauss, dlogZ_dlogage)


def sps_set_option(option: int, value: int):
    _check(lib().sps_set_option(int(option), int(value)), "sps_set_option")


def sps_table_cssp(table: Table) -> np.ndarray:
    out = np.empty((table.n_z, table.n_age * table.n_Z, table.n_band), np.float32)
    _check(lib().sps_table_cssp(table.handle, out.ctypes.data_as(C.POINTER(C.c_float))), "sps_table_cssp")
    return out


def _new(shape, dtype=None, like=None):
    import torch
    return torch.empty(shape, dtype=dtype or torch.float32, device=like.device if like is not None else "cuda")


def sps_weights(table, prior, theta, unbounded=True):
    n = theta.shape[0]
    w_age, w_met, mstar = _new((n, table.n_age), like=theta), _new((n, table.n_Z), like=theta), _new((n,), like=theta)
    _check(lib().sps_weights(table.handle, prior.ref() if prior else None, _dptr(theta), C.c_int64(n), int(unbounded),
                             _dptr(w_age), _dptr(w_met), _dptr(mstar), _stream()), "sps_weights")
    return w_age, w_met, mstar


def sps_photometry(table, prior, path, theta, unbounded=True, flux_bar=None):
    n = theta.shape[0]
    flux = _new((n, table.n_band), like=theta)
    theta_bar = _new((n, NDIM), like=theta) if flux_bar is not None else None
    _check(lib().sps_photometry(table.handle, prior.ref() if prior else None, int(path), _dptr(theta), C.c_int64(n),
                                int(unbounded), _dptr(flux), _dptr(flux_bar), _dptr(theta_bar), _stream()), "sps_photometry")
    return (flux, theta_bar) if flux_bar is not None else flux


def sps_loglike_grad(table, prior, path, theta_unb, obs_flux, obs_sigma, gal_of_row=None, want_grad=True, out=None):
    n = theta_unb.shape[0]
    logp, grad = out if out is not None else (_new((n,), like=theta_unb), _new((n, NDIM), like=theta_unb) if want_grad else None)
    _check(lib().sps_loglike_grad(table.handle, prior.ref() if prior is not None else None, int(path), _dptr(theta_unb), C.c_int64(n), _dptr(gal_of_row),
                                  _dptr(obs_flux), _dptr(obs_sigma), _dptr(logp), _dptr(grad), _stream()), "sps_loglike_grad")
    return logp, grad


NOALLOC_MAX_ROWS, NOALLOC_MAX_NZ = 4096, 1024


def sps_loglike_grad_noalloc(table, prior, theta_unb, obs_flux, obs_sigma, logp, grad, gal_of_row=None):
    """sps_loglike_grad on the approximate path with the library's fixed scratch array: no allocation here or in the
    library (the caller passes the outputs: logp [n], grad [n, 13] or None).  n <= NOALLOC_MAX_ROWS."""
    n = theta_unb.shape[0]
    _check(lib().sps_loglike_grad_noalloc(table.handle, prior.ref(), _dptr(theta_unb), C.c_int64(n), _dptr(gal_of_row), _dptr(obs_flux),
                                          _dptr(obs_sigma), _dptr(logp), _dptr(grad), _stream()), "sps_loglike_grad_noalloc")
    return logp, grad


def sps_leapfrog(table, prior, path, theta0, p0, eps, inv_mass, obs_flux, obs_sigma, n_steps, gal_of_row=None):
    n = theta0.shape[0]
    traj = _new((n_steps, n, 2, NDIM), like=theta0)
    logp = _new((n_steps, n), like=theta0)
    _check(lib().sps_leapfrog(table.handle, prior.ref() if prior is not None else None, int(path), _dptr(theta0), _dptr(p0), _dptr(eps), _dptr(inv_mass),
                              C.c_int64(n), _dptr(gal_of_row), _dptr(obs_flux), _dptr(obs_sigma), C.c_int32(n_steps),
                              _dptr(traj), _dptr(logp), _stream()), "sps_leapfrog")
    return traj, logp


def sps_hmc_run(table, prior, obs_flux, obs_sigma, *, sampler=SAMPLER_HMC, path=PATH_APPROX, n_chain=4, n_warmup=500,
                n_sample=500, n_leapfrog=16, max_depth=8, eps0=0.05, target_accept=0.8, seed=1, path_of_gal=None,
                theta0=None, keep_samples=False, first_transition=0, eps_in=None, inv_mass_in=None, gal_id=None, n_gal=None):
    """obs_flux / obs_sigma [n_gal, n_band] (None for MODEL_GAUSS_TEST, which takes n_gal = number of independent groups of
    n_chain chains)."""
    import torch
    n_gal = obs_flux.shape[0] if obs_flux is not None else int(n_gal)
    nc = n_gal * n_chain
    dev = obs_flux.device if obs_flux is not None else torch.device("cuda")
    f32 = lambda *s: torch.zeros(s, dtype=torch.float32, device=dev)
    i32 = lambda *s: torch.zeros(s, dtype=torch.int32, device=dev)
    out = dict(mean=f32(nc, NDIM), sd=f32(nc, NDIM), accept=f32(nc), eps=f32(nc), inv_mass=f32(nc, NDIM),
               n_leapfrog=i32(nc), divergences=i32(nc), rhat=f32(n_gal, NDIM), theta_last=f32(nc, NDIM), ess=f32(n_gal, NDIM),
               depth_hist=i32(11))
    samples = f32(nc, n_sample, NDIM) if keep_samples else None
    cfg = _HmcConfig(int(sampler), int(path), int(n_chain), int(n_warmup), int(n_sample), int(n_leapfrog), int(max_depth),
                     float(eps0), float(target_accept), int(seed), int(first_transition),
                     eps_in.data_ptr() if eps_in is not None else None, inv_mass_in.data_ptr() if inv_mass_in is not None else None,
                     gal_id.data_ptr() if gal_id is not None else None)
    summ = _HmcSummary(*[out[k].data_ptr() for k in ("mean", "sd", "accept", "eps", "inv_mass", "n_leapfrog", "divergences", "rhat", "theta_last",
                                                     "ess", "depth_hist")])
    _check(lib().sps_hmc_run(table.handle, prior.ref() if prior is not None else None, C.byref(cfg), _dptr(obs_flux), _dptr(obs_sigma), C.c_int64(n_gal),
                             _dptr(path_of_gal), _dptr(theta0), _dptr(samples), C.byref(summ), _stream()), "sps_hmc_run")
    if keep_samples:
        out["samples"] = samples
    return out


def sps_philox_words(seed, first_chain, transition, purpose, index, n):
    import torch
    out = torch.empty((n, 4), dtype=torch.int32, device="cuda")
    _check(lib().sps_philox_words(C.c_uint64(seed), C.c_uint32(first_chain), C.c_uint32(transition), C.c_uint32(purpose),
                                  C.c_uint32(index), C.c_int64(n), _dptr(out), _stream()), "sps_philox_words")
    return out


def sps_exact_last_work(table) -> int:
    v = C.c_int64()
    _check(lib().sps_exact_last_work(table.handle, C.byref(v)), "sps_exact_last_work")
    return int(v.value)


def sps_exact_work_since(table):
    """-> ((row, wavelength) pairs, exact forward calls) since the previous call."""
    v, c = C.c_int64(), C.c_int64()
    _check(lib().sps_exact_work_since(table.handle, C.byref(v), C.byref(c)), "sps_exact_work_since")
    return int(v.value), int(c.value)


def sps_measure_peak(what: str) -> float:
    """'mufu' (ex2.approx / s) or 'ffma' (fp32 FMA / s), measured now on the current device."""
    v = C.c_double()
    _check(lib().sps_measure_peak({"mufu": 0, "ffma": 1}[what], C.byref(v), _stream()), "sps_measure_peak")
    return float(v.value)


def sps_launch_count() -> int:
    return int(lib().sps_launch_count())


KERNEL_IDS = {"prologue": 0, "approx_contract": 1, "epilogue": 2, "exact_fwd": 3, "exact_bwd": 4}


def sps_profile(enable: bool, stride: int = 1):
    _check(lib().sps_profile(int(enable), int(stride)), "sps_profile")


def sps_profile_read(kernel: str):
    """-> (total_ms over the timed launches, timed launches, all launches) since the last read."""
    ms, n, a = C.c_double(), C.c_int64(), C.c_int64()
    _check(lib().sps_profile_read(KERNEL_IDS[kernel], C.byref(ms), C.byref(n), C.byref(a)), "sps_profile_read")
    return ms.value, n.value, a.value
