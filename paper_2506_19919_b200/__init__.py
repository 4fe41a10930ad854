"""paper_2506_19919_b200 -- B200-native (sm_100a) SPS photometry log-likelihood / HMC hot path of
arXiv:2506.19919 behind a C ABI (include/sps.h).  Importing the package does not load the CUDA
library; the first call does, and fails loudly if it is missing (no CPU fallback)."""
from . import workloads  # noqa: F401  (numpy-only input generators)
from .binding import (EXACT_BF16X3, EXACT_TF32X3, MODEL_DPL13, MODEL_GAUSS_TEST, MODEL_TINY5, OPT_APPROX_SIMT, OPT_CHECK_FINITE, OPT_EXACT_SIMT,
                      OPT_NO_GRAPH, OPT_NO_PDL, OPT_NO_TC_SETUP, OPT_ROW_GROUPS, PATH_APPROX, PATH_EXACT, SAMPLER_HMC, SAMPLER_NUTS, PriorHandle, SpsError, Table,  # noqa: F401
                      sps_create_table, sps_exact_last_work, sps_exact_work_since, sps_hmc_run, sps_launch_count, sps_measure_peak, sps_leapfrog, sps_loglike_grad, sps_loglike_grad_noalloc,
                      sps_philox_words, sps_photometry, sps_profile, sps_profile_read, sps_set_option, sps_table_cssp, sps_weights)
