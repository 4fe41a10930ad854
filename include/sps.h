/* sps.h -- C ABI of the B200-native SPS photometry / HMC library (libsps_b200.so).
 *
 * The library computes, on one NVIDIA B200 (sm_100a), the data-parallel hot path of
 * arXiv:2506.19919 ("Bayesian posteriors with stellar population synthesis on GPUs"): the batched
 * galaxy-photometry log-likelihood and its gradient inside every HMC / NUTS leapfrog step.
 * Citations are PAPER.md:<line> of the reference text; R# are the readings listed in DESIGN.md.
 *
 * Conventions (all entry points):
 *   - `*_dev` / "device" pointers are raw CUDA device pointers owned by the CALLER (e.g. torch
 *     data_ptr()); "host" pointers are ordinary host memory.  The library never frees caller memory.
 *   - Arrays are row-major, float32 unless stated.  A parameter row always has SPS_NDIM = 13 slots; the table's model
 *     (sps_table_desc.model) fixes what they mean and how many of them are SAMPLED (sps_model_ndim):
 *       SPS_MODEL_DPL13 (the paper's model; 13 sampled):
 *         logM, tau, alpha, beta, F_burst, logT_peak, logT_max, logZ, sigma_logZ, A_V, delta, F_floor, z
 *         (z per BASELINE.json configs[1])
 *       SPS_MODEL_TINY5 (BASELINE.json configs[0]; R19; 4 sampled + the redshift as data):
 *         logM_star, log10 tau [Gyr], logZ, tau_V, z (slot 4: read, never transformed, never moved by the samplers),
 *         slots 5-12 ignored
 *       SPS_MODEL_GAUSS_TEST (a correlated Gaussian target for the samplers; gauss_ndim sampled): theta_0 .. theta_{D-1}
 *     Slots that are not sampled are ignored on input (except TINY5's z) and written as zero in gradients.
 *   - `stream` is a cudaStream_t passed as void* (NULL = default stream).  Calls enqueue work and
 *     return without synchronising unless stated.
 *   - Every call returns an sps_status; no exception crosses the ABI; sps_last_error() gives a
 *     thread-local message for the last non-OK status.
 *   - A table is immutable after sps_create_table.  Scratch memory is owned by the library PER (table, stream): calls on
 *     different streams (from one or several host threads) use different scratch and may overlap; calls on the same
 *     stream are ordered by the stream and must be issued from one host thread at a time.  Scratch grows on demand
 *     (growing synchronises that stream) and is freed by sps_destroy_table.
 *   - obs_sigma must be > 0 everywhere (it divides); with SPS_OPT_CHECK_FINITE set, non-finite parameters or
 *     observations and non-positive sigmas are reported as SPS_ENONFINITE (a device reduction + one synchronisation per
 *     call: a debugging aid, off by default so that the hot path never synchronises).
 *   - There is NO CPU fallback: without a compute-capability-10.x device every compute call returns
 *     SPS_EUNSUPPORTED.
 */
#ifndef SPS_H_
#define SPS_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define SPS_NDIM 13

typedef enum {
  SPS_OK = 0,
  SPS_EINVAL = 1,        /* null pointer, bad enum, non-monotonic grid ...            */
  SPS_ESHAPE = 2,        /* a size is out of the supported range                      */
  SPS_ECUDA = 3,         /* a CUDA runtime call failed (message has the CUDA string)  */
  SPS_ENOMEM = 4,
  SPS_EUNSUPPORTED = 5,  /* no sm_100 device                                          */
  SPS_ENONFINITE = 6     /* SPS_OPT_CHECK_FINITE found a non-finite input             */
} sps_status;

enum { SPS_MODEL_TINY5 = 0, SPS_MODEL_DPL13 = 1, SPS_MODEL_GAUSS_TEST = 2 };
enum { SPS_PATH_EXACT = 0, SPS_PATH_APPROX = 1 };
enum { SPS_SAMPLER_HMC = 0, SPS_SAMPLER_NUTS = 1 };
/* Operand format of the exact path's tensor-core contractions (three split products a_lo b_hi + a_hi b_lo + a_hi b_hi,
 * fp32 accumulation in TMEM).  BF16X3: ~2^-17 per product, 16 K-elements per accumulator update.  TF32X3: ~2^-21 per
 * product but twice the operand bytes, half the MMA rate and twice the accumulator updates; since tcgen05 accumulation
 * truncates (measured ~2.4e-8 relative per update) BF16X3 is both faster and, end to end, more accurate
 * on this problem, hence the default. */
enum { SPS_EXACT_BF16X3 = 0, SPS_EXACT_TF32X3 = 1 };

typedef struct sps_table sps_table;      /* opaque; owns device memory */

/* Everything that is fixed before the analysis.  HOST pointers; copied. */
typedef struct {
  int32_t n_age, n_Z, n_wave, n_band, n_z;   /* n_age<=128, n_Z<=16, n_band<=16, n_z>=2; and       */
                                             /* 8 n_age (n_Z n_band + 4) + 119 KB <= 227 KB (SPS_ESHAPE otherwise) */
  const double* log10_age_yr;  /* [n_age]  increasing                                              */
  const double* log10_Z;       /* [n_Z]    increasing, log10(Z/Zsun)                               */
  const double* wave_A;        /* [n_wave] strictly increasing rest-frame wavelength, Angstrom     */
  const float*  ssp;           /* [n_age*n_Z][n_wave] L_SSP(lambda|age_i,Z_j), row = i*n_Z + j     */
  const double* filt_mu_A;     /* [n_band] Gaussian filter centre, observed frame   */
  const double* filt_sigma_A;  /* [n_band] Gaussian sigma; support truncated at 5 sigma (R4)       */
  double z_min, z_max;         /* uniform redshift grid of the c_SSP lookup table    */
  double H0, Om;               /* flat LCDM for t_obs(z) (R11)                       */
  double log10_mass_unit;      /* M_star is expressed in 10^this Msun so that fluxes are O(1)      */
  int32_t exact_precision;     /* SPS_EXACT_BF16X3 (0, default) or SPS_EXACT_TF32X3                */
  int32_t model;               /* SPS_MODEL_TINY5 (0) | SPS_MODEL_DPL13 (1) | SPS_MODEL_GAUSS_TEST (2)            */
  /* Tabulated filters (T(lambda) is a general transmission curve; R4): when filt_offsets != NULL the
   * Gaussian arrays above are ignored and band b is the curve through the knots offsets[b] .. offsets[b+1]-1 of
   * (filt_wave_A, filt_trans): observed-frame Angstrom, strictly increasing inside a band, at least 2 and at most 4096
   * knots per band; linear interpolation between knots, zero outside [first knot, last knot]. */
  const double*  filt_wave_A;  /* [filt_offsets[n_band]] or NULL                                    */
  const double*  filt_trans;   /* [filt_offsets[n_band]] or NULL                                    */
  const int32_t* filt_offsets; /* [n_band + 1] or NULL (Gaussian filters)                           */
  /* Non-separable weights (R26; SPS_MODEL_DPL13 only): the median of the lognormal MDF of
   * age bin i is logZ + dlogZ_dlogage (log10 age_i/yr - 9).  0 = the paper's separable model, Eq. (2). */
  double dlogZ_dlogage;
  /* SPS_MODEL_GAUSS_TEST: logP(theta) = -1/2 (theta - mu)^T P (theta - mu) over gauss_ndim <= 13 parameters; the grids,
   * spectra and filters above may be NULL / 0 for this model, and observations are ignored by every call. */
  int32_t gauss_ndim;
  const double* gauss_mu;      /* [gauss_ndim]                                                      */
  const double* gauss_prec;    /* [gauss_ndim][gauss_ndim] symmetric positive definite precision    */
} sps_table_desc;

/* Per-parameter hyper-parameters, HOST arrays of SPS_NDIM doubles each.
 * Bounding sigmoid Eq. (C1): theta = y_lo + (y_hi-y_lo)/(1+exp(-k(theta~-x0))).
 * Skew-normal prior on theta~ Eq. (C2): (2/omega) N(u) Phi(s u), u=(theta~-xi)/omega. */
typedef struct {
  const double *y_lo, *y_hi, *k, *x0, *xi, *omega, *skew;
} sps_prior;

/* sps_create_table: upload the grids, precompute quadrature weights (R4), per-wavelength dust
 * constants (Eq. A8, R10), lambda_eff (Eq. 5) and the c_SSP[n_z][n_age][n_Z][n_band] lookup table
 * (Eq. 7) ON THE GPU, and build the tensor-core operand layouts of the SSP table.
 * Synchronises.  On success *out owns all device memory until sps_destroy_table. */
sps_status sps_create_table(const sps_table_desc* desc, sps_table** out);
sps_status sps_destroy_table(sps_table* t);

/* Number of sampled parameters of the table's model: 13 (DPL13), 4 (TINY5), gauss_ndim (GAUSS_TEST); -1 for NULL. */
int32_t sps_model_ndim(const sps_table* t);

/* Library options (process-wide; testing and debugging aids, none is needed for normal use).  Returns SPS_EINVAL for an
 * unknown option.
 *   SPS_OPT_CHECK_FINITE   1: sps_weights / sps_photometry / sps_loglike_grad / sps_leapfrog / sps_hmc_run validate their
 *                             device inputs (one reduction kernel + one synchronisation) and return SPS_ENONFINITE
 *   SPS_OPT_EXACT_SIMT     1: the exact path runs its fp32 SIMT contraction kernels instead of the tcgen05 ones
 *   SPS_OPT_APPROX_SIMT    1: the approximate path runs its fp32 SIMT contraction kernel instead of the tcgen05 one
 *   SPS_OPT_NO_TC_SETUP    1: tables created from now on build no tensor-core operands (SIMT kernels only)
 *   SPS_OPT_NO_GRAPH       1: sps_hmc_run launches every kernel directly instead of replaying a CUDA graph
 *   SPS_OPT_ROW_GROUPS     n: fixed-length HMC splits its chains into n (1..4) groups whose evaluations run on different
 *                             streams (an experiment in overlapping one group's contraction with another's row
 *                             kernels; measured slower); 0 or 1 = one group.  Results do not depend on it.
 *   SPS_OPT_NO_PDL         1: the prologue / contraction / epilogue kernels are launched with plain stream order instead of
 *                             programmatic dependent launch (each kernel's launch and set-up then no longer overlap the
 *                             tail of the one before it).  Results do not depend on it. */
enum { SPS_OPT_CHECK_FINITE = 0, SPS_OPT_EXACT_SIMT = 1, SPS_OPT_APPROX_SIMT = 2, SPS_OPT_NO_TC_SETUP = 3, SPS_OPT_NO_GRAPH = 4,
       SPS_OPT_ROW_GROUPS = 5, SPS_OPT_NO_PDL = 6, SPS_OPT_COUNT = 7 };
sps_status sps_set_option(int option, int value);

/* Copy the c_SSP table to a HOST buffer of n_z*n_age*n_Z*n_band floats (diagnostic; synchronises). */
sps_status sps_table_cssp(const sps_table* t, float* cssp_host);

/* sps_weights (diagnostic observable for the 1e-5 weights tolerance): Eq. (A3)-(A7), (2).
 * theta_dev [n,13]; unbounded != 0 means theta_dev holds theta~ and needs `prior` for Eq. (C1)
 * (prior may be NULL when unbounded == 0).  Outputs (device): w_age [n,n_age] = P_SFH (Eq. A6),
 * w_met [n,n_Z] = P_met, mstar [n] = M_star / mass_unit (Eq. A3).  For a table with dlogZ_dlogage != 0 (non-separable
 * weights: every age bin has its own MDF) w_met is the MDF at age 1 Gyr, i.e. with median logZ itself. */
sps_status sps_weights(const sps_table* t, const sps_prior* prior, const float* theta_dev, int64_t n,
                       int unbounded, float* w_age_dev, float* w_met_dev, float* mstar_dev, void* stream);

/* sps_photometry: band fluxes by the exact path (Eq. 4: tensor-core contraction
 * against the SSP table, dust and redshifted filters in the epilogue) or the approximate path
 * (Eq. 6: F_att(lambda_eff) times P_SSP-weighted sums of the z-interpolated c_SSP).
 * flux_dev [n,n_band] out.  If flux_bar_dev [n,n_band] and theta_bar_dev [n,13] are both non-NULL the
 * vector-Jacobian product theta_bar = flux_bar^T dflux/dtheta is also written (w.r.t. theta~ when
 * unbounded != 0, else w.r.t. theta) (R20). */
sps_status sps_photometry(const sps_table* t, const sps_prior* prior, int path, const float* theta_dev,
                          int64_t n, int unbounded, float* flux_dev, const float* flux_bar_dev,
                          float* theta_bar_dev, void* stream);

/* sps_loglike_grad: logP(theta~) = -1/2 sum_b((flux_b-d_b)/sigma_b)^2 + sum_p log SN(theta~_p)
 * (R12) and its gradient w.r.t. theta~ (fused reverse mode).
 * theta_unb_dev [n,13]; gal_of_row_dev [n] int32 row -> galaxy index (NULL: row r uses galaxy r);
 * obs_flux_dev, obs_sigma_dev [n_gal,n_band]; outputs logp_dev [n], grad_dev [n,13]. */
sps_status sps_loglike_grad(const sps_table* t, const sps_prior* prior, int path,
                            const float* theta_unb_dev, int64_t n, const int32_t* gal_of_row_dev,
                            const float* obs_flux_dev, const float* obs_sigma_dev, float* logp_dev,
                            float* grad_dev, void* stream);

/* sps_loglike_grad_noalloc: sps_loglike_grad on the approximate path (Eq. 6) for callers that may not
 * allocate (code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc).  Same arguments, results
 * and kernels; the per-row scratch lives in one fixed 15.8 MB device array inside the library (held by every GPU that loads
 * it until the process exits) instead of the per-stream workspace, and the call makes no cudaMalloc / cudaFree.
 * Limits: n <= SPS_NOALLOC_MAX_ROWS and the table's n_z <= SPS_NOALLOC_MAX_NZ, else SPS_ESHAPE; not for
 * SPS_MODEL_GAUSS_TEST (no scratch there) and not while sps_profile is on (SPS_EINVAL); SPS_OPT_CHECK_FINITE is not applied.
 * All calls on a device share the array: calls that overlap on the GPU (different streams) race, so order them.  The first
 * call on each device resolves the array's device address and should be made outside graph capture.  Does not synchronise. */
#define SPS_NOALLOC_MAX_ROWS 4096
#define SPS_NOALLOC_MAX_NZ 1024
sps_status sps_loglike_grad_noalloc(const sps_table* t, const sps_prior* prior, const float* theta_unb_dev, int64_t n,
                                    const int32_t* gal_of_row_dev, const float* obs_flux_dev, const float* obs_sigma_dev,
                                    float* logp_dev, float* grad_dev, void* stream);

/* sps_leapfrog (diagnostic for the trajectory tolerance): n_steps leapfrog steps
 * p += eps/2 grad; theta~ += eps invM*p; p += eps/2 grad from (theta0, p0); per-row eps
 * [n] and diagonal inverse mass [n,13].  traj_dev [n_steps,n,2,13] receives (theta~, p) after each
 * step; logp_traj_dev [n_steps,n] the log-posterior. */
sps_status sps_leapfrog(const sps_table* t, const sps_prior* prior, int path, const float* theta0_dev,
                        const float* p0_dev, const float* eps_dev, const float* inv_mass_dev, int64_t n,
                        const int32_t* gal_of_row_dev, const float* obs_flux_dev,
                        const float* obs_sigma_dev, int32_t n_steps, float* traj_dev,
                        float* logp_traj_dev, void* stream);

typedef struct {
  int32_t sampler;        /* SPS_SAMPLER_HMC | SPS_SAMPLER_NUTS          */
  int32_t path;           /* default path; overridden per galaxy by path_of_gal_dev when non-NULL     */
  int32_t n_chain;        /* chains per galaxy                                                        */
  int32_t n_warmup;       /* adaptation transitions (R14: windowed dual averaging + diagonal mass)    */
  int32_t n_sample;       /* kept transitions                                                         */
  int32_t n_leapfrog;     /* HMC trajectory length                                                    */
  int32_t max_depth;      /* NUTS maximum tree depth (<= 10)                                          */
  float   eps0;           /* initial step size                                                        */
  float   target_accept;  /* dual-averaging target (0.8)                                              */
  uint64_t seed;          /* Philox4x32-10 key (R16)                                                  */
  /* Continuing chains (unconverged fits "require an additional ~N_steps"): the transition counter of the
   * RNG streams starts at first_transition, and the adapted step sizes / inverse masses of an earlier run are taken
   * instead of (eps0, unit mass) when the DEVICE arrays below are non-NULL.  With theta0 = the earlier run's theta_last,
   * n_warmup = 0 and first_transition = transitions already done, a run continues exactly where it stopped. */
  uint32_t first_transition;
  const float* eps_in_dev;       /* [n_gal*n_chain]    or NULL */
  const float* inv_mass_in_dev;  /* [n_gal*n_chain,13] or NULL */
  /* RNG stream of each galaxy: chain k of galaxy g draws from Philox stream gal_id[g]*n_chain + k (NULL: gal_id[g] = g).
   * Continuing only the unconverged galaxies of an earlier run with their original ids reproduces, bit for
   * bit, what continuing every galaxy would have given them. */
  const int32_t* gal_id_dev;     /* [n_gal] or NULL */
} sps_hmc_config;

/* Per-chain summaries, DEVICE pointers, any may be NULL.  Chain index c = gal*n_chain + chain. */
typedef struct {
  float* mean;          /* [n_gal*n_chain,13] posterior mean of theta~ over kept samples              */
  float* sd;            /* [n_gal*n_chain,13] posterior standard deviation (n-1)                      */
  float* accept;        /* [n_gal*n_chain]    mean accept statistic over the sampling phase           */
  float* eps;           /* [n_gal*n_chain]    adapted step size                                       */
  float* inv_mass;      /* [n_gal*n_chain,13] adapted diagonal inverse mass                           */
  int32_t* n_leapfrog;  /* [n_gal*n_chain]    total leapfrog steps taken                              */
  int32_t* divergences; /* [n_gal*n_chain]    divergent transitions in the sampling phase             */
  float* rhat;          /* [n_gal,13]         Gelman-Rubin statistic over the galaxy's chains */
  float* theta_last;    /* [n_gal*n_chain,13] state of every chain after its last transition (to continue from)     */
  float* ess;           /* [n_gal,13]         effective sample size by batch means pooled over the galaxy's chains (R25)  */
  int32_t* depth_hist;  /* [11]               NUTS: kept transitions per final tree depth 0..10       */
} sps_hmc_summary;

/* (sps_hmc_run and sps_leapfrog take their per-run device buffers from a process-wide cache of blocks and hand them back at
 * the end: no cudaFree per call; sps_destroy_table releases the blocks that are not in use.) */
/* sps_hmc_run: n_gal galaxies x n_chain chains of (n_warmup + n_sample) transitions.
 * obs_flux_dev/obs_sigma_dev [n_gal,n_band]; path_of_gal_dev [n_gal] int32 or NULL;
 * theta0_unb_dev [n_gal*n_chain,13] or NULL (R17: xi + 0.1 omega N(0,1));
 * samples_dev [n_gal*n_chain, n_sample, 13] or NULL.  Synchronises before returning. */
sps_status sps_hmc_run(const sps_table* t, const sps_prior* prior, const sps_hmc_config* cfg,
                       const float* obs_flux_dev, const float* obs_sigma_dev, int64_t n_gal,
                       const int32_t* path_of_gal_dev, const float* theta0_unb_dev, float* samples_dev,
                       const sps_hmc_summary* summary, void* stream);

/* Raw Philox4x32-10 words for the bit-exact RNG parity test (R16): out_dev [n,4] uint32 for counters
 * (chain = first_chain + i, transition, purpose, index), key from seed. */
sps_status sps_philox_words(uint64_t seed, uint32_t first_chain, uint32_t transition, uint32_t purpose,
                            uint32_t index, int64_t n, uint32_t* out_dev, void* stream);

/* Per-kernel device timing for bench.py's roofline line.  sps_profile(1) makes the library bracket
 * every `stride`-th launch of its main kernels with CUDA events on the launching stream;
 * sps_profile_read(kernel_id, &total_ms, &timed_launches, &all_launches) synchronises, sums the recorded
 * pairs for that kernel and clears them.  kernel_id: 0 prologue (weights), 1 approximate contraction,
 * 2 epilogue (reverse of the weights + prior), 3 exact forward GEMM, 4 exact reverse GEMM. */
enum { SPS_K_PROLOGUE = 0, SPS_K_APPROX = 1, SPS_K_EPILOGUE = 2, SPS_K_EXACT_FWD = 3, SPS_K_EXACT_BWD = 4, SPS_K_COUNT = 5 };
sps_status sps_profile(int enable, int stride);
sps_status sps_profile_read(int kernel_id, double* total_ms, int64_t* timed_launches, int64_t* all_launches);

/* Algorithmic work of the last exact-path forward call on this table: the number of (row, wavelength) pairs that lie
 * under some filter's 5-sigma support at the row's redshift (everything else contributes exactly zero to Eq. 4 and is
 * skipped).  bench.py's tensor roofline counts 3 x 2 x n_age*n_Z flop per pair and pass.  Synchronises. */
sps_status sps_exact_last_work(const sps_table* t, int64_t* row_wavelength_pairs);
/* The same summed over the exact-path forward calls (on the stream used last) since the previous call of this function,
 * and their number: the average work per launch of a sampler run, whose launches shrink as trees finish.  Synchronises. */
sps_status sps_exact_work_since(const sps_table* t, int64_t* row_wavelength_pairs, int64_t* calls);

/* Throughput of one execution pipe, measured now on the current device (a microbenchmark of ~10 ms; synchronises):
 * SPS_PEAK_MUFU: ex2.approx operations per second (the special-function units the SFH quadrature is bound by),
 * SPS_PEAK_FFMA: fp32 fused multiply-adds per second.  bench.py's "alu" roofline uses them as denominators, so that
 * they are taken at the clocks of the same run. */
enum { SPS_PEAK_MUFU = 0, SPS_PEAK_FFMA = 1 };
sps_status sps_measure_peak(int what, double* per_second, void* stream);

/* Number of kernels this library launched since load (for bench.py's gpu_launches). */
int64_t sps_launch_count(void);

const char* sps_last_error(void);
const char* sps_version(void);

#ifdef __cplusplus
}
#endif
#endif /* SPS_H_ */
