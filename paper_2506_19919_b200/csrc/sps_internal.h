// sps_internal.h -- host-side internals of libsps_b200 (not part of the ABI).
#pragma once
#include <cuda.h>
#include <map>
#include <mutex>
#include "sps_rows.cuh"

struct ExactState;   // sps_exact.cuh: table-constant operands of the exact path
struct ApproxTc;     // sps_approx_tc.cu: table-constant operands of the tensor-core approximate contraction

// Scratch of the exact path for one (table, stream): everything a call writes.
struct ExactScratch {
  float* W;                 // [cap][ldw]  forward operand W = Mn a (x) m  (fp32 SIMT kernels)
  float* Wbar;              // [cap][ldw]  reverse result
  long long* part;          // [cap][5][SPS_MAX_BAND] band sums (flux and its direct partials A_V, delta, F_floor, z) as
                            //                        fixed-point integers: integer atomics make them order-independent
  float* gbuf;              // [cap][SPS_MAX_BAND]    d logL / d flux_b
  int* sorted;              // [cap] rows of the current call ordered by redshift
  int* zhist;               // [2][1024] counting-sort histogram / cursors
  int64_t cap;
  // tensor-core row operands (split W and SEDbar), their TMA maps and the per-row-tile plan
  void *W_hi, *W_lo, *SB_hi, *SB_lo;
  int* plan; int plan_cap;
  unsigned long long* work; // [2] (row, wavelength) pairs of the last forward call; running total since the last sps_exact_work_since
  int64_t work_calls;       // forward calls since then
  CUtensorMap mW_hi, mW_lo, mSB_hi, mSB_lo;
  int64_t tc_cap;
};

struct Workspace {
  RowBuffers rows;
  ExactScratch x;
  // the z-cell counts in rows.bins are all zero (stream order): true after the tensor-core contraction, whose last CTA to
  // read them clears them, so the next prologue of this workspace needs no memset node in front of it
  bool bins_clean;
  Workspace() : bins_clean(false) { rows = RowBuffers(); x = ExactScratch(); }
};

struct sps_table {
  TableDev dev;
  ExactState* exact;        // built at creation, immutable afterwards
  ApproxTc* approx_tc;      // or null: the SIMT contraction kernel is used
  int sm_count;
  // scratch per stream, created on first use (the table itself is immutable, hence `const sps_table*` at the ABI)
  mutable std::mutex mu;
  mutable std::map<cudaStream_t, Workspace*> ws;
  mutable Workspace* last_ws;          // for sps_exact_last_work
  mutable cudaStream_t own_stream;     // sps_hmc_run on the legacy default stream runs here (graph capture needs a real stream)
  mutable cudaStream_t aux_stream[3];  // streams of the sampler's additional row groups (sps_sampler.cu)
  sps_table() : exact(nullptr), approx_tc(nullptr), sm_count(0), last_ws(nullptr), own_stream(nullptr) { aux_stream[0] = aux_stream[1] = aux_stream[2] = nullptr; }
};

// library options (sps_set_option)
int sps_option(int option);

sps_status sps_require_device();
Workspace* sps_workspace(const sps_table* t, cudaStream_t s);                 // never null; thread-safe
sps_status sps_ensure_row_buffers(const sps_table* t, Workspace& ws, int64_t n, cudaStream_t s);
void sps_free_workspace(Workspace* ws);
// process-wide cache of device blocks for the samplers' per-run state (sps_api.cu): alloc reuses a free block of a fitting
// size, free hands the block back (no cudaFree), release_unused frees the idle ones (sps_destroy_table)
cudaError_t sps_pool_alloc(void** p, size_t bytes);
void sps_pool_free(void* p);
void sps_pool_release_unused();
sps_status sps_prior_to_dev(const sps_table* t, const sps_prior* p, PriorDev& out);
// SPS_OPT_CHECK_FINITE: device reduction over the given arrays (any may be null); SPS_ENONFINITE if one entry is not finite
// or a `positive` entry is <= 0.  No-op (SPS_OK) when the option is off.
sps_status sps_check_finite(const float* a, int64_t na, const float* b, int64_t nb, const float* positive, int64_t np, cudaStream_t s);

// exact path (sps_exact.cu)
sps_status sps_exact_setup(sps_table* t, int precision);
void sps_exact_teardown(sps_table* t);
void sps_exact_free_scratch(ExactScratch& X);
// flux + (optional) reverse pass over the SSP table for rows whose prologue has run:
// fills B.flux, B.sc[*].logp_like and, if want_grad, B.a_bar, B.m_bar and the scalar bars.
sps_status sps_exact_contract(const sps_table* t, Workspace& ws, int64_t n, const int* rows, const int* gal_of_row, const float* obs_flux,
                              const float* obs_sigma, const float* flux_bar, bool want_grad, cudaStream_t s);

// tensor-core approximate contraction (sps_approx_tc.cu); same contract as launch_approx_contract
sps_status sps_approx_tc_setup(sps_table* t);
void sps_approx_tc_teardown(sps_table* t);
bool sps_approx_tc_active(const sps_table* t);
sps_status sps_approx_tc_contract(const sps_table* t, Workspace& ws, int64_t n, const int* rows, const int* gal_of_row, const float* obs_flux,
                                  const float* obs_sigma, const float* flux_bar, bool want_grad, cudaStream_t s);

// full model evaluation used by the API and the sampler (sps_api.cu)
sps_status sps_eval(const sps_table* t, Workspace& ws, const PriorDev& P, int path, const float* theta, int64_t n, bool unbounded,
                    bool with_prior, const int* rows, const int* gal_of_row, const float* obs_flux,
                    const float* obs_sigma, const float* flux_bar, bool want_grad, float* logp, float* grad,
                    cudaStream_t s, const LeapfrogFuse* lf = nullptr, bool overlap = false);

// approximate path with non-separable weights (sps_nonsep.cu; R26)
void launch_nonsep_approx(const TableDev& T, int64_t n, const int* rows, const int* gal_of_row, const float* obs_flux, const float* obs_sigma,
                          const float* flux_bar, bool want_grad, RowBuffers B, cudaStream_t s);

// other models (sps_models.cu): SPS_MODEL_TINY5 row kernels and the SPS_MODEL_GAUSS_TEST target
void launch_prologue_tiny5(const TableDev& T, const PriorDev& P, const float* theta, int64_t n, bool unbounded, const int* rows,
                           RowBuffers B, bool with_hist, cudaStream_t s);
void launch_epilogue_tiny5(const TableDev& T, const PriorDev& P, const float* theta, int64_t n, bool unbounded, bool with_prior,
                           const int* rows, RowBuffers B, float* logp, float* grad, LeapfrogFuse lf, cudaStream_t s);
void launch_gauss_eval(const TableDev& T, const float* theta, int64_t n, const int* rows, float* logp, float* grad, LeapfrogFuse lf,
                       cudaStream_t s);
