// sps_internal.h -- host-side internals of libsps_b200 (not part of the ABI).
#pragma once
#include "sps_rows.cuh"

struct ExactState;   // sps_exact.cu

struct sps_table {
  TableDev dev;
  RowBuffers rows;         // scratch, grown on demand; a table must not be used from two host threads at once
  ExactState* exact;
  void* approx_tc;         // ApproxTc (sps_approx_tc.cu) or null: the SIMT contraction kernel is used
  sps_table() : exact(nullptr), approx_tc(nullptr) { rows = RowBuffers(); }
};

sps_status sps_require_device();
sps_status sps_ensure_row_buffers(sps_table* t, int64_t n);
void sps_free_row_buffers(sps_table* t);
sps_status sps_prior_to_dev(const sps_prior* p, PriorDev& out);

// exact path (sps_exact.cu)
sps_status sps_exact_setup(sps_table* t, int precision);
void sps_exact_teardown(sps_table* t);
// flux + (optional) reverse pass over the SSP table for rows whose prologue has run:
// fills B.flux, B.sc[*].logp_like and, if want_grad, B.a_bar, B.m_bar and the scalar bars.
sps_status sps_exact_contract(sps_table* t, int64_t n, const int* rows, const int* gal_of_row, const float* obs_flux,
                              const float* obs_sigma, const float* flux_bar, bool want_grad, cudaStream_t s);

// tensor-core approximate contraction (sps_approx_tc.cu); same contract as launch_approx_contract
sps_status sps_approx_tc_setup(sps_table* t);
void sps_approx_tc_teardown(sps_table* t);
bool sps_approx_tc_active(const sps_table* t);
sps_status sps_approx_tc_contract(sps_table* t, int64_t n, const int* rows, const int* gal_of_row, const float* obs_flux,
                                  const float* obs_sigma, const float* flux_bar, bool want_grad, cudaStream_t s);

// full model evaluation used by the API and the sampler (sps_api.cu)
sps_status sps_eval(sps_table* t, const PriorDev& P, int path, const float* theta, int64_t n, bool unbounded,
                    bool with_prior, const int* rows, const int* gal_of_row, const float* obs_flux,
                    const float* obs_sigma, const float* flux_bar, bool want_grad, float* logp, float* grad,
                    cudaStream_t s, const LeapfrogFuse* lf = nullptr);
