// sps_rows.cuh -- buffers exchanged between the per-row prologue / epilogue kernels (one warp per
// parameter row; shared by the exact and the approximate photometry paths) and the contraction kernels.
#pragma once
#include <utility>
#include "sps_model.cuh"

// Work buffers for n rows (device memory owned by the library, grown on demand).
#define ROW_PARTS 5
struct RowBuffers {
  float* a;        // [n][ROW_A_STRIDE]  P_SFH (Eq. A6)
  float* m;        // [n][ROW_M_STRIDE]  P_met
  float* a_bar;    // [n][ROW_A_STRIDE]  d logL / d a_i
  float* m_bar;    // [n][ROW_M_STRIDE]  d logL / d m_j
  RowScalars* sc;  // [n]
  float* flux;     // [n][SPS_MAX_BAND]  model band fluxes
  float* part;     // [n][ROW_PARTS][ROW_A_STRIDE] per-bin dM and its partials (tau, alpha, beta, t_obs), written by the
                   //                              gradient prologue and contracted with a_bar by the epilogue
  int* order;      // [n]  rows of the current approximate-path call grouped by z cell
  int* bins;       // [4][n_z + 1] histogram, row offsets, CTA offsets, cursors of that grouping
  int* cell_list;  // [n_z - 1][cell_cap] rows of every z cell, appended by the prologue (or null: scan / scatter pass instead)
  int64_t cell_cap;
  int64_t capacity;
};

// Optional leapfrog update fused into the epilogue (HMC inner steps): after the gradient of a row is known,
//   p += eps grad;  theta~ += eps invM p     (the two half kicks between consecutive evaluations merged)
struct LeapfrogFuse { float* theta_w; float* p_w; const float* eps; const float* inv_mass; };
// (sps_eval's `overlap` flag: the call is one of several row groups running on different streams, see sps_sampler.cu)

// Launch with the programmatic-stream-serialisation attribute (see pdl_wait in sps_common.cuh) unless SPS_OPT_NO_PDL is set
// or the per-kernel profiling hooks are on (their events sit between the kernels anyway).
int sps_option(int option);
template <class... KA, class... A>
inline cudaError_t sps_launch(void (*kernel)(KA...), dim3 grid, dim3 block, size_t smem, cudaStream_t s, A&&... args) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = s;
  cudaLaunchAttribute at = {};
  at.id = cudaLaunchAttributeProgrammaticStreamSerialization;
  at.val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = &at;
  cfg.numAttrs = (sps_option(6 /* SPS_OPT_NO_PDL */) || sps_prof_enabled()) ? 0 : 1;
  return cudaLaunchKernelEx(&cfg, kernel, std::forward<A>(args)...);
}

// kernels (sps_kernels.cu)
void launch_prologue(const TableDev& T, const PriorDev& P, const float* theta, int64_t n, bool unbounded, bool want_grad,
                     const int* rows, RowBuffers B, bool with_hist, cudaStream_t s, bool small_blocks = false, bool zero_bins = true);
void launch_approx_contract(const TableDev& T, int sm_count, int64_t n, const int* rows, const int* gal_of_row,
                            const float* obs_flux, const float* obs_sigma, const float* flux_bar,
                            bool want_grad, RowBuffers B, cudaStream_t s);
sps_status approx_contract_setup(const TableDev& T);
void approx_group_rows(const TableDev& T, int64_t n, const int* rows, RowBuffers B, int rows_per_item, cudaStream_t s);
void launch_epilogue(const TableDev& T, const PriorDev& P, const float* theta, int64_t n, bool unbounded,
                     bool with_prior, const int* rows, RowBuffers B, float* logp, float* grad, LeapfrogFuse lf, cudaStream_t s);
void launch_copy_weights(const TableDev& T, int64_t n, RowBuffers B, float* w_age, float* w_met, float* mstar,
                         cudaStream_t s);
void launch_copy_flux(const TableDev& T, int64_t n, RowBuffers B, float* flux, cudaStream_t s);
