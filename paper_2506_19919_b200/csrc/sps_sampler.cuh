// sps_sampler.cuh -- chain state and device helpers shared by the HMC and NUTS engines.
#pragma once
#include <cstring>
#include "sps_internal.h"
#include "sps_philox.cuh"

// vectors of 13 floats per chain that NUTS needs on top of the common state (see sps_nuts.cu)
#define NUTS_MAX_DEPTH 10
#define NUTS_VECTORS (13 + 2 * (NUTS_MAX_DEPTH + 1))

struct ChainState {
  int64_t n;
  int D;                               // sampled parameters of the table's model: lanes p >= D carry no momentum
  float* base;
  // [n,13]
  float *theta, *grad;                 // current state and gradient of logP there
  float *theta_w, *p_w, *grad_w;       // trajectory working point
  float *inv_mass;                     // diagonal inverse mass
  float *w_mean, *w_m2;                // Welford over the current slow window (warmup)
  float *s_mean, *s_m2;                // Welford over kept samples
  float *bm_sum, *bm_mean, *bm_m2;     // batch means of the kept samples (ESS, R25): running batch sum, Welford over batch means
  float *nuts;                         // [n, NUTS_VECTORS, 13] (NUTS only)
  // [n]
  float *logp, *logp_w, *H0, *eps, *da_mu, *da_hbar, *da_logepsbar, *acc_sum, *nuts_sc;
  int *da_m, *n_leapfrog, *n_div;
  int *rng_id;                         // [n] Philox stream of each chain (gal_id * n_chain + chain)
};

struct AdaptFlags { int warmup, in_window, window_end, last_warmup, welford_n; float target; };

// Warmup windows (R14) in a form kernels can evaluate: slow windows end at ends[0..n_ends) inside [slow_lo, slow_hi).
// `first` = transition index of the RNG streams at local transition 0 (continued runs).
struct WarmupSched { int n_warmup, n_sample, slow_lo, slow_hi, n_ends; int ends[16]; float target; int first; int bm_len, bm_n; };

__device__ __forceinline__ AdaptFlags adapt_flags_dev(int it, const WarmupSched& S) {
  AdaptFlags A; A.warmup = it < S.n_warmup; A.in_window = 0; A.window_end = 0; A.last_warmup = (it + 1 == S.n_warmup); A.welford_n = 0;
  A.target = S.target;
  if (A.warmup && it >= S.slow_lo && it < S.slow_hi) {
    A.in_window = 1;
    int start = S.slow_lo;
    for (int k = 0; k < S.n_ends; ++k) {
      const int e = S.ends[k];
      if (it < e) { A.welford_n = it - start + 1; A.window_end = (it + 1 == e); break; }
      start = e;
    }
  }
  return A;
}

// Per-run control block in device memory: the transition counter and its adaptation flags are advanced on the device,
// so that one HMC transition is a self-contained sequence of launches (capturable in a CUDA graph and replayed).
struct HmcCtl { int it; int sample_index; AdaptFlags A; };

WarmupSched make_warmup_sched(const sps_hmc_config* cfg);            // sps_sampler.cu

struct HmcProblem {
  int64_t n;                 // chains
  int* rng_id;               // [n] device: Philox stream of each chain
  int* gal_of_chain;         // [n] device
  unsigned char* path_of_chain;   // [n] device: photometry path of each chain
  int* rows_path[2];         // device index lists per path, or NULL = all rows
  int64_t n_rows_path[2];
  // row groups of fixed-length HMC (SPS_OPT_ROW_GROUPS): group g evaluates rows_path[p][g_off[g][p] .. + g_n[g][p]) of each path
  int n_groups;
  int64_t g_off[4][2], g_n[4][2];
  const float *obs_flux, *obs_sigma;
};

#define CHAIN_WARP_PROLOGUE(N)                                                         \
  const int64_t c = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;             \
  const int l = threadIdx.x & 31;                                                      \
  if (c >= (N)) return;

// the idx-th standard normal of stream (chain, transition, purpose): block idx/4, component idx%4
__device__ __forceinline__ float chain_normal(uint2 key, uint32_t chain, uint32_t transition, uint32_t purpose, int idx) {
  const float4 z = philox_normal4(make_uint4(chain, transition, purpose, (uint32_t)(idx >> 2)), key);
  const int k = idx & 3;
  return k == 0 ? z.x : (k == 1 ? z.y : (k == 2 ? z.z : z.w));
}

// Warmup adaptation (R14: dual averaging gamma=0.05, t0=10, kappa=0.75; Welford diagonal mass with
// shrinkage) and running summaries; called by the whole warp at the end of every transition.
__device__ __forceinline__ void chain_adapt_and_record(ChainState& C, int64_t c, int l, bool act, int64_t o, float th,
                                                       float acc_stat, int n_lf, int diverged, const AdaptFlags& A,
                                                       float* __restrict__ samples, int sample_index, int n_sample, int bm_len, int bm_n) {
  if (l == 0) C.n_leapfrog[c] += n_lf;
  if (A.warmup) {
    float eps_new = 0.f;
    if (l == 0) {
      const int m = C.da_m[c] + 1;
      const float fm = (float)m;
      const float hbar = (1.f - 1.f / (fm + 10.f)) * C.da_hbar[c] + (A.target - acc_stat) / (fm + 10.f);
      const float log_eps = C.da_mu[c] - sqrtf(fm) / 0.05f * hbar;
      const float eta = powf(fm, -0.75f);
      const float leb = eta * log_eps + (1.f - eta) * C.da_logepsbar[c];
      eps_new = expf(log_eps);
      C.da_m[c] = m; C.da_hbar[c] = hbar; C.da_logepsbar[c] = leb;
      if (A.last_warmup) eps_new = expf(leb);
      C.eps[c] = eps_new;
    }
    if (A.in_window) {
      if (act) {
        const float nn = (float)A.welford_n;
        float mean = C.w_mean[o], m2 = C.w_m2[o];
        const float d = th - mean;
        mean += d / nn;
        m2 += d * (th - mean);
        if (A.window_end) {
          const float var = m2 / (nn - 1.f);
          C.inv_mass[o] = (nn / (nn + 5.f)) * var + 1e-3f * (5.f / (nn + 5.f));
          mean = 0.f; m2 = 0.f;
        }
        C.w_mean[o] = mean; C.w_m2[o] = m2;
      }
      if (A.window_end && l == 0 && !A.last_warmup) {       // restart dual averaging around the current step size
        C.da_mu[c] = logf(10.f * eps_new); C.da_hbar[c] = 0.f; C.da_logepsbar[c] = 0.f; C.da_m[c] = 0;
      }
    }
  } else {
    if (act) {
      const float k = (float)(sample_index + 1);
      float mean = C.s_mean[o], m2 = C.s_m2[o];
      const float d = th - mean;
      mean += d / k; m2 += d * (th - mean);
      C.s_mean[o] = mean; C.s_m2[o] = m2;
      if (samples) samples[(c * n_sample + sample_index) * SPS_NDIM + l] = th;
      // batch means for the ESS (R25): batches of bm_len consecutive kept samples, bm_n of them
      float bs = C.bm_sum[o] + th;
      const int k1 = sample_index + 1;
      if (bm_len > 0 && k1 % bm_len == 0 && k1 / bm_len <= bm_n) {
        const float cnt = (float)(k1 / bm_len), bmv = bs / (float)bm_len;
        float bmean = C.bm_mean[o], bm2 = C.bm_m2[o];
        const float db = bmv - bmean;
        bmean += db / cnt; bm2 += db * (bmv - bmean);
        C.bm_mean[o] = bmean; C.bm_m2[o] = bm2;
        bs = 0.f;
      }
      C.bm_sum[o] = bs;
    }
    if (l == 0) { C.acc_sum[c] += acc_stat; C.n_div[c] += diverged; }
  }
}

sps_status chain_state_alloc(ChainState& C, int64_t n, int ckpt_vectors);
void chain_state_free(ChainState& C);
