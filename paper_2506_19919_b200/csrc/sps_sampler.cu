// sps_sampler.cu -- counter-based RNG, leapfrog, fixed-length HMC with windowed warmup (a11, a12).
// One warp owns one chain (lane p < 13 owns parameter p); the model evaluation between the
// sampler kernels is the batch-wide prologue / contraction / epilogue pipeline (sps_eval).
// NUTS lives in sps_nuts.cu and reuses the state and helpers declared in sps_sampler.cuh.
#include <algorithm>
#include <cmath>
#include <vector>
#include "sps_sampler.cuh"

// ---------------------------------------------------------------------------------------------
__global__ void philox_words_kernel(uint32_t k0, uint32_t k1, uint32_t first_chain, uint32_t transition, uint32_t purpose,
                                    uint32_t index, int64_t n, uint32_t* out) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  reinterpret_cast<uint4*>(out)[i] = philox4x32_10(make_uint4(first_chain + (uint32_t)i, transition, purpose, index), make_uint2(k0, k1));
}

extern "C" sps_status sps_philox_words(uint64_t seed, uint32_t first_chain, uint32_t transition, uint32_t purpose,
                                       uint32_t index, int64_t n, uint32_t* out, void* stream) {
  if (!out || n < 0) { sps_set_error("sps_philox_words: bad argument"); return SPS_EINVAL; }
  if (n == 0) return SPS_OK;
  sps_status st = sps_require_device(); if (st != SPS_OK) return st;
  philox_words_kernel<<<(unsigned)((n + 255) / 256), 256, 0, (cudaStream_t)stream>>>((uint32_t)seed, (uint32_t)(seed >> 32), first_chain,
                                                                                 transition, purpose, index, n, out);
  sps_count_launch();
  return sps_check_cuda(cudaGetLastError(), "philox launch");
}

// ---------------------------------------------------------------------------------------------
// chain initialisation (R17): theta~_0 = xi + 0.1 omega N(0,1) from (chain, transition 0, purpose 5)
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) chain_init_kernel(ChainState C, PriorDev P, const float* __restrict__ theta0, float eps0, const float* __restrict__ eps_in,
                                                         const float* __restrict__ inv_mass_in, uint2 key) {
  CHAIN_WARP_PROLOGUE(C.n);
  if (l < SPS_NDIM) {
    float v;
    if (theta0) v = theta0[c * SPS_NDIM + l];
    else v = P.xi[l] + (l < C.D ? 0.1f * P.omega[l] * chain_normal(key, (uint32_t)C.rng_id[c], 0u, RNG_INIT, l) : 0.f);   // unsampled slots: xi exactly
    C.theta[c * SPS_NDIM + l] = v;
    C.inv_mass[c * SPS_NDIM + l] = inv_mass_in ? inv_mass_in[c * SPS_NDIM + l] : 1.f;
    C.w_mean[c * SPS_NDIM + l] = 0.f; C.w_m2[c * SPS_NDIM + l] = 0.f;
    C.s_mean[c * SPS_NDIM + l] = 0.f; C.s_m2[c * SPS_NDIM + l] = 0.f;
    C.bm_sum[c * SPS_NDIM + l] = 0.f; C.bm_mean[c * SPS_NDIM + l] = 0.f; C.bm_m2[c * SPS_NDIM + l] = 0.f;
  }
  if (l == 0) {
    const float e0 = eps_in ? eps_in[c] : eps0;
    C.eps[c] = e0; C.da_mu[c] = logf(10.f * e0); C.da_hbar[c] = 0.f; C.da_logepsbar[c] = 0.f; C.da_m[c] = 0;
    C.acc_sum[c] = 0.f; C.n_leapfrog[c] = 0; C.n_div[c] = 0;
  }
}

// ---------------------------------------------------------------------------------------------
// HMC transition (R-step 13).  Draw order: 13 normals (purpose 0), one uniform (purpose 1).
// begin: p = N / sqrt(invM); H0 = -logP + 1/2 sum invM p^2; first half kick and drift.
// ---------------------------------------------------------------------------------------------
__global__ void hmc_ctl_kernel(HmcCtl* ctl, WarmupSched W) {      // next transition: counter and adaptation flags
  const int it = ctl->it + 1;
  ctl->it = it; ctl->sample_index = it - W.n_warmup; ctl->A = adapt_flags_dev(it, W);
}

__global__ void __launch_bounds__(256) hmc_begin_kernel(ChainState C, const HmcCtl* __restrict__ ctl, uint32_t first, uint2 key) {
  CHAIN_WARP_PROLOGUE(C.n);
  const uint32_t transition = (uint32_t)ctl->it + first;
  float kin = 0.f;
  if (l < SPS_NDIM) {
    const int64_t o = c * SPS_NDIM + l;
    const float v = C.inv_mass[o], eps = C.eps[c];
    float p = l < C.D ? chain_normal(key, (uint32_t)C.rng_id[c], transition, RNG_MOMENTUM, l) * rsqrtf(v) : 0.f;
    kin = 0.5f * v * p * p;
    p += 0.5f * eps * C.grad[o];
    C.p_w[o] = p;
    C.theta_w[o] = C.theta[o] + eps * v * p;
  }
  kin = warp_sum(kin);
  if (l == 0) C.H0[c] = -C.logp[c] + kin;
}

// (between two gradient evaluations the update p += eps grad; theta~ += eps invM p rides in the epilogue kernel: LeapfrogFuse)

// end: last half kick, Metropolis test, warmup adaptation (R14), running summaries.
__global__ void __launch_bounds__(256) hmc_end_kernel(ChainState C, const HmcCtl* __restrict__ ctl, uint32_t first, uint2 key, int n_leapfrog,
                                                      float* __restrict__ samples, int n_sample, int bm_len, int bm_n) {
  CHAIN_WARP_PROLOGUE(C.n);
  const uint32_t transition = (uint32_t)ctl->it + first;
  const AdaptFlags A = ctl->A;
  const int sample_index = ctl->sample_index;
  const int64_t o = c * SPS_NDIM + (l < SPS_NDIM ? l : 0);
  const bool act = l < SPS_NDIM;
  const float v = C.inv_mass[o], eps = C.eps[c];
  const float gw = C.grad_w[o], thw = C.theta_w[o];
  const float p = C.p_w[o] + 0.5f * eps * gw;
  const float kin = warp_sum(act ? 0.5f * v * p * p : 0.f);
  const float lpw = C.logp_w[c];
  const float dH = (-lpw + kin) - C.H0[c];
  const bool fin = __all_sync(FULL_MASK, !act || (isfinite(gw) && isfinite(thw))) && isfinite(dH);
  const float acc_prob = fin ? fminf(1.f, expf(fminf(0.f, -dH))) : 0.f;
  const float u = philox_u01(philox4x32_10(make_uint4((uint32_t)C.rng_id[c], transition, RNG_ACCEPT, 0u), key).x);
  const bool accept = fin && (u < acc_prob);
  float th = C.theta[o];
  if (accept) {
    th = thw;
    if (act) { C.theta[o] = thw; C.grad[o] = gw; }
    if (l == 0) C.logp[c] = lpw;
  }
  chain_adapt_and_record(C, c, l, act, o, th, acc_prob, n_leapfrog, 0, A, samples, sample_index, n_sample, bm_len, bm_n);
}

// ---------------------------------------------------------------------------------------------
// finalisation: mean / sd per chain, Gelman-Rubin R-hat per galaxy
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) finalize_kernel(ChainState C, int n_chain, int n_sample, int bm_len, int bm_n, sps_hmc_summary S) {
  const int64_t gidx = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  const int l = threadIdx.x & 31;
  const int64_t n_gal = C.n / n_chain;
  if (gidx >= n_gal || l >= SPS_NDIM) return;
  float mean_of_means = 0.f, W = 0.f, tau2 = 0.f;
  for (int k = 0; k < n_chain; ++k) {
    const int64_t c = gidx * n_chain + k, o = c * SPS_NDIM + l;
    const float mu = C.s_mean[o], var = n_sample > 1 ? C.s_m2[o] / (float)(n_sample - 1) : 0.f;
    if (S.mean) S.mean[o] = mu;
    if (S.sd) S.sd[o] = sqrtf(var);
    if (S.inv_mass) S.inv_mass[o] = C.inv_mass[o];
    if (S.theta_last) S.theta_last[o] = C.theta[o];
    if (l == 0) {
      if (S.accept) S.accept[c] = C.acc_sum[c] / (float)max(n_sample, 1);
      if (S.eps) S.eps[c] = C.eps[c];
      if (S.n_leapfrog) S.n_leapfrog[c] = C.n_leapfrog[c];
      if (S.divergences) S.divergences[c] = C.n_div[c];
    }
    mean_of_means += mu; W += var;
    tau2 += bm_n > 1 ? (float)bm_len * C.bm_m2[o] / (float)(bm_n - 1) : 0.f;
  }
  // ESS by batch means pooled over the galaxy's chains (R25): m n mean(s2_c) / mean(tau2_c)
  if (S.ess) S.ess[gidx * SPS_NDIM + l] = tau2 > 0.f ? (float)n_chain * (float)n_sample * W / tau2 : 0.f;
  mean_of_means /= n_chain; W /= n_chain;
  float Bn = 0.f;                                   // B/n: variance of the chain means
  for (int k = 0; k < n_chain; ++k) { const float d = C.s_mean[(gidx * n_chain + k) * SPS_NDIM + l] - mean_of_means; Bn += d * d; }
  Bn = n_chain > 1 ? Bn / (float)(n_chain - 1) : 0.f;
  if (S.rhat) {
    const float ns = (float)n_sample;
    S.rhat[gidx * SPS_NDIM + l] = (W > 0.f && n_chain > 1) ? sqrtf(((ns - 1.f) / ns * W + Bn) / W) : 1.f;
  }
}

// ---------------------------------------------------------------------------------------------
// host side
// ---------------------------------------------------------------------------------------------
sps_status chain_state_alloc(ChainState& C, int64_t n, int ckpt_vectors) {
  memset(&C, 0, sizeof(C));
  C.n = n;
  const size_t nv = 13 + (size_t)ckpt_vectors;      // vectors of 13 floats per chain
  const size_t ns = 17;                             // scalars per chain
  const size_t bytes = n * (nv * SPS_NDIM + ns) * sizeof(float);
  float* base = nullptr;
  sps_status st = sps_check_cuda(sps_pool_alloc((void**)&base, bytes), "chain state allocation");
  if (st != SPS_OK) return st;
  cudaMemset(base, 0, bytes);
  C.base = base;
  float* p = base;
  auto vec = [&]() { float* r = p; p += n * SPS_NDIM; return r; };
  auto sca = [&]() { float* r = p; p += n; return r; };
  C.theta = vec(); C.grad = vec(); C.theta_w = vec(); C.p_w = vec(); C.grad_w = vec(); C.inv_mass = vec();
  C.w_mean = vec(); C.w_m2 = vec(); C.s_mean = vec(); C.s_m2 = vec(); C.bm_sum = vec(); C.bm_mean = vec(); C.bm_m2 = vec();
  C.nuts = p; p += n * (size_t)ckpt_vectors * SPS_NDIM;
  C.logp = sca(); C.logp_w = sca(); C.H0 = sca(); C.eps = sca(); C.da_mu = sca(); C.da_hbar = sca(); C.da_logepsbar = sca();
  C.acc_sum = sca();
  C.da_m = (int*)sca(); C.n_leapfrog = (int*)sca(); C.n_div = (int*)sca();
  C.rng_id = (int*)sca();
  C.nuts_sc = sca();   // 5 scalars left for NUTS
  return SPS_OK;
}
void chain_state_free(ChainState& C) { if (C.base) sps_pool_free(C.base); C.base = nullptr; }

// R14 windows (restated): <20 warmup steps: step size only.  >=150: 75 | 25,50,100,... | 50; else 15% | one window | 10%.
void warmup_schedule(int W, std::vector<int>& ends, int& slow_lo, int& slow_hi) {
  ends.clear();
  if (W < 20) { slow_lo = slow_hi = W; return; }
  int init, term, base;
  if (W >= 150) { init = 75; term = 50; base = 25; }
  else { init = (int)(0.15 * W); term = (int)(0.1 * W); base = W - init - term; }
  int start = init, size = base; const int stop = W - term;
  while (start < stop) {
    int end = start + size;
    if (end + 2 * size > stop) end = stop;
    ends.push_back(end);
    start = end; size *= 2;
  }
  slow_lo = init; slow_hi = stop;
}

WarmupSched make_warmup_sched(const sps_hmc_config* cfg) {
  WarmupSched W; memset(&W, 0, sizeof(W));
  std::vector<int> ends; int lo, hi;
  warmup_schedule(cfg->n_warmup, ends, lo, hi);
  W.n_warmup = cfg->n_warmup; W.n_sample = cfg->n_sample; W.slow_lo = lo; W.slow_hi = hi; W.target = cfg->target_accept;
  W.first = (int)cfg->first_transition;
  W.bm_len = cfg->n_sample > 0 ? (int)std::floor(std::sqrt((double)cfg->n_sample)) : 0;       // R25: batch length floor(sqrt(n))
  while (W.bm_len > 0 && (int64_t)(W.bm_len + 1) * (W.bm_len + 1) <= cfg->n_sample) ++W.bm_len;    // (guard the rounding of sqrt)
  while (W.bm_len > 0 && (int64_t)W.bm_len * W.bm_len > cfg->n_sample) --W.bm_len;
  W.bm_n = W.bm_len > 0 ? cfg->n_sample / W.bm_len : 0;
  W.n_ends = (int)std::min<size_t>(ends.size(), 16);
  for (int k = 0; k < W.n_ends; ++k) W.ends[k] = ends[k];
  return W;
}

static inline unsigned chain_blocks(int64_t n) { return (unsigned)((n * 32 + 255) / 256); }

// One evaluation at the working points: all rows (group < 0) or the rows of one row group.
static sps_status eval_working(const sps_table* t, Workspace& ws, const PriorDev& P, const HmcProblem& Q, ChainState& C, cudaStream_t s,
                               bool fuse_leapfrog = false, int group = -1) {
  const LeapfrogFuse lf = {C.theta_w, C.p_w, C.eps, C.inv_mass};
  // rows per path: rows_path[0] exact, [1] approx (index lists) or all rows on one path
  sps_status st = SPS_OK;
  for (int path = 0; path < 2 && st == SPS_OK; ++path) {
    const int64_t cnt = group < 0 ? Q.n_rows_path[path] : Q.g_n[group][path];
    if (cnt == 0) continue;
    const int* rows = Q.rows_path[path] ? Q.rows_path[path] + (group < 0 ? 0 : Q.g_off[group][path]) : nullptr;
    st = sps_eval(t, ws, P, path, C.theta_w, cnt, true, true, rows, Q.gal_of_chain, Q.obs_flux,
                  Q.obs_sigma, nullptr, true, C.logp_w, C.grad_w, s, fuse_leapfrog ? &lf : nullptr, group >= 0 && Q.n_groups > 1);
  }
  return st;
}

sps_status hmc_problem_setup(HmcProblem& Q, const sps_hmc_config* cfg, int64_t n_gal, const int32_t* path_of_gal_dev,
                             const float* obs_flux, const float* obs_sigma, int n_groups);
void hmc_problem_free(HmcProblem& Q);
sps_status nuts_run(const sps_table* t, Workspace& ws, const PriorDev& P, const sps_hmc_config* cfg, HmcProblem& Q, ChainState& C, float* samples,
                    int32_t* depth_hist_out, cudaStream_t s);

extern "C" sps_status sps_hmc_run(const sps_table* t, const sps_prior* prior, const sps_hmc_config* cfg, const float* obs_flux,
                                  const float* obs_sigma, int64_t n_gal, const int32_t* path_of_gal, const float* theta0,
                                  float* samples, const sps_hmc_summary* summary, void* stream) {
  if (!t || !cfg) { sps_set_error("sps_hmc_run: null argument"); return SPS_EINVAL; }
  const bool gauss = t->dev.model == SPS_MODEL_GAUSS_TEST;
  if (!gauss && (!prior || !obs_flux || !obs_sigma)) { sps_set_error("sps_hmc_run: null argument"); return SPS_EINVAL; }
  if (n_gal < 0 || cfg->n_chain < 1 || cfg->n_warmup < 0 || cfg->n_sample < 0 || !(cfg->eps0 > 0)) { sps_set_error("sps_hmc_run: bad config"); return SPS_EINVAL; }
  if (cfg->sampler == SPS_SAMPLER_HMC && cfg->n_leapfrog < 1) { sps_set_error("sps_hmc_run: n_leapfrog < 1"); return SPS_EINVAL; }
  if (cfg->sampler == SPS_SAMPLER_NUTS && (cfg->max_depth < 1 || cfg->max_depth > 10)) { sps_set_error("sps_hmc_run: max_depth must be 1..10"); return SPS_EINVAL; }
  if (cfg->sampler != SPS_SAMPLER_HMC && cfg->sampler != SPS_SAMPLER_NUTS) { sps_set_error("sps_hmc_run: bad sampler"); return SPS_EINVAL; }
  if (n_gal == 0) return SPS_OK;
  sps_status st = sps_require_device(); if (st != SPS_OK) return st;
  cudaStream_t s = (cudaStream_t)stream;
  if (!s) {
    // The legacy default stream cannot be captured into a graph: the run (which synchronises before returning anyway)
    // goes on a stream the table owns, after everything already queued on the caller's stream.
    std::lock_guard<std::mutex> lock(t->mu);
    if (!t->own_stream && cudaStreamCreateWithFlags(&t->own_stream, cudaStreamNonBlocking) != cudaSuccess) { t->own_stream = nullptr; cudaGetLastError(); }
    if (t->own_stream) { cudaStreamSynchronize(nullptr); s = t->own_stream; }
  }
  PriorDev P; st = sps_prior_to_dev(t, prior, P); if (st != SPS_OK) return st;
  const int64_t n = n_gal * cfg->n_chain;
  if (!gauss) { st = sps_check_finite(obs_flux, n_gal * t->dev.n_band, theta0, theta0 ? n * SPS_NDIM : 0, obs_sigma, n_gal * t->dev.n_band, s); if (st != SPS_OK) return st; }
  Workspace& ws = *sps_workspace(t, s);
  if (!gauss) { st = sps_ensure_row_buffers(t, ws, n, s); if (st != SPS_OK) return st; }
  HmcProblem Q; ChainState C;
  memset(&C, 0, sizeof(C));
  // Row groups (fixed-length HMC, SPS_OPT_ROW_GROUPS; off by default): the chains are split into G groups whose leapfrog
  // evaluations run on G streams, meant to let the latency-bound contraction of one group share the SMs with the
  // issue-bound row kernels of another.  A chain's result does not depend on the grouping (its RNG streams and its
  // arithmetic are its own).  Measured at 40,000 chains: 188 us per evaluation as one group, 196 as two, 244 as
  // four: the block scheduler does not co-schedule the persistent contraction CTAs with the row kernels' blocks.
  int G = 1;
  if (cfg->sampler == SPS_SAMPLER_HMC && !gauss) {
    const int opt = sps_option(SPS_OPT_ROW_GROUPS);
    G = opt > 0 ? std::min(opt, 4) : 1;
  }
  cudaStream_t sg[4] = {s, nullptr, nullptr, nullptr};
  Workspace* wsg[4] = {&ws, nullptr, nullptr, nullptr};
  cudaEvent_t ev_fork = nullptr, ev_join[4] = {nullptr, nullptr, nullptr, nullptr};
  if (G > 1) {
    std::lock_guard<std::mutex> lock(t->mu);
    for (int g = 1; g < G; ++g)
      if (!t->aux_stream[g - 1] && cudaStreamCreateWithFlags(&t->aux_stream[g - 1], cudaStreamNonBlocking) != cudaSuccess) { cudaGetLastError(); G = 1; }
  }
  for (int g = 1; g < G && st == SPS_OK; ++g) {
    sg[g] = t->aux_stream[g - 1];
    wsg[g] = sps_workspace(t, sg[g]);
    st = sps_ensure_row_buffers(t, *wsg[g], n, sg[g]);
    cudaEventCreateWithFlags(&ev_join[g], cudaEventDisableTiming);
  }
  if (G > 1) cudaEventCreateWithFlags(&ev_fork, cudaEventDisableTiming);
  if (st != SPS_OK) return st;
  st = hmc_problem_setup(Q, cfg, n_gal, path_of_gal, obs_flux, obs_sigma, G);
  if (st == SPS_OK) st = chain_state_alloc(C, n, cfg->sampler == SPS_SAMPLER_NUTS ? NUTS_VECTORS : 0);
  if (st != SPS_OK) { hmc_problem_free(Q); chain_state_free(C); return st; }
  C.D = t->dev.n_dim;
  const WarmupSched W = make_warmup_sched(cfg);
  const uint2 key = make_uint2((uint32_t)cfg->seed, (uint32_t)(cfg->seed >> 32));
  cudaDeviceSynchronize();                                   // the set-up above ran on the default stream
  cudaMemcpyAsync(C.rng_id, Q.rng_id, n * sizeof(int), cudaMemcpyDeviceToDevice, s);
  chain_init_kernel<<<chain_blocks(n), 256, 0, s>>>(C, P, theta0, cfg->eps0, cfg->eps_in_dev, cfg->inv_mass_in_dev, key); sps_count_launch();
  // logp / grad at the start: evaluate through the working buffers
  cudaMemcpyAsync(C.theta_w, C.theta, n * SPS_NDIM * sizeof(float), cudaMemcpyDeviceToDevice, s);
  st = eval_working(t, ws, P, Q, C, s);
  cudaMemcpyAsync(C.grad, C.grad_w, n * SPS_NDIM * sizeof(float), cudaMemcpyDeviceToDevice, s);
  cudaMemcpyAsync(C.logp, C.logp_w, n * sizeof(float), cudaMemcpyDeviceToDevice, s);
  if (st == SPS_OK && cfg->sampler == SPS_SAMPLER_HMC) {
    // One transition = control update, momentum draw, n_leapfrog evaluations (each five launches), accept/adapt.  Every
    // launch argument is the same from one transition to the next (the counter lives in device memory), so the
    // sequence is captured once in a CUDA graph and replayed: small batches are launch-latency bound.
    // Plain launches are used when per-kernel profiling is on, with SPS_OPT_NO_GRAPH, or if capture fails.
    const int n_tr = cfg->n_warmup + cfg->n_sample;
    HmcCtl* ctl = nullptr;
    st = sps_check_cuda(sps_pool_alloc((void**)&ctl, sizeof(HmcCtl)), "HMC control block");
    if (st == SPS_OK) cudaMemsetAsync(ctl, 0xff, sizeof(int), s);          // it = -1
    auto enqueue_transition = [&]() -> sps_status {
      hmc_ctl_kernel<<<1, 1, 0, s>>>(ctl, W);
      hmc_begin_kernel<<<chain_blocks(n), 256, 0, s>>>(C, ctl, cfg->first_transition, key);
      sps_count_launch(2);
      sps_status e = SPS_OK;
      if (G == 1) {
        for (int k = 0; k < cfg->n_leapfrog && e == SPS_OK; ++k) e = eval_working(t, ws, P, Q, C, s, k + 1 < cfg->n_leapfrog);
      } else {
        cudaEventRecord(ev_fork, s);
        for (int g = 0; g < G; ++g) {
          if (g > 0) cudaStreamWaitEvent(sg[g], ev_fork, 0);
          for (int k = 0; k < cfg->n_leapfrog && e == SPS_OK; ++k) e = eval_working(t, *wsg[g], P, Q, C, sg[g], k + 1 < cfg->n_leapfrog, g);
          if (g > 0) { cudaEventRecord(ev_join[g], sg[g]); cudaStreamWaitEvent(s, ev_join[g], 0); }
        }
      }
      hmc_end_kernel<<<chain_blocks(n), 256, 0, s>>>(C, ctl, cfg->first_transition, key, cfg->n_leapfrog, samples, cfg->n_sample, W.bm_len, W.bm_n);
      sps_count_launch();
      return e;
    };
    cudaGraphExec_t exec = nullptr;
    int64_t per_graph = 0;
    if (st == SPS_OK && n_tr > 2 && s != nullptr && !sps_prof_enabled() && !sps_option(SPS_OPT_NO_GRAPH)) {
      const int64_t c0 = sps_launch_count();
      cudaGraph_t graph = nullptr;
      if (cudaStreamBeginCapture(s, cudaStreamCaptureModeRelaxed) == cudaSuccess) {
        const sps_status e = enqueue_transition();
        const cudaError_t ce = cudaStreamEndCapture(s, &graph);
        if (e == SPS_OK && ce == cudaSuccess && graph && cudaGraphInstantiate(&exec, graph, 0) != cudaSuccess) exec = nullptr;
        if (graph) cudaGraphDestroy(graph);
      }
      cudaGetLastError();
      per_graph = sps_launch_count() - c0;                                 // launches one replay stands for
      sps_count_launch(-(int)per_graph);                                   // (capturing launched nothing)
    }
    for (int it = 0; it < n_tr && st == SPS_OK; ++it) {
      if (exec) { st = sps_check_cuda(cudaGraphLaunch(exec, s), "HMC transition graph"); sps_count_launch((int)per_graph); }
      else st = enqueue_transition();
    }
    if (exec) { cudaStreamSynchronize(s); cudaGraphExecDestroy(exec); }
    if (ctl) { cudaStreamSynchronize(s); sps_pool_free(ctl); }
  } else if (st == SPS_OK) {
    st = nuts_run(t, ws, P, cfg, Q, C, samples, summary ? summary->depth_hist : nullptr, s);
  }
  if (st == SPS_OK && summary) {
    finalize_kernel<<<chain_blocks(n_gal), 256, 0, s>>>(C, cfg->n_chain, cfg->n_sample, W.bm_len, W.bm_n, *summary); sps_count_launch();
  }
  if (st == SPS_OK) st = sps_check_cuda(cudaStreamSynchronize(s), "sps_hmc_run");
  else cudaStreamSynchronize(s);
  chain_state_free(C); hmc_problem_free(Q);
  if (ev_fork) cudaEventDestroy(ev_fork);
  for (int g = 1; g < 4; ++g) if (ev_join[g]) cudaEventDestroy(ev_join[g]);
  return st;
}
