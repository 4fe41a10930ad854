// sps_leapfrog.cu -- sps_leapfrog (trajectory diagnostic) and the per-run problem
// description shared by the samplers.
#include <vector>
#include "sps_sampler.cuh"

__global__ void gal_of_chain_kernel(int* out, int* rng_id, const int* __restrict__ gal_id, int64_t n, int n_chain) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const int g = (int)(i / n_chain), k = (int)(i - (int64_t)g * n_chain);
  out[i] = g;
  rng_id[i] = (gal_id ? gal_id[g] : g) * n_chain + k;        // Philox stream of the chain (sps_hmc_config.gal_id_dev)
}

static sps_status hmc_problem_fill(HmcProblem& Q, const sps_hmc_config* cfg, int64_t n_gal, const int32_t* path_of_gal_dev) {
  sps_status st = sps_check_cuda(sps_pool_alloc((void**)&Q.gal_of_chain, Q.n * sizeof(int)), "gal_of_chain allocation");
  if (st == SPS_OK) st = sps_check_cuda(sps_pool_alloc((void**)&Q.rng_id, Q.n * sizeof(int)), "rng_id allocation");
  if (st != SPS_OK) return st;
  gal_of_chain_kernel<<<(unsigned)((Q.n + 255) / 256), 256>>>(Q.gal_of_chain, Q.rng_id, cfg->gal_id_dev, Q.n, cfg->n_chain); sps_count_launch();
  st = sps_check_cuda(sps_pool_alloc((void**)&Q.path_of_chain, Q.n), "path_of_chain allocation");
  if (st != SPS_OK) return st;
  if (!path_of_gal_dev) {
    if (cfg->path != SPS_PATH_EXACT && cfg->path != SPS_PATH_APPROX) { sps_set_error("bad path"); return SPS_EINVAL; }
    Q.n_rows_path[cfg->path] = Q.n;
    cudaMemset(Q.path_of_chain, cfg->path, Q.n);
    if (Q.n_groups > 1) {                                     // row groups need an explicit (identity) list to offset into
      std::vector<int> ident(Q.n);
      for (int64_t i = 0; i < Q.n; ++i) ident[i] = (int)i;
      st = sps_check_cuda(sps_pool_alloc((void**)&Q.rows_path[cfg->path], Q.n * sizeof(int)), "row list allocation");
      if (st != SPS_OK) return st;
      cudaMemcpy(Q.rows_path[cfg->path], ident.data(), Q.n * sizeof(int), cudaMemcpyHostToDevice);
    }
    return SPS_OK;
  }
  std::vector<int32_t> pg(n_gal);
  st = sps_check_cuda(cudaMemcpy(pg.data(), path_of_gal_dev, n_gal * sizeof(int32_t), cudaMemcpyDeviceToHost), "path_of_gal D2H");
  if (st != SPS_OK) return st;
  std::vector<int> rows[2];
  std::vector<unsigned char> pc(Q.n);
  for (int64_t g = 0; g < n_gal; ++g) {
    if (pg[g] != 0 && pg[g] != 1) { sps_set_error("path_of_gal[%lld] = %d is not 0/1", (long long)g, pg[g]); return SPS_EINVAL; }
    for (int k = 0; k < cfg->n_chain; ++k) { rows[pg[g]].push_back((int)(g * cfg->n_chain + k)); pc[g * cfg->n_chain + k] = (unsigned char)pg[g]; }
  }
  cudaMemcpy(Q.path_of_chain, pc.data(), Q.n, cudaMemcpyHostToDevice);
  for (int p = 0; p < 2; ++p) {
    Q.n_rows_path[p] = (int64_t)rows[p].size();
    if (rows[p].empty()) continue;
    st = sps_check_cuda(sps_pool_alloc((void**)&Q.rows_path[p], rows[p].size() * sizeof(int)), "row list allocation");
    if (st != SPS_OK) return st;
    cudaMemcpy(Q.rows_path[p], rows[p].data(), rows[p].size() * sizeof(int), cudaMemcpyHostToDevice);
  }
  return SPS_OK;
}

void hmc_problem_free(HmcProblem& Q);
sps_status hmc_problem_setup(HmcProblem& Q, const sps_hmc_config* cfg, int64_t n_gal, const int32_t* path_of_gal_dev,
                             const float* obs_flux, const float* obs_sigma, int n_groups) {
  memset(&Q, 0, sizeof(Q));
  Q.n = n_gal * cfg->n_chain; Q.obs_flux = obs_flux; Q.obs_sigma = obs_sigma; Q.n_groups = n_groups;
  const sps_status st = hmc_problem_fill(Q, cfg, n_gal, path_of_gal_dev);
  if (st != SPS_OK) { hmc_problem_free(Q); return st; }     // nothing allocated here outlives a rejected call
  for (int p = 0; p < 2; ++p)                               // contiguous, balanced shares of each path's rows
    for (int g = 0; g < n_groups; ++g) {
      const int64_t a = Q.n_rows_path[p] * g / n_groups, b = Q.n_rows_path[p] * (g + 1) / n_groups;
      Q.g_off[g][p] = a; Q.g_n[g][p] = b - a;
    }
  return SPS_OK;
}

void hmc_problem_free(HmcProblem& Q) {
  if (Q.gal_of_chain) sps_pool_free(Q.gal_of_chain);
  if (Q.rng_id) sps_pool_free(Q.rng_id);
  if (Q.path_of_chain) sps_pool_free(Q.path_of_chain);
  for (int p = 0; p < 2; ++p) if (Q.rows_path[p]) sps_pool_free(Q.rows_path[p]);
  memset(&Q, 0, sizeof(Q));
}

// first half kick + drift from (theta0, p0) with the gradient at theta0
__global__ void lf_first_kernel(int64_t n, const float* __restrict__ theta0, const float* __restrict__ p0, const float* __restrict__ grad0,
                                const float* __restrict__ eps, const float* __restrict__ inv_mass, float* theta_w, float* p_w) {
  const int64_t o = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (o >= n * SPS_NDIM) return;
  const float e = eps[o / SPS_NDIM];
  const float p = p0[o] + 0.5f * e * grad0[o];
  p_w[o] = p;
  theta_w[o] = theta0[o] + e * inv_mass[o] * p;
}
// finish step k (half kick), record, and start step k+1 (half kick + drift)
__global__ void lf_record_kernel(int64_t n, int step, const float* __restrict__ grad_w, const float* __restrict__ logp_w,
                                 const float* __restrict__ eps, const float* __restrict__ inv_mass, float* theta_w, float* p_w,
                                 float* __restrict__ traj, float* __restrict__ logp_traj) {
  const int64_t o = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (o >= n * SPS_NDIM) return;
  const int64_t r = o / SPS_NDIM; const int d = (int)(o % SPS_NDIM);
  const float e = eps[r];
  float p = p_w[o] + 0.5f * e * grad_w[o];
  const float th = theta_w[o];
  traj[(((int64_t)step * n + r) * 2 + 0) * SPS_NDIM + d] = th;
  traj[(((int64_t)step * n + r) * 2 + 1) * SPS_NDIM + d] = p;
  if (d == 0) logp_traj[(int64_t)step * n + r] = logp_w[r];
  p += 0.5f * e * grad_w[o];
  p_w[o] = p;
  theta_w[o] = th + e * inv_mass[o] * p;
}

extern "C" sps_status sps_leapfrog(const sps_table* t, const sps_prior* prior, int path, const float* theta0, const float* p0,
                                   const float* eps, const float* inv_mass, int64_t n, const int32_t* gal_of_row,
                                   const float* obs_flux, const float* obs_sigma, int32_t n_steps, float* traj, float* logp_traj,
                                   void* stream) {
  if (!t || !theta0 || !p0 || !eps || !inv_mass || !traj || !logp_traj ||
      (t->dev.model != SPS_MODEL_GAUSS_TEST && (!prior || !obs_flux || !obs_sigma))) {
    sps_set_error("sps_leapfrog: null argument"); return SPS_EINVAL; }
  if (n < 0 || n_steps < 0 || (path != SPS_PATH_EXACT && path != SPS_PATH_APPROX)) { sps_set_error("sps_leapfrog: bad argument"); return SPS_EINVAL; }
  if (n == 0 || n_steps == 0) return SPS_OK;
  sps_status st = sps_require_device(); if (st != SPS_OK) return st;
  cudaStream_t s = (cudaStream_t)stream;
  PriorDev P; st = sps_prior_to_dev(t, prior, P); if (st != SPS_OK) return st;
  st = sps_check_finite(theta0, n * SPS_NDIM, p0, n * SPS_NDIM, eps, n, s); if (st != SPS_OK) return st;
  Workspace& ws = *sps_workspace(t, s);
  if (t->dev.model != SPS_MODEL_GAUSS_TEST) { st = sps_ensure_row_buffers(t, ws, n, s); if (st != SPS_OK) return st; }
  float* w = nullptr;
  const size_t nv = (size_t)n * SPS_NDIM;
  st = sps_check_cuda(sps_pool_alloc((void**)&w, (3 * nv + n) * sizeof(float)), "sps_leapfrog scratch"); if (st != SPS_OK) return st;
  float *theta_w = w, *p_w = w + nv, *grad_w = w + 2 * nv, *logp_w = w + 3 * nv;
  const unsigned eb = (unsigned)((nv + 255) / 256);
  st = sps_eval(t, ws, P, path, theta0, n, true, true, nullptr, gal_of_row, obs_flux, obs_sigma, nullptr, true, logp_w, grad_w, s);
  if (st == SPS_OK) { lf_first_kernel<<<eb, 256, 0, s>>>(n, theta0, p0, grad_w, eps, inv_mass, theta_w, p_w); sps_count_launch(); }
  for (int k = 0; k < n_steps && st == SPS_OK; ++k) {
    st = sps_eval(t, ws, P, path, theta_w, n, true, true, nullptr, gal_of_row, obs_flux, obs_sigma, nullptr, true, logp_w, grad_w, s);
    if (st == SPS_OK) { lf_record_kernel<<<eb, 256, 0, s>>>(n, k, grad_w, logp_w, eps, inv_mass, theta_w, p_w, traj, logp_traj); sps_count_launch(); }
  }
  cudaStreamSynchronize(s);
  sps_pool_free(w);
  return st == SPS_OK ? sps_check_cuda(cudaGetLastError(), "sps_leapfrog") : st;
}
