// sps_models.cu -- the models besides the paper's 13-parameter one:
//   SPS_MODEL_TINY5      BASELINE.json configs[0] (R19): delayed-exponential SFH by its closed form, lognormal MDF of
//                        fixed scatter 0.2, power-law dust screen, redshift as data.  Row kernels only: the photometry
//                        contractions (Eq. 4, Eq. 6) are the ones of the 13-parameter model, fed through the same RowBuffers.
//   SPS_MODEL_GAUSS_TEST a correlated Gaussian target for the samplers (north_star: "HMC on a Gaussian target recovers its
//                        mean and variance").
// One warp per parameter row, as in sps_kernels.cu.
#include "sps_internal.h"

#define TINY5_SIGMA_LOGZ 0.2f
#define TINY5_DUST_SLOPE -0.7f
#define TINY5_AV_PER_TAUV 1.0857362047581296f        // 2.5 / ln 10: exp(-tau) = 10^(-0.4 A)  <=>  A = 1.0857 tau

// E(t) = (1 + t/tau) exp(-t/tau): the mass formed after cosmic time t is proportional to E(t) (SFR ~ (t/tau^2) e^{-t/tau},
// int t e^{-t/tau} dt = -tau (t + tau) e^{-t/tau}), and dE/dtau = (t/tau)^2 e^{-t/tau} / tau.  Double precision: the
// narrow young bins are differences of nearly equal values.
__device__ __forceinline__ void tiny5_E(double t, double inv_tau, double& E, double& dE_dtau) {
  const double x = t * inv_tau, e = exp(-x);
  E = (1.0 + x) * e; dE_dtau = x * x * e * inv_tau;
}

struct Tiny5Row { float th[4]; float z; double t_obs, tau, inv_tau, G_obs, dEo; };

__device__ __forceinline__ void tiny5_params(const TableDev& T, const PriorDev& P, const float* __restrict__ row, bool unbounded,
                                             Tiny5Row& R, float& v_lane, float& slope_lane) {
  const int l = lane_id();
  float v = 0.f, d = 1.f;
  if (l < 4) {
    v = row[l];
    if (unbounded) {                                         // Eq. (C1)
      const float s = 1.f / (1.f + expf(-P.k[l] * (v - P.x0[l]))), w = P.y_hi[l] - P.y_lo[l];
      v = P.y_lo[l] + w * s; d = w * P.k[l] * s * (1.f - s);
    }
  }
  v_lane = v; slope_lane = d;
#pragma unroll
  for (int p = 0; p < 4; ++p) R.th[p] = __shfl_sync(FULL_MASK, v, p);
  R.z = row[4];                                              // data, not a sampled parameter
  float dt_dz;
  cosmic_time(T, (double)R.z, R.t_obs, dt_dz);
  R.tau = exp10((double)R.th[1]); R.inv_tau = 1.0 / R.tau;
  double Eo;
  tiny5_E(R.t_obs, R.inv_tau, Eo, R.dEo);
  R.G_obs = 1.0 - Eo;
}

__global__ void __launch_bounds__(256) tiny5_prologue_kernel(TableDev T, PriorDev P, const float* __restrict__ theta, int64_t n, bool unbounded,
                                                             const int* __restrict__ rows, RowBuffers B, int* __restrict__ hist) {
  const int64_t r = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  if (r >= n) return;
  const int64_t row = rows ? rows[r] : r;
  const int l = lane_id();
  Tiny5Row R; float v_l, d_l;
  tiny5_params(T, P, theta + row * SPS_NDIM, unbounded, R, v_l, d_l);
  const double inv_G = 1.0 / R.G_obs;
#pragma unroll
  for (int q = 0; q < SPS_AGE_PER_LANE; ++q) {
    const int i = l + 32 * q;
    float a = 0.f;
    if (i < T.n_age) {
      const double t_hi = fmax(R.t_obs - T.A_edge_d[i], 0.0), t_lo = fmax(R.t_obs - T.A_edge_d[i + 1], 0.0);   // R5
      double E_hi, E_lo, d0, d1;
      tiny5_E(t_hi, R.inv_tau, E_hi, d0); tiny5_E(t_lo, R.inv_tau, E_lo, d1);
      a = (float)((E_lo - E_hi) * inv_G);
    }
    B.a[row * ROW_A_STRIDE + i] = a;
  }
  float m, dm_lz, dm_s;
  met_bin(T, R.th[2], TINY5_SIGMA_LOGZ, m, dm_lz, dm_s);
  if (l < ROW_M_STRIDE) B.m[row * ROW_M_STRIDE + l] = m;
  if (l == 0) {
    RowScalars sc;
    sc.Mn = exp2f((R.th[0] - T.log10_mass_unit) * 3.321928094887362f);      // the mass formed by t_obs is 10^logM_star
    float zi = floorf((R.z - T.z_min) * T.inv_dz);
    zi = fminf(fmaxf(zi, 0.f), (float)(T.n_z - 2));
    sc.z = R.z; sc.zbin = (int)zi; sc.zfrac = (R.z - (T.z_min + zi * T.dz)) * T.inv_dz;
    sc.AV = R.th[3] * TINY5_AV_PER_TAUV; sc.delta = TINY5_DUST_SLOPE; sc.Ffloor = 0.f;
    sc.logp_like = 0.f; sc.Mn_bar = sc.z_bar = sc.AV_bar = sc.delta_bar = sc.Ffloor_bar = 0.f;
    sc.Msum = (float)R.G_obs; sc.pad1 = sc.pad2 = 0.f;
    B.sc[row] = sc;
    if (hist) {
      const int pos = atomicAdd(&hist[sc.zbin], 1);
      if (B.cell_list) B.cell_list[(int64_t)sc.zbin * B.cell_cap + pos] = (int)row;
    }
  }
}

// Reverse of the TINY5 weights + skew-normal prior over the four sampled parameters (+ the fused leapfrog update).
__global__ void __launch_bounds__(256) tiny5_epilogue_kernel(TableDev T, PriorDev P, const float* theta, int64_t n, bool unbounded, bool with_prior,
                                                             const int* __restrict__ rows, RowBuffers B, float* __restrict__ logp,
                                                             float* __restrict__ grad, LeapfrogFuse lf) {
  const int64_t r = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  if (r >= n) return;
  const int64_t row = rows ? rows[r] : r;
  const int l = lane_id();
  const RowScalars sc = B.sc[row];
  float lp = 0.f, dlp = 0.f;
  if (with_prior && l < 4) log_skew_normal(theta[row * SPS_NDIM + l], P.xi[l], P.omega[l], P.skew[l], lp, dlp);
  lp = warp_sum(lp);
  if (!grad) { if (l == 0 && logp) logp[row] = sc.logp_like + lp; return; }
  float lf_eps = 0.f, lf_p = 0.f, lf_im = 0.f, lf_th = 0.f;
  if (lf.p_w && l < SPS_NDIM) {
    const int64_t o = row * SPS_NDIM + l;
    lf_eps = lf.eps[row]; lf_p = lf.p_w[o]; lf_im = lf.inv_mass[o]; lf_th = lf.theta_w[o];
  }
  Tiny5Row R; float v_l, d_l;
  tiny5_params(T, P, theta + row * SPS_NDIM, unbounded, R, v_l, d_l);
  // tau_bar = (1/G_obs) [ sum_i a_bar_i (dE_lo/dtau - dE_hi/dtau) + (sum_i a_bar_i a_i) dE_obs/dtau ]
  double s_d = 0.0, s_aa = 0.0;
  const double inv_G = 1.0 / R.G_obs;
#pragma unroll
  for (int q = 0; q < SPS_AGE_PER_LANE; ++q) {
    const int i = l + 32 * q;
    if (i < T.n_age) {
      const double ab = (double)B.a_bar[row * ROW_A_STRIDE + i];
      const double t_hi = fmax(R.t_obs - T.A_edge_d[i], 0.0), t_lo = fmax(R.t_obs - T.A_edge_d[i + 1], 0.0);
      double E_hi, E_lo, dE_hi, dE_lo;
      tiny5_E(t_hi, R.inv_tau, E_hi, dE_hi); tiny5_E(t_lo, R.inv_tau, E_lo, dE_lo);
      s_d += ab * (dE_lo - dE_hi);
      s_aa += ab * (E_lo - E_hi) * inv_G;
    }
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) { s_d += __shfl_xor_sync(FULL_MASK, s_d, o); s_aa += __shfl_xor_sync(FULL_MASK, s_aa, o); }
  const float tau_bar = (float)((s_d + s_aa * R.dEo) * inv_G);
  float m_unused, dm_lz, dm_s;
  met_bin(T, R.th[2], TINY5_SIGMA_LOGZ, m_unused, dm_lz, dm_s);
  const float mb = (l < ROW_M_STRIDE) ? B.m_bar[row * ROW_M_STRIDE + l] : 0.f;
  const float lz_bar = warp_sum(mb * dm_lz);
  float g = 0.f;
  if (l == 0) g = sc.Mn_bar * sc.Mn * LN10F;
  else if (l == 1) g = tau_bar * (float)R.tau * LN10F;
  else if (l == 2) g = lz_bar;
  else if (l == 3) g = sc.AV_bar * TINY5_AV_PER_TAUV;
  if (l < SPS_NDIM) {
    g = (l < 4) ? g * d_l + dlp : 0.f;
    grad[row * SPS_NDIM + l] = g;
    if (lf.p_w) {
      const int64_t o = row * SPS_NDIM + l;
      const float pn = lf_p + lf_eps * g;
      lf.p_w[o] = pn;
      lf.theta_w[o] = lf_th + lf_eps * lf_im * pn;
    }
  }
  if (l == 0 && logp) logp[row] = sc.logp_like + lp;
}

// SPS_MODEL_GAUSS_TEST: logP = -1/2 d^T P d, grad = -P d, d = theta - mu (lane p owns parameter p < D)
__global__ void __launch_bounds__(256) gauss_eval_kernel(TableDev T, const float* theta, int64_t n, const int* __restrict__ rows,
                                                         float* __restrict__ logp, float* __restrict__ grad, LeapfrogFuse lf) {
  const int64_t r = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  if (r >= n) return;
  const int64_t row = rows ? rows[r] : r;
  const int l = lane_id(), D = T.n_dim;
  const bool act = l < D;
  const int64_t o = row * SPS_NDIM + (l < SPS_NDIM ? l : 0);
  const float th = theta[o];
  const float d = act ? th - T.gauss[l] : 0.f;
  float Pd = 0.f;
  for (int q = 0; q < D; ++q) {
    const float dq = __shfl_sync(FULL_MASK, d, q);
    if (act) Pd = fmaf(T.gauss[SPS_NDIM + l * SPS_NDIM + q], dq, Pd);
  }
  const float quad = warp_sum(d * Pd);
  if (l == 0 && logp) logp[row] = -0.5f * quad;
  if (grad && l < SPS_NDIM) {
    const float g = -Pd;
    float lf_eps = 0.f, lf_p = 0.f, lf_im = 0.f;
    if (lf.p_w) { lf_eps = lf.eps[row]; lf_p = lf.p_w[o]; lf_im = lf.inv_mass[o]; }
    grad[o] = g;
    if (lf.p_w) {
      const float pn = lf_p + lf_eps * g;
      lf.p_w[o] = pn;
      lf.theta_w[o] = th + lf_eps * lf_im * pn;            // theta aliases lf.theta_w in the samplers: read above, written here
    }
  }
}

static inline unsigned warp_blocks(int64_t n) { return (unsigned)((n * 32 + 255) / 256); }

void launch_prologue_tiny5(const TableDev& T, const PriorDev& P, const float* theta, int64_t n, bool unbounded, const int* rows,
                           RowBuffers B, bool with_hist, cudaStream_t s) {
  if (n <= 0) return;
  int* hist = nullptr;
  if (with_hist) { hist = B.bins; cudaMemsetAsync(B.bins, 0, 4 * (size_t)(T.n_z + 1) * sizeof(int), s); }
  sps_prof_begin(SPS_K_PROLOGUE, s);
  tiny5_prologue_kernel<<<warp_blocks(n), 256, 0, s>>>(T, P, theta, n, unbounded, rows, B, hist);
  sps_prof_end(SPS_K_PROLOGUE, s);
  sps_count_launch();
}
void launch_epilogue_tiny5(const TableDev& T, const PriorDev& P, const float* theta, int64_t n, bool unbounded, bool with_prior,
                           const int* rows, RowBuffers B, float* logp, float* grad, LeapfrogFuse lf, cudaStream_t s) {
  if (n <= 0) return;
  sps_prof_begin(SPS_K_EPILOGUE, s);
  tiny5_epilogue_kernel<<<warp_blocks(n), 256, 0, s>>>(T, P, theta, n, unbounded, with_prior, rows, B, logp, grad, lf);
  sps_prof_end(SPS_K_EPILOGUE, s);
  sps_count_launch();
}
void launch_gauss_eval(const TableDev& T, const float* theta, int64_t n, const int* rows, float* logp, float* grad, LeapfrogFuse lf,
                       cudaStream_t s) {
  if (n <= 0) return;
  gauss_eval_kernel<<<warp_blocks(n), 256, 0, s>>>(T, theta, n, rows, logp, grad, lf);
  sps_count_launch();
}
