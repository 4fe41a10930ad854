// sps_kernels.cu -- prologue (a0-a5), approximate-photometry contraction (a7, a9, a10) and
// epilogue (reverse of a0-a5 + prior) kernels.  One warp per parameter row.
#include "sps_rows.cuh"

#define WARPS_PER_BLOCK 8

// ---------------------------------------------------------------------------------------------
// Forward model of one row: everything a0-a5 needs, held per lane.
// ---------------------------------------------------------------------------------------------
struct RowFwd {
  float th[SPS_NDIM], dth[SPS_NDIM];
  double t_obs_d, z_d;
  float dt_dz, Msum, Mf;
  AgeQuad Q;
  BurstQuad Bq;
  float m, dm_lz, dm_s;
};

template <bool WANT_GRAD>
__device__ __forceinline__ void row_forward(const TableDev& T, const PriorDev& P, const float* __restrict__ row,
                                            bool unbounded, RowFwd& R) {
  load_params(row, unbounded, P, R.th, R.dth, R.z_d);
  cosmic_time(T, R.z_d, R.t_obs_d, R.dt_dz);
  smooth_bins<WANT_GRAD>(T, R.t_obs_d, R.th[1], R.th[2], R.th[3], R.Q);
  float s = 0.f;
#pragma unroll
  for (int q = 0; q < SPS_AGE_PER_LANE; ++q) s += R.Q.dM[q];
  R.Msum = warp_sum(s);                                        // Eq. (A3) for M_formed = 1
  R.Mf = exp2f((R.th[0] - T.log10_mass_unit) * 3.321928094887362f);
  burst_bins(T, R.th[5], R.th[6], R.Bq);
  met_bin(T, R.th[7], R.th[8], R.m, R.dm_lz, R.dm_s);
}

__global__ void __launch_bounds__(32 * WARPS_PER_BLOCK)
prologue_kernel(TableDev T, PriorDev P, const float* __restrict__ theta, int64_t n, bool unbounded,
                const int* __restrict__ rows, RowBuffers B) {
  const int64_t r = (int64_t)blockIdx.x * WARPS_PER_BLOCK + (threadIdx.x >> 5);
  if (r >= n) return;
  const int64_t row = rows ? rows[r] : r;
  const int l = lane_id();
  RowFwd R;
  row_forward<false>(T, P, theta + row * SPS_NDIM, unbounded, R);
  const float Fb = R.th[4], inv_M = 1.f / R.Msum;
#pragma unroll
  for (int q = 0; q < SPS_AGE_PER_LANE; ++q) {
    const int i = l + 32 * q;
    if (i < ROW_A_STRIDE) B.a[row * ROW_A_STRIDE + i] = (i < T.n_age) ? (1.f - Fb) * R.Q.dM[q] * inv_M + Fb * R.Bq.P[q] : 0.f;  // Eq. (A6)
  }
  if (l < ROW_M_STRIDE) B.m[row * ROW_M_STRIDE + l] = R.m;
  if (l == 0) {
    RowScalars sc;
    sc.Mn = R.Mf * R.Msum;
    const float z = R.th[12];
    float zi = floorf((z - T.z_min) * T.inv_dz);
    zi = fminf(fmaxf(zi, 0.f), (float)(T.n_z - 2));
    sc.z = z; sc.zbin = (int)zi; sc.zfrac = (z - (T.z_min + zi * T.dz)) * T.inv_dz;
    sc.AV = R.th[9]; sc.delta = R.th[10]; sc.Ffloor = R.th[11];
    sc.logp_like = 0.f; sc.Mn_bar = sc.z_bar = sc.AV_bar = sc.delta_bar = sc.Ffloor_bar = 0.f;
    sc.pad0 = sc.pad1 = sc.pad2 = 0.f;
    B.sc[row] = sc;
  }
}

// ---------------------------------------------------------------------------------------------
// a7 + a9 + a10: approximate photometry (Eq. 6) fused with the Gaussian likelihood
// and the reverse pass over the c_SSP table.  v0: one warp per row, the two z-slices are read from
// L2; lane l owns the entries e = 4l..4l+3 of a slice row (e = j*n_band + b).
//   pass 1:  Q^(s)_e = sum_i a_i c^(s)[i][e]            (s = 0: c_t, s = 1: D_t = c_{t+1} - c_t)
//   S^(s)_b = sum_j m_j Q^(s)_{jb};  flux_b = F_att,b Mn [S^(0)_b + f S^(1)_b]
//   g_b = d logL / d flux_b = -(flux_b - d_b)/sigma_b^2   (or the caller's flux_bar)
//   pass 2:  a_bar_i = sum_e [v^(0)_e c^(0)[i][e] + v^(1)_e c^(1)[i][e]],  v^(s)_e = g_b F_b Mn {1, f} m_j
// ---------------------------------------------------------------------------------------------
struct ApproxSmem {
  float a[ROW_A_STRIDE];
  float Q0[128], Q1[128];
  float m[ROW_M_STRIDE], sbar[SPS_MAX_BAND];
};

__global__ void __launch_bounds__(32 * WARPS_PER_BLOCK)
approx_contract_kernel(TableDev T, int64_t n, const int* __restrict__ rows, const int* __restrict__ gal_of_row,
                       const float* __restrict__ obs_flux, const float* __restrict__ obs_sigma,
                       const float* __restrict__ flux_bar, bool want_grad, RowBuffers B) {
  __shared__ ApproxSmem smem_all[WARPS_PER_BLOCK];
  const int64_t r = (int64_t)blockIdx.x * WARPS_PER_BLOCK + (threadIdx.x >> 5);
  if (r >= n) return;
  const int64_t row = rows ? rows[r] : r;
  ApproxSmem& S = smem_all[threadIdx.x >> 5];
  const int l = lane_id();
  const int E = T.n_Z * T.n_band;
  RowScalars sc = B.sc[row];
#pragma unroll
  for (int q = 0; q < SPS_AGE_PER_LANE; ++q) S.a[l + 32 * q] = B.a[row * ROW_A_STRIDE + l + 32 * q];
  if (l < ROW_M_STRIDE) S.m[l] = B.m[row * ROW_M_STRIDE + l];
  __syncwarp();
  const float* c0p = T.cssp + ((int64_t)sc.zbin * 2 * T.n_age) * T.cs_stride + 4 * l;     // c_t, then D_t
  const float* c1p = c0p + (int64_t)T.n_age * T.cs_stride;
  const bool act = 4 * l < T.cs_stride;
  float4 q0 = make_float4(0, 0, 0, 0), q1 = make_float4(0, 0, 0, 0);
  if (act) {
#pragma unroll 4
    for (int i = 0; i < T.n_age; ++i) {
      const float4 c0 = __ldg(reinterpret_cast<const float4*>(c0p + (int64_t)i * T.cs_stride));
      const float4 c1 = __ldg(reinterpret_cast<const float4*>(c1p + (int64_t)i * T.cs_stride));
      const float ai = S.a[i];
      q0.x += ai * c0.x; q0.y += ai * c0.y; q0.z += ai * c0.z; q0.w += ai * c0.w;
      q1.x += ai * c1.x; q1.y += ai * c1.y; q1.z += ai * c1.z; q1.w += ai * c1.w;
    }
  }
  reinterpret_cast<float4*>(S.Q0)[l] = q0;
  reinterpret_cast<float4*>(S.Q1)[l] = q1;
  __syncwarp();
  // per-band quantities on lanes b < n_band
  const float f = sc.zfrac;
  float S0 = 0.f, S1 = 0.f, F = 1.f, F_av = 0.f, F_del = 0.f, F_fl = 0.f, F_lam = 0.f, lam_r = 1.f, g = 0.f, flux = 0.f;
  float chi2 = 0.f;
  const bool isb = l < T.n_band;
  if (isb) {
    for (int j = 0; j < T.n_Z; ++j) { S0 += S.m[j] * S.Q0[j * T.n_band + l]; S1 += S.m[j] * S.Q1[j * T.n_band + l]; }
    lam_r = T.lam_eff[l] / (1.f + sc.z);
    dust_at(lam_r, sc.AV, sc.delta, sc.Ffloor, F, F_av, F_del, F_fl, F_lam);
    const float Sint = S0 + f * S1;
    flux = F * sc.Mn * Sint;
    B.flux[row * SPS_MAX_BAND + l] = flux;
    if (flux_bar) g = flux_bar[row * T.n_band + l];
    else {
      const int64_t gal = gal_of_row ? gal_of_row[row] : row;
      const float d = obs_flux[gal * T.n_band + l], sg = obs_sigma[gal * T.n_band + l];
      const float rr = (flux - d) / sg;
      chi2 = rr * rr;
      g = -rr / sg;
    }
  }
  chi2 = warp_sum(chi2);
  if (!want_grad) {
    if (l == 0) B.sc[row].logp_like = -0.5f * chi2;
    return;
  }
  {
    const float Sint = S0 + f * S1;
    float Mn_bar = warp_sum(isb ? g * F * Sint : 0.f);
    float z_bar = warp_sum(isb ? g * (F * sc.Mn * S1 * T.inv_dz + sc.Mn * Sint * F_lam * (-lam_r / (1.f + sc.z))) : 0.f);
    float av_bar = warp_sum(isb ? g * sc.Mn * Sint * F_av : 0.f);
    float del_bar = warp_sum(isb ? g * sc.Mn * Sint * F_del : 0.f);
    float fl_bar = warp_sum(isb ? g * sc.Mn * Sint * F_fl : 0.f);
    if (l == 0) {
      sc.logp_like = -0.5f * chi2; sc.Mn_bar = Mn_bar; sc.z_bar = z_bar;
      sc.AV_bar = av_bar; sc.delta_bar = del_bar; sc.Ffloor_bar = fl_bar;
      B.sc[row] = sc;
    }
    if (isb) S.sbar[l] = g * F * sc.Mn;
  }
  __syncwarp();
  // m_bar_j
  if (l < ROW_M_STRIDE) {
    float mb = 0.f;
    if (l < T.n_Z)
      for (int b = 0; b < T.n_band; ++b) mb += S.sbar[b] * (S.Q0[l * T.n_band + b] + f * S.Q1[l * T.n_band + b]);
    B.m_bar[row * ROW_M_STRIDE + l] = mb;
  }
  // v quads
  float v0[4], v1[4];
#pragma unroll
  for (int k = 0; k < 4; ++k) {
    const int e = 4 * l + k;
    float v = 0.f;
    if (e < E) { const int j = e / T.n_band, b = e - j * T.n_band; v = S.sbar[b] * S.m[j]; }
    v0[k] = v; v1[k] = f * v;
  }
  // pass 2
  float abar[SPS_AGE_PER_LANE] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
  for (int qq = 0; qq < SPS_AGE_PER_LANE; ++qq) {
    const int i0 = 32 * qq;
    float keep = 0.f;
    const int i1 = min(32, T.n_age - i0);
    for (int ii = 0; ii < i1; ++ii) {
      float part = 0.f;
      if (act) {
        const float4 c0 = __ldg(reinterpret_cast<const float4*>(c0p + (int64_t)(i0 + ii) * T.cs_stride));
        const float4 c1 = __ldg(reinterpret_cast<const float4*>(c1p + (int64_t)(i0 + ii) * T.cs_stride));
        part = v0[0] * c0.x + v0[1] * c0.y + v0[2] * c0.z + v0[3] * c0.w + v1[0] * c1.x + v1[1] * c1.y + v1[2] * c1.z + v1[3] * c1.w;
      }
      part = warp_sum(part);
      if (l == ii) keep = part;
    }
    abar[qq] = keep;
  }
#pragma unroll
  for (int q = 0; q < SPS_AGE_PER_LANE; ++q) B.a_bar[row * ROW_A_STRIDE + l + 32 * q] = abar[q];
}

// ---------------------------------------------------------------------------------------------
// Reverse of a0-a5 (a10) + skew-normal prior (a9): one warp per row recomputes the quadratures with
// their parameter partials and contracts them with a_bar, m_bar, Mn_bar and the direct bars.
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(32 * WARPS_PER_BLOCK)
epilogue_kernel(TableDev T, PriorDev P, const float* __restrict__ theta, int64_t n, bool unbounded, bool with_prior,
                const int* __restrict__ rows, RowBuffers B, float* __restrict__ logp, float* __restrict__ grad) {
  const int64_t r = (int64_t)blockIdx.x * WARPS_PER_BLOCK + (threadIdx.x >> 5);
  if (r >= n) return;
  const int64_t row = rows ? rows[r] : r;
  const int l = lane_id();
  RowFwd R;
  row_forward<true>(T, P, theta + row * SPS_NDIM, unbounded, R);
  const RowScalars sc = B.sc[row];
  const float Fb = R.th[4], inv_M = 1.f / R.Msum;
  float abar[SPS_AGE_PER_LANE], Ps[SPS_AGE_PER_LANE];
  float s_fb = 0.f, s_pp = 0.f, s_ltp = 0.f, s_ltm = 0.f;
#pragma unroll
  for (int q = 0; q < SPS_AGE_PER_LANE; ++q) {
    abar[q] = B.a_bar[row * ROW_A_STRIDE + l + 32 * q];
    Ps[q] = R.Q.dM[q] * inv_M;
    s_fb += abar[q] * (R.Bq.P[q] - Ps[q]);             // dL/dF_burst           (Eq. A6)
    s_pp += abar[q] * Ps[q];
    s_ltp += abar[q] * R.Bq.d_ltp[q];
    s_ltm += abar[q] * R.Bq.d_ltm[q];
  }
  s_fb = warp_sum(s_fb); s_pp = warp_sum(s_pp); s_ltp = warp_sum(s_ltp) * Fb; s_ltm = warp_sum(s_ltm) * Fb;
  // dL/d(dM_i) = (1-Fb)/Msum (a_bar_i - sum_k a_bar_k Ps_k) + Mn_bar * Mf
  float s_tau = 0.f, s_al = 0.f, s_be = 0.f, s_t = 0.f;
#pragma unroll
  for (int q = 0; q < SPS_AGE_PER_LANE; ++q) {
    const float dMb = (1.f - Fb) * inv_M * (abar[q] - s_pp) + sc.Mn_bar * R.Mf;
    s_tau += dMb * R.Q.g_tau[q]; s_al += dMb * R.Q.g_al[q]; s_be += dMb * R.Q.g_be[q]; s_t += dMb * R.Q.g_t[q];
  }
  s_tau = warp_sum(s_tau); s_al = warp_sum(s_al); s_be = warp_sum(s_be); s_t = warp_sum(s_t);
  const float mb = (l < ROW_M_STRIDE) ? B.m_bar[row * ROW_M_STRIDE + l] : 0.f;
  const float s_lz = warp_sum(mb * R.dm_lz), s_s = warp_sum(mb * R.dm_s);
  float g = 0.f;
  switch (l) {
    case 0: g = sc.Mn_bar * sc.Mn * LN10F; break;
    case 1: g = s_tau; break;
    case 2: g = s_al; break;
    case 3: g = s_be; break;
    case 4: g = s_fb; break;
    case 5: g = s_ltp; break;
    case 6: g = s_ltm; break;
    case 7: g = s_lz; break;
    case 8: g = s_s; break;
    case 9: g = sc.AV_bar; break;
    case 10: g = sc.delta_bar; break;
    case 11: g = sc.Ffloor_bar; break;
    case 12: g = sc.z_bar + s_t * R.dt_dz; break;
    default: break;
  }
  float lp = 0.f;
  if (l < SPS_NDIM) {
    float dth = 1.f;
#pragma unroll
    for (int p = 0; p < SPS_NDIM; ++p) if (p == l) dth = R.dth[p];
    g *= dth;
    if (with_prior) {
      float dlp;
      log_skew_normal(theta[row * SPS_NDIM + l], P.xi[l], P.omega[l], P.skew[l], lp, dlp);
      g += dlp;
    }
    if (grad) grad[row * SPS_NDIM + l] = g;
  }
  lp = warp_sum(lp);
  if (l == 0 && logp) logp[row] = sc.logp_like + lp;
}

__global__ void copy_weights_kernel(TableDev T, int64_t n, RowBuffers B, float* w_age, float* w_met, float* mstar) {
  const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  const int64_t row = idx / ROW_A_STRIDE; const int i = (int)(idx % ROW_A_STRIDE);
  if (row >= n) return;
  if (w_age && i < T.n_age) w_age[row * T.n_age + i] = B.a[row * ROW_A_STRIDE + i];
  if (w_met && i < T.n_Z) w_met[row * T.n_Z + i] = B.m[row * ROW_M_STRIDE + i];
  if (mstar && i == 0) mstar[row] = B.sc[row].Mn;
}

__global__ void copy_flux_kernel(TableDev T, int64_t n, RowBuffers B, float* flux) {
  const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  const int64_t row = idx / SPS_MAX_BAND; const int b = (int)(idx % SPS_MAX_BAND);
  if (row < n && b < T.n_band) flux[row * T.n_band + b] = B.flux[row * SPS_MAX_BAND + b];
}

static inline unsigned blocks_for_rows(int64_t n) { return (unsigned)((n + WARPS_PER_BLOCK - 1) / WARPS_PER_BLOCK); }

void launch_prologue(const TableDev& T, const PriorDev& P, const float* theta, int64_t n, bool unbounded,
                     const int* rows, RowBuffers B, cudaStream_t s) {
  if (n <= 0) return;
  sps_prof_begin(SPS_K_PROLOGUE, s);
  prologue_kernel<<<blocks_for_rows(n), 32 * WARPS_PER_BLOCK, 0, s>>>(T, P, theta, n, unbounded, rows, B);
  sps_prof_end(SPS_K_PROLOGUE, s);
  sps_count_launch();
}
void launch_approx_contract(const TableDev& T, int64_t n, const int* rows, const int* gal_of_row,
                            const float* obs_flux, const float* obs_sigma, const float* flux_bar,
                            bool want_grad, RowBuffers B, cudaStream_t s) {
  if (n <= 0) return;
  sps_prof_begin(SPS_K_APPROX, s);
  approx_contract_kernel<<<blocks_for_rows(n), 32 * WARPS_PER_BLOCK, 0, s>>>(T, n, rows, gal_of_row, obs_flux, obs_sigma,
                                                                           flux_bar, want_grad, B);
  sps_prof_end(SPS_K_APPROX, s);
  sps_count_launch();
}
void launch_epilogue(const TableDev& T, const PriorDev& P, const float* theta, int64_t n, bool unbounded,
                     bool with_prior, const int* rows, RowBuffers B, float* logp, float* grad, cudaStream_t s) {
  if (n <= 0) return;
  sps_prof_begin(SPS_K_EPILOGUE, s);
  epilogue_kernel<<<blocks_for_rows(n), 32 * WARPS_PER_BLOCK, 0, s>>>(T, P, theta, n, unbounded, with_prior, rows, B, logp, grad);
  sps_prof_end(SPS_K_EPILOGUE, s);
  sps_count_launch();
}
void launch_copy_weights(const TableDev& T, int64_t n, RowBuffers B, float* w_age, float* w_met, float* mstar, cudaStream_t s) {
  if (n <= 0) return;
  const int64_t tot = n * ROW_A_STRIDE;
  copy_weights_kernel<<<(unsigned)((tot + 255) / 256), 256, 0, s>>>(T, n, B, w_age, w_met, mstar);
  sps_count_launch();
}
void launch_copy_flux(const TableDev& T, int64_t n, RowBuffers B, float* flux, cudaStream_t s) {
  if (n <= 0) return;
  const int64_t tot = n * SPS_MAX_BAND;
  copy_flux_kernel<<<(unsigned)((tot + 255) / 256), 256, 0, s>>>(T, n, B, flux);
  sps_count_launch();
}
