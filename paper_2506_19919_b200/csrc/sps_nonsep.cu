// sps_nonsep.cu -- approximate photometry (Eq. 6) with NON-SEPARABLE weights (
// PAPER.md:52, 378; R26): P_SSP(i, j) = a_i m_ij, the lognormal MDF of age bin i centred on
// logZ + gamma (log10 age_i - 9).  The factorisation that the separable kernels exploit (sum over ages first, then over
// metallicities) is gone: the contraction is over all n_age n_Z pairs,
//     flux_b = F_att,b Mn sum_ij a_i m_ij [c_t + f D_t]_ijb .
// One warp per row, fp32: lanes own the table entries e = (j, b) of an age row (four per lane) and walk the ages; the MDF
// of each age bin is evaluated by the lanes j < n_Z (met_bin) and broadcast.  Pass 1 gives the fluxes, the likelihood and
// its derivative g_b; pass 2 walks the ages again for a_bar_i and the bars of (logZ, sigma_logZ) through every bin's MDF.
// This is the plain SIMT formulation (the table rows come from L2); the tensor-core formulation as a K = n_age n_Z
// contraction is listed in DESIGN.md section 9.
#include "sps_internal.h"

#define NS_E 4                                   // table entries per lane: 4 x 32 >= n_Z n_band (<= 128)

__global__ void __launch_bounds__(256) nonsep_approx_kernel(TableDev T, int64_t n, const int* __restrict__ rows, const int* __restrict__ gal_of_row,
                                                            const float* __restrict__ obs_flux, const float* __restrict__ obs_sigma,
                                                            const float* __restrict__ flux_bar, bool want_grad, RowBuffers B) {
  __shared__ float s_u[8][2][128];               // per warp: sum_i a_i m_ij c_ijb for the two arrays of the z cell, by entry
  __shared__ float s_sbar[8][SPS_MAX_BAND];
  const int64_t r = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  if (r >= n) return;
  const int w = threadIdx.x >> 5, l = lane_id();
  const int64_t row = rows ? rows[r] : r;
  const RowScalars sc = B.sc[row];
  const float lz = sc.pad1, slz = sc.pad2, f = sc.zfrac, Mn = sc.Mn;
  const int E = T.n_Z * T.n_band;
  int ej[NS_E]; bool ok[NS_E];
#pragma unroll
  for (int k = 0; k < NS_E; ++k) { const int e = l + 32 * k; ok[k] = e < E; ej[k] = ok[k] ? e / T.n_band : 0; }
  float a[SPS_AGE_PER_LANE];
#pragma unroll
  for (int q = 0; q < SPS_AGE_PER_LANE; ++q) a[q] = B.a[row * ROW_A_STRIDE + l + 32 * q];
  const float* c0 = T.cssp + ((int64_t)sc.zbin * 2) * T.n_age * T.cs_stride;
  const float* c1 = c0 + (int64_t)T.n_age * T.cs_stride;
  // ---- pass 1: U^(s)_e = sum_i a_i m_i,j(e) c^(s)_i,e ----
  float u0[NS_E] = {0.f, 0.f, 0.f, 0.f}, u1[NS_E] = {0.f, 0.f, 0.f, 0.f};
  for (int i = 0; i < T.n_age; ++i) {
    float m, d_mu, d_s;
    met_bin(T, lz + T.agez_gamma * T.la9[i], slz, m, d_mu, d_s);
    const float ai = __shfl_sync(FULL_MASK, a[i >> 5], i & 31);
#pragma unroll
    for (int k = 0; k < NS_E; ++k) {
      const float mj = __shfl_sync(FULL_MASK, m, ej[k]) * ai;
      if (ok[k]) {
        u0[k] = fmaf(mj, __ldg(c0 + (int64_t)i * T.cs_stride + l + 32 * k), u0[k]);
        u1[k] = fmaf(mj, __ldg(c1 + (int64_t)i * T.cs_stride + l + 32 * k), u1[k]);
      }
    }
  }
#pragma unroll
  for (int k = 0; k < NS_E; ++k) { s_u[w][0][l + 32 * k] = ok[k] ? u0[k] : 0.f; s_u[w][1][l + 32 * k] = ok[k] ? u1[k] : 0.f; }
  __syncwarp();
  // ---- band step (lane = band): dust at lambda_eff / (1+z), flux, likelihood, direct bars ----
  const int b = l;
  const bool isb = b < T.n_band;
  const float zp = 1.f + sc.z;
  float S0 = 0.f, S1 = 0.f, F = 1.f, F_av = 0.f, F_del = 0.f, F_fl = 0.f, F_lam = 0.f, lam_r = 1.f, g = 0.f, chi2 = 0.f;
  if (isb) {
    for (int j = 0; j < T.n_Z; ++j) { S0 += s_u[w][0][j * T.n_band + b]; S1 += s_u[w][1][j * T.n_band + b]; }
    lam_r = T.lam_eff[b] / zp;
    dust_at(lam_r, sc.AV, sc.delta, sc.Ffloor, F, F_av, F_del, F_fl, F_lam, T.model == SPS_MODEL_TINY5);
    const float flux = F * Mn * (S0 + f * S1);
    B.flux[row * SPS_MAX_BAND + b] = flux;
    if (flux_bar) g = flux_bar[row * T.n_band + b];
    else {
      const int64_t gal = gal_of_row ? gal_of_row[row] : row;
      const float d = obs_flux[gal * T.n_band + b], sg = obs_sigma[gal * T.n_band + b];
      const float rr = (flux - d) / sg;
      chi2 = rr * rr; g = -rr / sg;
    }
  }
  const float Sint = S0 + f * S1;
  const float v_mn = warp_sum(g * F * Sint);
  const float v_z = warp_sum(g * (F * Mn * S1 * T.inv_dz + Mn * Sint * F_lam * (-lam_r / zp)));
  const float v_av = warp_sum(g * Mn * Sint * F_av), v_de = warp_sum(g * Mn * Sint * F_del), v_fl = warp_sum(g * Mn * Sint * F_fl);
  chi2 = warp_sum(chi2);
  if (l == 0) {
    RowScalars* out = B.sc + row;
    out->logp_like = -0.5f * chi2;
    if (want_grad) { out->Mn_bar = v_mn; out->z_bar = v_z; out->AV_bar = v_av; out->delta_bar = v_de; out->Ffloor_bar = v_fl; }
  }
  if (!want_grad) return;
  if (l < SPS_MAX_BAND) s_sbar[w][l] = isb ? g * F * Mn : 0.f;
  __syncwarp();
  // ---- pass 2: t_e = sbar_b (c_t + f D_t)_i,e;  a_bar_i = sum_e m_ij t_e;  lz_bar, slz_bar += a_i sum_e dm_ij t_e ----
  float sb[NS_E];
#pragma unroll
  for (int k = 0; k < NS_E; ++k) { const int e = l + 32 * k; sb[k] = ok[k] ? s_sbar[w][e - ej[k] * T.n_band] : 0.f; }
  float lz_bar = 0.f, slz_bar = 0.f, abar[SPS_AGE_PER_LANE] = {0.f, 0.f, 0.f, 0.f};
  for (int i = 0; i < T.n_age; ++i) {
    float m, d_mu, d_s;
    met_bin(T, lz + T.agez_gamma * T.la9[i], slz, m, d_mu, d_s);
    const float ai = __shfl_sync(FULL_MASK, a[i >> 5], i & 31);
    float pa = 0.f, pl = 0.f, ps = 0.f;
#pragma unroll
    for (int k = 0; k < NS_E; ++k) {
      const float mj = __shfl_sync(FULL_MASK, m, ej[k]), dl = __shfl_sync(FULL_MASK, d_mu, ej[k]), ds = __shfl_sync(FULL_MASK, d_s, ej[k]);
      if (ok[k]) {
        const float t = sb[k] * fmaf(f, __ldg(c1 + (int64_t)i * T.cs_stride + l + 32 * k), __ldg(c0 + (int64_t)i * T.cs_stride + l + 32 * k));
        pa = fmaf(mj, t, pa); pl = fmaf(dl, t, pl); ps = fmaf(ds, t, ps);
      }
    }
    pa = warp_sum(pa);
    lz_bar = fmaf(ai, pl, lz_bar); slz_bar = fmaf(ai, ps, slz_bar);
    if ((i & 31) == l) abar[i >> 5] = pa;
  }
  lz_bar = warp_sum(lz_bar); slz_bar = warp_sum(slz_bar);
#pragma unroll
  for (int q = 0; q < SPS_AGE_PER_LANE; ++q) B.a_bar[row * ROW_A_STRIDE + l + 32 * q] = abar[q];
  if (l < ROW_M_STRIDE) B.m_bar[row * ROW_M_STRIDE + l] = 0.f;
  if (l == 0) { B.sc[row].pad1 = lz_bar; B.sc[row].pad2 = slz_bar; }
}

void launch_nonsep_approx(const TableDev& T, int64_t n, const int* rows, const int* gal_of_row, const float* obs_flux, const float* obs_sigma,
                          const float* flux_bar, bool want_grad, RowBuffers B, cudaStream_t s) {
  if (n <= 0) return;
  sps_prof_begin(SPS_K_APPROX, s);
  nonsep_approx_kernel<<<(unsigned)((n * 32 + 255) / 256), 256, 0, s>>>(T, n, rows, gal_of_row, obs_flux, obs_sigma, flux_bar, want_grad, B);
  sps_prof_end(SPS_K_APPROX, s);
  sps_count_launch();
}
