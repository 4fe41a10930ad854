// sps_table.cu -- sps_create_table / sps_destroy_table: device-resident grids, per-wavelength
// constants and the c_SSP lookup table (Eq. 7), which is built on the GPU.
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <vector>
#include "sps_internal.h"

// T_b(lambda_obs): Gaussian transmission truncated at 5 sigma (R4)
__device__ __forceinline__ float filter_T(float lam_obs, float mu, float sigma) {
  const float x = (lam_obs - mu) / sigma;
  return (fabsf(x) <= 5.f) ? expf(-0.5f * x * x) : 0.f;
}

// c_SSP[t][i][j*n_band+b] = sum_k L_ij(lam_k) T_b(lam_k (1+z_t)) dlam_k  (Eq. 7).  One warp per (t, ij).
// Slice t of the device table holds TWO arrays: c_t and the increment D_t = c_{t+1} - c_t (zero for the
// last slice), so that the linear interpolation c_t + f D_t and its z-derivative D_t / dz
// carry no fp32 cancellation.  Both are accumulated in double and rounded once.
__device__ __forceinline__ double filter_T_d(double lam_obs, double mu, double sigma) {
  const double x = (lam_obs - mu) / sigma;
  return (fabs(x) <= 5.0) ? exp(-0.5 * x * x) : 0.0;
}
// tabulated curve in double (R4): linear interpolation between the band's knots, zero outside its support
__device__ __forceinline__ double filter_tab_d(const double* __restrict__ w, const double* __restrict__ t, int n, double lam) {
  if (!(lam >= w[0]) || !(lam <= w[n - 1])) return 0.0;
  int a = 0, c = n - 1;                                     // largest a with w[a] <= lam, capped at n - 2
  while (c - a > 1) { const int mid = (a + c) >> 1; if (w[mid] <= lam) a = mid; else c = mid; }
  return t[a] + (lam - w[a]) * (t[a + 1] - t[a]) / (w[a + 1] - w[a]);
}
__global__ void __launch_bounds__(256) cssp_build_kernel(TableDev T, const double* __restrict__ wave_d, const double* __restrict__ dlam_d,
                                                          double z_min_d, double dz_d, const double* __restrict__ fw, const double* __restrict__ ft,
                                                          const int* __restrict__ foff, float* __restrict__ cssp) {
  const int64_t w = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  if (w >= (int64_t)T.n_z * T.K) return;
  const int t = (int)(w / T.K), ij = (int)(w % T.K);
  const int i = ij / T.n_Z, j = ij % T.n_Z;
  const int l = threadIdx.x & 31;
  const float* L = T.ssp + (int64_t)ij * T.n_wave_pad;
  const bool last = (t == T.n_z - 1);
  const double zp0 = 1.0 + z_min_d + dz_d * (double)t, zp1 = last ? zp0 : 1.0 + z_min_d + dz_d * (double)(t + 1);
  for (int b = 0; b < T.n_band; ++b) {
    const double mu = (double)T.filt_mu[b], sg = (double)T.filt_sigma[b];
    const bool tab = T.filt_tab != 0;
    const double* bw = tab ? fw + foff[b] : nullptr; const double* bt = tab ? ft + foff[b] : nullptr;
    const int bn = tab ? foff[b + 1] - foff[b] : 0;
    const double lo = (tab ? bw[0] : mu - 5.0 * sg) / zp1, hi = (tab ? bw[bn - 1] : mu + 5.0 * sg) / zp0;      // union of the two supports
    int a = 0, c = T.n_wave;
    while (a < c) { int mid = (a + c) >> 1; if (wave_d[mid] < lo) a = mid + 1; else c = mid; }
    const int k0 = max(a - 1, 0);
    a = k0; c = T.n_wave;
    while (a < c) { int mid = (a + c) >> 1; if (wave_d[mid] <= hi) a = mid + 1; else c = mid; }
    const int k1 = min(a + 1, T.n_wave);
    double acc0 = 0.0, acc1 = 0.0;
    for (int k = k0 + l; k < k1; k += 32) {
      const double Lk = (double)L[k] * dlam_d[k];
      acc0 += Lk * (tab ? filter_tab_d(bw, bt, bn, wave_d[k] * zp0) : filter_T_d(wave_d[k] * zp0, mu, sg));
      acc1 += Lk * (tab ? filter_tab_d(bw, bt, bn, wave_d[k] * zp1) : filter_T_d(wave_d[k] * zp1, mu, sg));
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) { acc0 += __shfl_xor_sync(FULL_MASK, acc0, o); acc1 += __shfl_xor_sync(FULL_MASK, acc1, o); }
    if (l == 0) {
      float* row = cssp + (((int64_t)t * 2) * T.n_age + i) * T.cs_stride + j * T.n_band + b;
      row[0] = (float)acc0;
      row[(int64_t)T.n_age * T.cs_stride] = (float)(acc1 - acc0);
    }
  }
}

template <class T>
static T* upload(const std::vector<T>& v, sps_status& st) {
  T* d = nullptr;
  if (st != SPS_OK) return nullptr;
  if (cudaMalloc(&d, v.size() * sizeof(T)) != cudaSuccess) { st = SPS_ENOMEM; sps_set_error("cudaMalloc of %zu bytes failed", v.size() * sizeof(T)); return nullptr; }
  if (cudaMemcpy(d, v.data(), v.size() * sizeof(T), cudaMemcpyHostToDevice) != cudaSuccess) { st = SPS_ECUDA; sps_set_error("cudaMemcpy H2D failed"); }
  return d;
}

static double calz_k0(double lam_A) {
  const double u = 1.0e4 / lam_A;
  double k = (u > 1.2809053864877329) ? 2.659 * (-2.156 + 1.509 * u - 0.198 * u * u + 0.011 * u * u * u) + 4.05
                                       : 2.659 * (-1.857 + 1.040 * u) + 4.05;
  return k > 0 ? k : 0.0;
}
static double drude_profile(double lam) {
  const double l0 = 2175.0, w = 350.0, n = (lam * w) * (lam * w), d = (lam * lam - l0 * l0);
  return n / (d * d + n);
}

// SPS_MODEL_GAUSS_TEST: no grids; the table holds mu and the precision matrix
static sps_status create_gauss_table(const sps_table_desc* d, sps_table** out) {
  if (d->gauss_ndim < 1 || d->gauss_ndim > SPS_NDIM || !d->gauss_mu || !d->gauss_prec) {
    sps_set_error("sps_create_table: SPS_MODEL_GAUSS_TEST needs 1 <= gauss_ndim <= 13, gauss_mu and gauss_prec"); return SPS_EINVAL; }
  const int D = d->gauss_ndim;
  for (int i = 0; i < D; ++i) {
    if (!(d->gauss_prec[i * D + i] > 0)) { sps_set_error("gauss_prec: non-positive diagonal"); return SPS_EINVAL; }
    for (int j = 0; j < i; ++j) if (fabs(d->gauss_prec[i * D + j] - d->gauss_prec[j * D + i]) > 1e-9 * fabs(d->gauss_prec[i * D + i])) {
      sps_set_error("gauss_prec is not symmetric"); return SPS_EINVAL; }
  }
  sps_status st = sps_require_device();
  if (st != SPS_OK) return st;
  sps_table* t = new sps_table();
  memset(&t->dev, 0, sizeof(TableDev));
  t->dev.model = SPS_MODEL_GAUSS_TEST; t->dev.n_dim = D; t->dev.n_z = 2;
  std::vector<float> g(SPS_NDIM + SPS_NDIM * SPS_NDIM, 0.f);
  for (int i = 0; i < D; ++i) { g[i] = (float)d->gauss_mu[i]; for (int j = 0; j < D; ++j) g[SPS_NDIM + i * SPS_NDIM + j] = (float)d->gauss_prec[i * D + j]; }
  t->dev.gauss = upload(g, st);
  int dev = 0; cudaGetDevice(&dev); cudaDeviceGetAttribute(&t->sm_count, cudaDevAttrMultiProcessorCount, dev);
  if (st != SPS_OK) { sps_destroy_table(t); return st; }
  *out = t;
  return SPS_OK;
}

extern "C" sps_status sps_create_table(const sps_table_desc* d, sps_table** out) {
  if (!d || !out) { sps_set_error("sps_create_table: null argument"); return SPS_EINVAL; }
  *out = nullptr;
  if (d->model != SPS_MODEL_TINY5 && d->model != SPS_MODEL_DPL13 && d->model != SPS_MODEL_GAUSS_TEST) {
    sps_set_error("sps_create_table: unknown model id %d", d->model); return SPS_EINVAL; }
  if (d->model == SPS_MODEL_GAUSS_TEST) return create_gauss_table(d, out);
  const bool tab = d->filt_offsets != nullptr;
  if (!d->log10_age_yr || !d->log10_Z || !d->wave_A || !d->ssp || (tab ? (!d->filt_wave_A || !d->filt_trans) : (!d->filt_mu_A || !d->filt_sigma_A))) {
    sps_set_error("sps_create_table: null array in descriptor"); return SPS_EINVAL; }
  if (d->n_age < 2 || d->n_age > SPS_MAX_AGE || d->n_Z < 2 || d->n_Z > SPS_MAX_Z || d->n_band < 1 ||
      d->n_band > SPS_MAX_BAND || d->n_wave < 8 || d->n_z < 2 || d->n_Z * d->n_band > 128) {
    sps_set_error("sps_create_table: size out of range (n_age<=128, n_Z<=16, n_band<=16, n_Z*n_band<=128, n_wave>=8, n_z>=2)");
    return SPS_ESHAPE; }
  for (int i = 1; i < d->n_age; ++i) if (!(d->log10_age_yr[i] > d->log10_age_yr[i - 1])) { sps_set_error("age grid not increasing"); return SPS_EINVAL; }
  for (int i = 1; i < d->n_Z; ++i) if (!(d->log10_Z[i] > d->log10_Z[i - 1])) { sps_set_error("Z grid not increasing"); return SPS_EINVAL; }
  for (int i = 1; i < d->n_wave; ++i) if (!(d->wave_A[i] > d->wave_A[i - 1])) { sps_set_error("wavelength grid not increasing"); return SPS_EINVAL; }
  if (!(d->z_max > d->z_min) || !(d->H0 > 0) || !(d->Om > 0 && d->Om < 1)) { sps_set_error("bad z grid or cosmology"); return SPS_EINVAL; }
  if (d->dlogZ_dlogage != 0.0 && d->model != SPS_MODEL_DPL13) { sps_set_error("dlogZ_dlogage needs SPS_MODEL_DPL13"); return SPS_EINVAL; }
  if (tab) {
    if (d->filt_offsets[0] != 0) { sps_set_error("filt_offsets[0] must be 0"); return SPS_EINVAL; }
    for (int b = 0; b < d->n_band; ++b) {
      const int n = d->filt_offsets[b + 1] - d->filt_offsets[b];
      if (n < 2 || n > SPS_FTAB_MAX_KNOTS) { sps_set_error("filter %d: 2 to %d knots per band", b, SPS_FTAB_MAX_KNOTS); return SPS_ESHAPE; }
      const double* w = d->filt_wave_A + d->filt_offsets[b];
      if (!(w[0] > 0)) { sps_set_error("filter %d: wavelengths must be positive", b); return SPS_EINVAL; }
      for (int k = 1; k < n; ++k) if (!(w[k] > w[k - 1])) { sps_set_error("filter %d: knots not strictly increasing", b); return SPS_EINVAL; }
    }
  }
  sps_status st = sps_require_device();
  if (st != SPS_OK) return st;

  sps_table* t = new sps_table();
  TableDev& T = t->dev;
  memset(&T, 0, sizeof(T));
  T.model = d->model; T.n_dim = d->model == SPS_MODEL_TINY5 ? 4 : SPS_NDIM;
  T.agez_gamma = (float)d->dlogZ_dlogage; T.filt_tab = tab ? 1 : 0;
  { int dev = 0; cudaGetDevice(&dev); cudaDeviceGetAttribute(&t->sm_count, cudaDevAttrMultiProcessorCount, dev); }
  T.n_age = d->n_age; T.n_Z = d->n_Z; T.n_wave = d->n_wave; T.n_band = d->n_band; T.n_z = d->n_z;
  T.K = d->n_age * d->n_Z;
  T.n_wave_pad = (d->n_wave + 255) / 256 * 256;
  int E4 = (d->n_Z * d->n_band + 3) / 4;
  if ((E4 & 1) == 0) E4 += 1;                       // odd number of float4 per age row: conflict-free smem tiles
  T.cs_stride = 4 * E4;
  const int na = d->n_age;
  std::vector<float> A_edge(na + 1), A_mid(na), A_half(na), e_edge(na + 1), g_mid(d->n_Z - 1 > 0 ? d->n_Z - 1 : 1);
  std::vector<double> Ae(na + 1);
  std::vector<float> la9(na);
  for (int i = 0; i < na; ++i) la9[i] = (float)(d->log10_age_yr[i] - 9.0);
  Ae[0] = 0.0; e_edge[0] = -1e30f;
  for (int i = 1; i < na; ++i) { const double mid = 0.5 * (d->log10_age_yr[i] + d->log10_age_yr[i - 1]); Ae[i] = pow(10.0, mid - 9.0); e_edge[i] = (float)mid; }
  Ae[na] = 1e30; e_edge[na] = 1e30f;
  for (int i = 0; i <= na; ++i) A_edge[i] = (float)Ae[i];
  for (int i = 0; i < na; ++i) { A_mid[i] = (float)(0.5 * (Ae[i] + Ae[i + 1])); A_half[i] = (float)(0.5 * (Ae[i + 1] - Ae[i])); }
  for (int j = 0; j + 1 < d->n_Z; ++j) g_mid[j] = (float)(0.5 * (d->log10_Z[j] + d->log10_Z[j + 1]));
  const int nw = d->n_wave, nwp = T.n_wave_pad;
  std::vector<float> wave(nwp), dlam(nwp, 0.f), k0(nwp), dr(nwp), l2r(nwp);
  for (int k = 0; k < nwp; ++k) {
    const double lam = d->wave_A[k < nw ? k : nw - 1];
    // SPS_MODEL_TINY5's screen exp(-tau_V (lam/5500)^-0.7) is Eq. (A8)-(A9) with k0 = 4.05, no bump, delta = -0.7, no floor
    const bool tiny5 = d->model == SPS_MODEL_TINY5;
    wave[k] = (float)lam; k0[k] = tiny5 ? 4.05f : (float)calz_k0(lam); dr[k] = tiny5 ? 0.f : (float)drude_profile(lam); l2r[k] = (float)log2(lam / 5500.0);
  }
  for (int k = 0; k < nw; ++k) {                     // R4: trapezoid weights
    const double lo = d->wave_A[k > 0 ? k - 1 : 0], hi = d->wave_A[k < nw - 1 ? k + 1 : nw - 1];
    dlam[k] = (float)(0.5 * (hi - lo));
  }
  std::vector<float> ssp((size_t)T.K * nwp, 0.f);
  for (int r = 0; r < T.K; ++r) memcpy(&ssp[(size_t)r * nwp], d->ssp + (size_t)r * nw, sizeof(float) * nw);
  std::vector<double> fw_h, ft_h; std::vector<int> foff_h;
  if (!tab) {
    for (int b = 0; b < d->n_band; ++b) {
      const double mu = d->filt_mu_A[b], sg = d->filt_sigma_A[b];
      if (!(sg > 0) || !(mu - 5 * sg > 0)) { sps_set_error("filter %d: need sigma > 0 and mu - 5 sigma > 0", b); delete t; return SPS_EINVAL; }
      T.filt_mu[b] = (float)mu; T.filt_sigma[b] = (float)sg;
      // Eq. (5) PAPER.md:73 at z = 0 on the filter's own grid
      const int nq = 4001; double num = 0, den = 0;
      for (int q = 0; q < nq; ++q) {
        const double lam = mu - 5 * sg + 10 * sg * q / (nq - 1), x = (lam - mu) / sg, w = (q == 0 || q == nq - 1) ? 0.5 : 1.0;
        const double Tq = exp(-0.5 * x * x); num += w * lam * Tq; den += w * Tq;
      }
      T.lam_eff[b] = (float)(num / den);
    }
  } else {
    // tabulated curves: knot records, the uniform index over each band's support, Eq. (5) with every segment integrated
    // exactly (T linear, lambda T quadratic: Simpson)
    const int nk = d->filt_offsets[d->n_band];
    fw_h.assign(d->filt_wave_A, d->filt_wave_A + nk); ft_h.assign(d->filt_trans, d->filt_trans + nk);
    foff_h.assign(d->filt_offsets, d->filt_offsets + d->n_band + 1);
    std::vector<float4> knots(nk);
    std::vector<int> first((size_t)d->n_band * SPS_FTAB_BINS);
    for (int b = 0; b < d->n_band; ++b) {
      const int o = foff_h[b], n = foff_h[b + 1] - o;
      const double* w = &fw_h[o]; const double* tr = &ft_h[o];
      double num = 0, den = 0;
      for (int k = 0; k < n; ++k) {
        const bool last = k == n - 1;
        knots[o + k] = make_float4((float)w[k], (float)tr[k], last ? 0.f : (float)((tr[k + 1] - tr[k]) / (w[k + 1] - w[k])), last ? 3.0e38f : (float)w[k + 1]);
        if (!last) {
          const double h = w[k + 1] - w[k], wm = 0.5 * (w[k] + w[k + 1]), tm = 0.5 * (tr[k] + tr[k + 1]);
          den += h * tm; num += h / 6.0 * (w[k] * tr[k] + 4.0 * wm * tm + w[k + 1] * tr[k + 1]);
        }
      }
      if (!(den > 0)) { sps_set_error("filter %d: zero or negative area", b); delete t; return SPS_EINVAL; }
      T.lam_eff[b] = (float)(num / den);
      T.ft.lo[b] = (float)w[0]; T.ft.hi[b] = (float)w[n - 1]; T.ft.inv_d[b] = (float)(SPS_FTAB_BINS / (w[n - 1] - w[0])); T.ft.last[b] = o + n - 2;
      T.filt_mu[b] = (float)(0.5 * (w[0] + w[n - 1])); T.filt_sigma[b] = (float)(0.1 * (w[n - 1] - w[0]));   // mu +- 5 sigma = the support
      int seg = 0;
      for (int q = 0; q < SPS_FTAB_BINS; ++q) {
        const double left = w[0] + (w[n - 1] - w[0]) * ((double)q - 1e-3) / SPS_FTAB_BINS;     // a little early: fp32 bin rounding
        while (seg < n - 2 && w[seg + 1] <= left) ++seg;
        first[(size_t)b * SPS_FTAB_BINS + q] = o + seg;
      }
    }
    T.ft.knots = upload(knots, st); T.ft.first = upload(first, st);
  }
  {
    // fixed-point band sums of the exact path (sps_exact.cuh): bounds per unit M_star
    double s_bol = 0.0, t_max = 1.0, slope_lam = 0.0;
    for (int r = 0; r < T.K; ++r) {
      double acc = 0.0;
      for (int k = 0; k < nw; ++k) acc += (double)d->ssp[(size_t)r * nw + k] * dlam[k];
      s_bol = std::max(s_bol, acc);
    }
    const double lam_max = d->wave_A[nw - 1];
    if (tab) {
      const int nk = d->filt_offsets[d->n_band];
      for (int k = 0; k < nk; ++k) t_max = std::max(t_max, fabs(d->filt_trans[k]));
      for (int b = 0; b < d->n_band; ++b)
        for (int k = d->filt_offsets[b]; k + 1 < d->filt_offsets[b + 1]; ++k)
          slope_lam = std::max(slope_lam, fabs((d->filt_trans[k + 1] - d->filt_trans[k]) / (d->filt_wave_A[k + 1] - d->filt_wave_A[k])) * lam_max);
    } else {
      for (int b = 0; b < d->n_band; ++b) slope_lam = std::max(slope_lam, lam_max / d->filt_sigma_A[b]);     // |x T'(x)| <= 1 in units of sigma
    }
    T.part_bound = (float)(s_bol * t_max);
    T.part_shift_z = std::min(40, std::max(0, (int)ceil(log2(std::max(slope_lam / t_max, 1.0)))) + 2);
  }
  T.z_min = (float)d->z_min; T.dz = (float)((d->z_max - d->z_min) / (d->n_z - 1)); T.inv_dz = (float)((d->n_z - 1) / (d->z_max - d->z_min));
  const double OL = 1.0 - d->Om, inv_H0 = 977.7922216807891 / d->H0;
  T.t_pref_d = 2.0 * inv_H0 / (3.0 * sqrt(OL)); T.t_arg_d = sqrt(OL / d->Om);
  T.t_pref = (float)T.t_pref_d; T.t_arg = (float)T.t_arg_d;
  T.H0_gyr = (float)(1.0 / inv_H0); T.Om = (float)d->Om; T.OL = (float)OL;
  T.log10_mass_unit = (float)d->log10_mass_unit;
  // t_obs(z) (R11) as piecewise degree-5 polynomials over [z_min, z_max]: interpolation of the closed form at the six
  // Chebyshev nodes of each interval (6 x 6 Vandermonde system in long double)
  T.tz_coef = nullptr; T.tz_n = 0; T.tz_lo = 0.0; T.tz_inv_h = 0.0;
  std::vector<double> tz;
  if (d->z_max > d->z_min) {
    const int N = 256;
    const double h = (d->z_max - d->z_min) / N;
    tz.resize((size_t)N * 6);
    long double un[6];
    for (int k = 0; k < 6; ++k) un[k] = cosl((2 * k + 1) * 3.14159265358979323846264338327950288L / 12.0L);
    for (int i = 0; i < N; ++i) {
      long double A[6][7];
      for (int k = 0; k < 6; ++k) {
        long double pw = 1.0L;
        for (int c = 0; c < 6; ++c) { A[k][c] = pw; pw *= un[k]; }
        const double z = d->z_min + (i + 0.5) * h + 0.5 * h * (double)un[k];
        A[k][6] = (long double)(T.t_pref_d * asinh(T.t_arg_d * pow(1.0 + z, -1.5)));
      }
      for (int c = 0; c < 6; ++c) {                          // Gauss-Jordan with partial pivoting
        int piv = c;
        for (int r = c + 1; r < 6; ++r) if (fabsl(A[r][c]) > fabsl(A[piv][c])) piv = r;
        for (int k = 0; k < 7; ++k) std::swap(A[c][k], A[piv][k]);
        for (int r = 0; r < 6; ++r) {
          if (r == c) continue;
          const long double f = A[r][c] / A[c][c];
          for (int k = c; k < 7; ++k) A[r][k] -= f * A[c][k];
        }
      }
      for (int c = 0; c < 6; ++c) tz[(size_t)i * 6 + c] = (double)(A[c][6] / A[c][c]);
    }
    T.tz_n = N; T.tz_lo = d->z_min; T.tz_inv_h = 1.0 / h;
  }

  std::vector<double> Amid_d(na);
  for (int i = 0; i < na; ++i) Amid_d[i] = 0.5 * (Ae[i] + Ae[i + 1]);
  T.A_edge_d = upload(Ae, st); T.A_mid_d = upload(Amid_d, st);
  std::vector<float2> Ahl(SPS_AGE_PER_LANE * 32, make_float2(1e30f, 0.f));
  for (int i = 0; i <= na && i < (int)Ahl.size(); ++i) { const float hi = (float)Ae[i]; Ahl[i] = make_float2(hi, (float)(Ae[i] - (double)hi)); }
  T.A_edge_hl = upload(Ahl, st);
  if (!tz.empty()) T.tz_coef = upload(tz, st);
  T.A_edge = upload(A_edge, st); T.A_mid = upload(A_mid, st); T.A_half = upload(A_half, st); T.e_edge = upload(e_edge, st);
  T.g_mid = upload(g_mid, st); T.la9 = upload(la9, st); T.wave = upload(wave, st); T.dlam = upload(dlam, st); T.k0 = upload(k0, st);
  T.drude = upload(dr, st); T.l2r = upload(l2r, st); T.ssp = upload(ssp, st);
  float* cssp = nullptr;
  const size_t cs_n = (size_t)T.n_z * 2 * T.n_age * T.cs_stride;
  std::vector<double> wave_h(d->wave_A, d->wave_A + nw), dlam_h(nw);
  for (int k = 0; k < nw; ++k) {
    const double lo = d->wave_A[k > 0 ? k - 1 : 0], hi = d->wave_A[k < nw - 1 ? k + 1 : nw - 1];
    dlam_h[k] = 0.5 * (hi - lo);
  }
  double* wave_dd = upload(wave_h, st); double* dlam_dd = upload(dlam_h, st);
  if (st == SPS_OK && cudaMalloc(&cssp, cs_n * sizeof(float)) != cudaSuccess) { st = SPS_ENOMEM; sps_set_error("cudaMalloc c_SSP failed"); }
  if (st == SPS_OK) {
    cudaMemset(cssp, 0, cs_n * sizeof(float));
    T.cssp = cssp;
    const int64_t warps = (int64_t)T.n_z * T.K;
    double* fw_d = tab ? upload(fw_h, st) : nullptr; double* ft_d = tab ? upload(ft_h, st) : nullptr; int* foff_d = tab ? upload(foff_h, st) : nullptr;
    if (st == SPS_OK) {
      cssp_build_kernel<<<(unsigned)((warps * 32 + 255) / 256), 256>>>(T, wave_dd, dlam_dd, d->z_min, (d->z_max - d->z_min) / (d->n_z - 1), fw_d, ft_d, foff_d, cssp);
      sps_count_launch();
      st = sps_check_cuda(cudaDeviceSynchronize(), "c_SSP build");
    }
    if (fw_d) cudaFree(fw_d); if (ft_d) cudaFree(ft_d); if (foff_d) cudaFree(foff_d);
  }
  if (wave_dd) cudaFree(wave_dd);
  if (dlam_dd) cudaFree(dlam_dd);
  if (st == SPS_OK && d->dlogZ_dlogage != 0.0 && d->n_age * d->n_Z > 2048) { sps_set_error("non-separable weights: n_age n_Z <= 2048"); st = SPS_ESHAPE; }
  if (st == SPS_OK) st = approx_contract_setup(T);
  if (st == SPS_OK) st = sps_approx_tc_setup(t);
  if (st == SPS_OK) st = sps_exact_setup(t, d->exact_precision);
  if (st != SPS_OK) { sps_destroy_table(t); return st; }
  *out = t;
  return SPS_OK;
}

extern "C" sps_status sps_destroy_table(sps_table* t) {
  if (!t) return SPS_OK;
  TableDev& T = t->dev;
  cudaDeviceSynchronize();
  const void* ptrs[] = {T.tz_coef, T.A_edge_d, T.A_mid_d, T.A_edge_hl, T.A_edge, T.A_mid, T.A_half, T.e_edge, T.g_mid, T.wave, T.dlam, T.k0, T.drude, T.l2r, T.ssp, T.cssp,
                        T.gauss, T.ft.knots, T.ft.first, T.la9};
  for (const void* p : ptrs) if (p) cudaFree(const_cast<void*>(p));
  sps_exact_teardown(t);
  sps_approx_tc_teardown(t);
  for (auto& kv : t->ws) sps_free_workspace(kv.second);
  t->ws.clear();
  sps_pool_release_unused();
  if (t->own_stream) cudaStreamDestroy(t->own_stream);
  for (cudaStream_t a : t->aux_stream) if (a) cudaStreamDestroy(a);
  delete t;
  return SPS_OK;
}

extern "C" sps_status sps_table_cssp(const sps_table* t, float* host) {
  if (!t || !host || !t->dev.cssp) { sps_set_error("sps_table_cssp: null argument or a table without photometry"); return SPS_EINVAL; }
  const TableDev& T = t->dev;
  const int E = T.n_Z * T.n_band;
  std::vector<float> tmp((size_t)T.n_z * 2 * T.n_age * T.cs_stride);
  sps_status st = sps_check_cuda(cudaMemcpy(tmp.data(), T.cssp, tmp.size() * sizeof(float), cudaMemcpyDeviceToHost), "c_SSP D2H");
  if (st != SPS_OK) return st;
  for (int64_t t2 = 0; t2 < T.n_z; ++t2)
    for (int64_t i = 0; i < T.n_age; ++i)
      memcpy(host + (t2 * T.n_age + i) * E, &tmp[((t2 * 2) * T.n_age + i) * T.cs_stride], sizeof(float) * E);
  return SPS_OK;
}
