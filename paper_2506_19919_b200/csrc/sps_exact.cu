// sps_exact.cu -- exact photometry path (Eq. 4) and its reverse pass.
//   W[r,ij]   = Mn a_i m_j                                   (a5, Eq. 2 + M_star)
//   S[r,k]    = sum_ij W[r,ij] L[ij,k]                       (a6: the dense contraction)
//   flux[r,b] = sum_k S[r,k] F_att(lam_k|r) T_b(lam_k (1+z_r)) dlam_k      (a8 + filters, fused epilogue)
//   reverse:  SEDbar[r,k] = F_att dlam_k sum_b g_b T_b ;  Wbar[r,ij] = sum_k SEDbar[r,k] L[ij,k]
// This file holds the row-wise glue kernels and a plain fp32 SIMT version of the two contractions
// (used as the in-library cross-check of the tcgen05 kernels in sps_exact_tc.cu and for tiny tables).
#include "sps_exact.cuh"

// ---- W = Mn a (x) m ---------------------------------------------------------------------------
__global__ void exact_weights_kernel(TableDev T, int64_t n, const int* __restrict__ rows, RowBuffers B, float* __restrict__ W, int ldw) {
  const int64_t r = blockIdx.x;
  const int64_t row = rows ? rows[r] : r;
  const float Mn = B.sc[row].Mn;
  __shared__ float mt_s[SPS_MAX_AGE * SPS_MAX_Z];            // non-separable weights (R26): the MDF of every age bin
  const bool nonsep = T.agez_gamma != 0.f;
  if (nonsep && threadIdx.x < T.n_age) {
    float d1[SPS_MAX_Z], d2[SPS_MAX_Z];
    mdf_row(T, B.sc[row].pad1 + T.agez_gamma * T.la9[threadIdx.x], B.sc[row].pad2, mt_s + threadIdx.x * SPS_MAX_Z, d1, d2);
  }
  __syncthreads();
  for (int e = threadIdx.x; e < ldw; e += blockDim.x) {
    float v = 0.f;
    if (e < T.K) {
      const int i = e / T.n_Z, j = e - i * T.n_Z;
      v = Mn * B.a[row * ROW_A_STRIDE + i] * (nonsep ? mt_s[i * SPS_MAX_Z + j] : B.m[row * ROW_M_STRIDE + j]);
    }
    W[r * ldw + e] = v;
  }
}

// per-(row, wavelength) dust factor (Eq. A8-A9 with the tabulated k0, Drude, log2(lam/lam_V))
__device__ __forceinline__ void dust_tab(float k0, float dr, float l2r, float AV, float delta, float Ffl,
                                         float& F, float& F_av, float& F_del, float& F_fl) {
  const float pw = exp2f(delta * l2r);
  const float Eb = 0.85f - 1.9f * delta;
  const float br = k0 * pw + Eb * dr;
  float A = AV * (1.f / 4.05f) * br;
  float A_av = br * (1.f / 4.05f);
  float A_del = AV * (1.f / 4.05f) * (k0 * pw * l2r * LN2F - 1.9f * dr);
  if (!(A > 0.f)) { A = 0.f; A_av = 0.f; A_del = 0.f; }
  const float Tt = exp2f(-0.4f * 3.321928094887362f * A);
  const float dF = -(1.f - Ffl) * 0.4f * LN10F * Tt;
  F = Ffl + (1.f - Ffl) * Tt; F_av = dF * A_av; F_del = dF * A_del; F_fl = 1.f - Tt;
}

// T_b(lam_obs) and dT_b/dlam_obs: Gaussian truncated at 5 sigma (R4) or tabulated curve
__device__ __forceinline__ void filter_eval(const TableDev& T, int b, float lam_obs, float& Tb, float& dTb) {
  if (T.filt_tab) { filter_tab_eval(T.ft, b, lam_obs, Tb, dTb); return; }
  const float x = (lam_obs - T.filt_mu[b]) / T.filt_sigma[b];
  Tb = 0.f; dTb = 0.f;
  if (fabsf(x) <= 5.f) { Tb = expf(-0.5f * x * x); dTb = -Tb * x / T.filt_sigma[b]; }
}

// ---- forward SIMT: 64 rows x 64 wavelengths per CTA, 4x4 per thread ---------------------------------
#define XB_M 64
#define XB_N 64
#define XB_K 16
__global__ void __launch_bounds__(256) exact_fwd_simt_kernel(TableDev T, int64_t n, const int* __restrict__ rows, RowBuffers B,
                                                             const float* __restrict__ W, int ldw, long long* __restrict__ part /*[n][5][16]*/) {
  __shared__ float As[XB_K][XB_M + 4], Bs[XB_K][XB_N + 4];
  __shared__ float red[5][SPS_MAX_BAND][XB_M + 1];
  const int tx = threadIdx.x & 15, ty = threadIdx.x >> 4;          // tx: wavelength group, ty: row group
  const int64_t r0 = (int64_t)blockIdx.y * XB_M; const int k0 = blockIdx.x * XB_N;
  float acc[4][4] = {};
  for (int kk = 0; kk < ldw; kk += XB_K) {
    for (int e = threadIdx.x; e < XB_M * XB_K; e += 256) {
      const int m = e / XB_K, k = e % XB_K; const int64_t r = r0 + m;
      As[k][m] = (r < n && kk + k < ldw) ? W[r * ldw + kk + k] : 0.f;
    }
    for (int e = threadIdx.x; e < XB_K * XB_N; e += 256) {
      const int k = e / XB_N, c = e % XB_N;
      Bs[k][c] = (kk + k < T.K) ? T.ssp[(int64_t)(kk + k) * T.n_wave_pad + k0 + c] : 0.f;
    }
    __syncthreads();
#pragma unroll
    for (int k = 0; k < XB_K; ++k) {
      float a[4], b[4];
#pragma unroll
      for (int i = 0; i < 4; ++i) { a[i] = As[k][ty * 4 + i]; b[i] = Bs[k][tx * 4 + i]; }
#pragma unroll
      for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) acc[i][j] += a[i] * b[j];
    }
    __syncthreads();
  }
  // epilogue: dust, filters, partial band sums per row over this CTA's 64 wavelengths
  for (int q = threadIdx.x; q < 5 * SPS_MAX_BAND * (XB_M + 1); q += 256) (&red[0][0][0])[q] = 0.f;
  __syncthreads();
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const int64_t r = r0 + ty * 4 + i;
    if (r >= n) continue;
    const int64_t row = rows ? rows[r] : r;
    const RowScalars sc = B.sc[row];
    const float zp = 1.f + sc.z;
    float s[5][SPS_MAX_BAND];
#pragma unroll
    for (int b = 0; b < SPS_MAX_BAND; ++b) s[0][b] = s[1][b] = s[2][b] = s[3][b] = s[4][b] = 0.f;
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      const int k = k0 + tx * 4 + j;
      float F, F_av, F_del, F_fl;
      dust_tab(T.k0[k], T.drude[k], T.l2r[k], sc.AV, sc.delta, sc.Ffloor, F, F_av, F_del, F_fl);
      const float lam = T.wave[k], Sd = acc[i][j] * T.dlam[k];
      for (int b = 0; b < T.n_band; ++b) {
        float Tv, dTv;
        filter_eval(T, b, lam * zp, Tv, dTv);
        if (Tv != 0.f || dTv != 0.f) {
          const float Tb = Tv * Sd;
          s[0][b] += Tb * F; s[1][b] += Tb * F_av; s[2][b] += Tb * F_del; s[3][b] += Tb * F_fl;
          s[4][b] += dTv * Sd * F * lam;                          // d/dz of T_b(lam (1+z))
        }
      }
    }
    for (int b = 0; b < T.n_band; ++b)
#pragma unroll
      for (int c = 0; c < 5; ++c) if (s[c][b] != 0.f) atomicAdd(&red[c][b][ty * 4 + i], s[c][b]);
  }
  __syncthreads();
  for (int q = threadIdx.x; q < 5 * SPS_MAX_BAND * XB_M; q += 256) {
    const int m = q % XB_M, cb = q / XB_M, c = cb / SPS_MAX_BAND, b = cb % SPS_MAX_BAND;
    const int64_t r = r0 + m;
    const float v = red[c][b][m];
    if (r < n && b < T.n_band && v != 0.f) {
      const int shift = c == 0 ? PART_SHIFT_FLUX : (c == 1 ? PART_SHIFT_AV : (c == 2 ? PART_SHIFT_DELTA : (c == 3 ? PART_SHIFT_FFLOOR : T.part_shift_z)));
      part_add(&part[(r * 5 + c) * SPS_MAX_BAND + b], v, part_scale(B.sc[rows ? rows[r] : r].Mn, T.part_bound, shift));
    }
  }
}

// ---- between the two contractions: flux -> likelihood -> g_b, and the direct (dust, z, Mn) bars ---------
__global__ void exact_mid_kernel(TableDev T, int64_t n, const int* __restrict__ rows, const int* __restrict__ gal_of_row,
                                 const float* __restrict__ obs_flux, const float* __restrict__ obs_sigma,
                                 const float* __restrict__ flux_bar, bool want_grad, RowBuffers B,
                                 const long long* __restrict__ part, float* __restrict__ gbuf) {
  const int64_t r = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  if (r >= n) return;
  const int l = threadIdx.x & 31;
  const int64_t row = rows ? rows[r] : r;
  const bool isb = l < T.n_band;
  const long long* p = part + r * 5 * SPS_MAX_BAND;
  const float Mn = B.sc[row].Mn;
  float flux = 0.f, g = 0.f, chi2 = 0.f, p_av = 0.f, p_de = 0.f, p_fl = 0.f, p_z = 0.f;
  if (isb) {
    flux = part_read(p + l, part_scale(Mn, T.part_bound, PART_SHIFT_FLUX));
    p_av = part_read(p + 1 * SPS_MAX_BAND + l, part_scale(Mn, T.part_bound, PART_SHIFT_AV));
    p_de = part_read(p + 2 * SPS_MAX_BAND + l, part_scale(Mn, T.part_bound, PART_SHIFT_DELTA));
    p_fl = part_read(p + 3 * SPS_MAX_BAND + l, part_scale(Mn, T.part_bound, PART_SHIFT_FFLOOR));
    p_z = part_read(p + 4 * SPS_MAX_BAND + l, part_scale(Mn, T.part_bound, T.part_shift_z));
    B.flux[row * SPS_MAX_BAND + l] = flux;
    if (flux_bar) g = flux_bar[row * T.n_band + l];
    else {
      const int64_t gal = gal_of_row ? gal_of_row[row] : row;
      const float d = obs_flux[gal * T.n_band + l], sg = obs_sigma[gal * T.n_band + l];
      const float rr = (flux - d) / sg;
      chi2 = rr * rr; g = -rr / sg;
    }
  }
  if (l < SPS_MAX_BAND) gbuf[r * SPS_MAX_BAND + l] = isb ? g : 0.f;
  chi2 = warp_sum(chi2);
  const float mn_bar = warp_sum(isb ? g * flux : 0.f) / Mn;
  const float av = warp_sum(g * p_av);
  const float de = warp_sum(g * p_de);
  const float fl = warp_sum(g * p_fl);
  const float zb = warp_sum(g * p_z);
  if (l == 0) {
    RowScalars* sc = &B.sc[row];
    sc->logp_like = -0.5f * chi2;
    if (want_grad) { sc->Mn_bar = mn_bar; sc->AV_bar = av; sc->delta_bar = de; sc->Ffloor_bar = fl; sc->z_bar = zb; }
  }
}

// ---- reverse SIMT: Wbar[r,ij] = sum_k SEDbar[r,k] L[ij,k], SEDbar generated on the fly -----------------
__global__ void __launch_bounds__(256) exact_bwd_simt_kernel(TableDev T, int64_t n, const int* __restrict__ rows, RowBuffers B,
                                                             const float* __restrict__ gbuf, float* __restrict__ Wbar, int ldw) {
  __shared__ float As[XB_K][XB_M + 4], Bs[XB_K][XB_N + 4];
  __shared__ float g_s[XB_M][SPS_MAX_BAND];
  __shared__ float sc_s[XB_M][4];                                  // 1+z, AV, delta, Ffloor
  const int tx = threadIdx.x & 15, ty = threadIdx.x >> 4;
  const int64_t r0 = (int64_t)blockIdx.y * XB_M; const int c0 = blockIdx.x * XB_N;   // c: ij index
  for (int e = threadIdx.x; e < XB_M * SPS_MAX_BAND; e += 256) {
    const int m = e / SPS_MAX_BAND, b = e % SPS_MAX_BAND;
    g_s[m][b] = (r0 + m < n) ? gbuf[(r0 + m) * SPS_MAX_BAND + b] : 0.f;
  }
  for (int m = threadIdx.x; m < XB_M; m += 256) {
    if (r0 + m < n) {
      const RowScalars sc = B.sc[rows ? rows[r0 + m] : r0 + m];
      sc_s[m][0] = 1.f + sc.z; sc_s[m][1] = sc.AV; sc_s[m][2] = sc.delta; sc_s[m][3] = sc.Ffloor;
    } else { sc_s[m][0] = 1.f; sc_s[m][1] = sc_s[m][2] = 0.f; sc_s[m][3] = 1.f; }
  }
  __syncthreads();
  float acc[4][4] = {};
  for (int kk = 0; kk < T.n_wave_pad; kk += XB_K) {
    for (int e = threadIdx.x; e < XB_M * XB_K; e += 256) {
      const int m = e / XB_K, k = e % XB_K, kg = kk + k;
      float v = 0.f;
      const float dl = T.dlam[kg];
      if (dl > 0.f) {
        const float lam = T.wave[kg] * sc_s[m][0];
        float tsum = 0.f;
        for (int b = 0; b < T.n_band; ++b) {
          float Tv, dTv;
          filter_eval(T, b, lam, Tv, dTv);
          tsum += g_s[m][b] * Tv;
        }
        if (tsum != 0.f) {
          float F, a1, a2, a3;
          dust_tab(T.k0[kg], T.drude[kg], T.l2r[kg], sc_s[m][1], sc_s[m][2], sc_s[m][3], F, a1, a2, a3);
          v = F * dl * tsum;
        }
      }
      As[k][m] = v;
    }
    for (int e = threadIdx.x; e < XB_K * XB_N; e += 256) {
      const int c = e / XB_K, k = e % XB_K;
      Bs[k][c] = (c0 + c < T.K) ? T.ssp[(int64_t)(c0 + c) * T.n_wave_pad + kk + k] : 0.f;
    }
    __syncthreads();
#pragma unroll
    for (int k = 0; k < XB_K; ++k) {
      float a[4], b[4];
#pragma unroll
      for (int i = 0; i < 4; ++i) { a[i] = As[k][ty * 4 + i]; b[i] = Bs[k][tx * 4 + i]; }
#pragma unroll
      for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) acc[i][j] += a[i] * b[j];
    }
    __syncthreads();
  }
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const int64_t r = r0 + ty * 4 + i;
    if (r >= n) continue;
#pragma unroll
    for (int j = 0; j < 4; ++j) { const int c = c0 + tx * 4 + j; if (c < ldw) Wbar[r * ldw + c] = acc[i][j]; }
  }
}

// ---- a_bar_i = Mn sum_j Wbar_ij m_j ;  m_bar_j = Mn sum_i Wbar_ij a_i -------------------------------------
__global__ void exact_final_kernel(TableDev T, int64_t n, const int* __restrict__ rows, RowBuffers B, const float* __restrict__ Wbar, int ldw) {
  const int64_t r = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  if (r >= n) return;
  const int l = threadIdx.x & 31;
  const int64_t row = rows ? rows[r] : r;
  const float Mn = B.sc[row].Mn;
  const float* wb = Wbar + r * ldw;
  if (T.agez_gamma != 0.f) {
    // non-separable weights (R26): w_ij = Mn a_i m_ij with an MDF per age bin; the metallicity parameters collect their
    // bars through every bin, handed to the epilogue in the row's scalars (m_bar is zero)
    const float lz = B.sc[row].pad1, slz = B.sc[row].pad2;
    float lz_bar = 0.f, slz_bar = 0.f;
    for (int i0 = 0; i0 < ROW_A_STRIDE; i0 += 32) {
      const int i = i0 + l;
      float ab = 0.f;
      if (i < T.n_age) {
        float m[SPS_MAX_Z], d_mu[SPS_MAX_Z], d_s[SPS_MAX_Z];
        mdf_row(T, lz + T.agez_gamma * T.la9[i], slz, m, d_mu, d_s);
        const float ai = B.a[row * ROW_A_STRIDE + i];
        for (int j = 0; j < T.n_Z; ++j) { const float w = wb[i * T.n_Z + j]; ab += w * m[j]; lz_bar += w * ai * d_mu[j]; slz_bar += w * ai * d_s[j]; }
      }
      B.a_bar[row * ROW_A_STRIDE + i] = Mn * ab;
    }
    lz_bar = warp_sum(lz_bar); slz_bar = warp_sum(slz_bar);
    if (l < ROW_M_STRIDE) B.m_bar[row * ROW_M_STRIDE + l] = 0.f;
    if (l == 0) { B.sc[row].pad1 = Mn * lz_bar; B.sc[row].pad2 = Mn * slz_bar; }
    return;
  }
  float mb[SPS_MAX_Z];
#pragma unroll
  for (int j = 0; j < SPS_MAX_Z; ++j) mb[j] = 0.f;
  for (int i0 = 0; i0 < ROW_A_STRIDE; i0 += 32) {
    const int i = i0 + l;
    float ab = 0.f;
    if (i < T.n_age) {
      const float ai = B.a[row * ROW_A_STRIDE + i];
#pragma unroll
      for (int j = 0; j < SPS_MAX_Z; ++j) if (j < T.n_Z) { const float w = wb[i * T.n_Z + j]; ab += w * B.m[row * ROW_M_STRIDE + j]; mb[j] += w * ai; }
    }
    B.a_bar[row * ROW_A_STRIDE + i] = Mn * ab;
  }
#pragma unroll
  for (int j = 0; j < SPS_MAX_Z; ++j) { const float s = warp_sum(mb[j]); if (l == j) B.m_bar[row * ROW_M_STRIDE + j] = Mn * s; }
}

// ---- order the rows of a call by redshift (counting sort over ZSORT_BINS uniform bins of the table's z range) --------
// The tensor-core kernels tile rows in groups of 128; rows of similar z share the wavelength range under the filters.
#define ZSORT_BINS 1024
__device__ __forceinline__ int zsort_bin(const TableDev& T, float z) {
  const float u = (z - T.z_min) / (T.dz * (float)(T.n_z - 1));
  return min(max((int)(u * ZSORT_BINS), 0), ZSORT_BINS - 1);
}
__global__ void zsort_hist_kernel(TableDev T, int64_t n, const int* __restrict__ rows, RowBuffers B, int* __restrict__ hist) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) atomicAdd(&hist[zsort_bin(T, B.sc[rows ? rows[i] : i].z)], 1);
}
__global__ void __launch_bounds__(ZSORT_BINS) zsort_scan_kernel(int* __restrict__ hist) {      // hist -> exclusive offsets, in place (+ copy)
  __shared__ int s[ZSORT_BINS];
  const int t = threadIdx.x;
  const int v = hist[t];
  s[t] = v;
  __syncthreads();
  for (int o = 1; o < ZSORT_BINS; o <<= 1) { const int a = (t >= o) ? s[t - o] : 0; __syncthreads(); s[t] += a; __syncthreads(); }
  hist[ZSORT_BINS + t] = s[t] - v;
}
__global__ void zsort_scatter_kernel(TableDev T, int64_t n, const int* __restrict__ rows, RowBuffers B, int* __restrict__ cursor, int* __restrict__ out) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const int row = rows ? rows[i] : (int)i;
  out[atomicAdd(&cursor[zsort_bin(T, B.sc[row].z)], 1)] = row;
}

// ---- host side ----------------------------------------------------------------------------------------

sps_status sps_exact_setup(sps_table* t, int precision) {
  ExactState* X = new ExactState();
  memset(X, 0, sizeof(*X));
  X->ldw = (t->dev.K + 31) / 32 * 32;
  t->exact = X;
  return sps_exact_tc_setup(t, precision);
}

void sps_exact_free_scratch(ExactScratch& X) {
  sps_exact_tc_free_scratch(X);
  void* ptrs[] = {X.W, X.Wbar, X.part, X.gbuf, X.sorted, X.zhist};
  for (void* p : ptrs) if (p) cudaFree(p);
  X.W = X.Wbar = X.gbuf = nullptr; X.part = nullptr; X.sorted = X.zhist = nullptr; X.cap = 0;
}

void sps_exact_teardown(sps_table* t) {
  if (!t->exact) return;
  sps_exact_tc_teardown(t);
  delete t->exact; t->exact = nullptr;
}

static sps_status exact_ensure(const sps_table* t, ExactScratch& X, int64_t n, cudaStream_t s) {
  const int ldw = t->exact->ldw;
  const int64_t need = (n + 127) / 128 * 128;                      // whole row tiles for the tensor-core kernels
  if (X.cap >= need) return SPS_OK;
  cudaStreamSynchronize(s);
  sps_exact_free_scratch(X);
  cudaError_t e = cudaMalloc(&X.W, need * ldw * sizeof(float));
  if (e == cudaSuccess) e = cudaMalloc(&X.Wbar, need * ldw * sizeof(float));
  if (e == cudaSuccess) e = cudaMalloc(&X.part, need * 5 * SPS_MAX_BAND * sizeof(long long));
  if (e == cudaSuccess) e = cudaMalloc(&X.gbuf, need * SPS_MAX_BAND * sizeof(float));
  if (e == cudaSuccess) e = cudaMalloc(&X.sorted, need * sizeof(int));
  if (e == cudaSuccess) e = cudaMalloc(&X.zhist, 2 * ZSORT_BINS * sizeof(int));
  if (e != cudaSuccess) { sps_exact_free_scratch(X); return sps_check_cuda(e, "exact-path scratch allocation"); }
  cudaMemsetAsync(X.W, 0, need * ldw * sizeof(float), s);
  cudaMemsetAsync(X.gbuf, 0, need * SPS_MAX_BAND * sizeof(float), s);
  X.cap = need;
  return sps_exact_tc_ensure(t, X, need);
}

sps_status sps_exact_contract(const sps_table* t, Workspace& ws, int64_t n, const int* rows, const int* gal_of_row, const float* obs_flux,
                              const float* obs_sigma, const float* flux_bar, bool want_grad, cudaStream_t s) {
  ExactScratch& X = ws.x;
  const TableDev& T = t->dev;
  const int ldw = t->exact->ldw;
  sps_status st = exact_ensure(t, X, n, s); if (st != SPS_OK) return st;
  const bool tc = t->exact->use_tc && !sps_option(SPS_OPT_EXACT_SIMT);
  if (tc) {                                                        // redshift-ordered row list for this call
    cudaMemsetAsync(X.zhist, 0, 2 * ZSORT_BINS * sizeof(int), s);
    const unsigned nb = (unsigned)((n + 255) / 256);
    zsort_hist_kernel<<<nb, 256, 0, s>>>(T, n, rows, ws.rows, X.zhist);
    zsort_scan_kernel<<<1, ZSORT_BINS, 0, s>>>(X.zhist);
    zsort_scatter_kernel<<<nb, 256, 0, s>>>(T, n, rows, ws.rows, X.zhist + ZSORT_BINS, X.sorted);
    sps_count_launch(3);
    rows = X.sorted;
  }
  if (!tc) { exact_weights_kernel<<<(unsigned)n, 128, 0, s>>>(T, n, rows, ws.rows, X.W, ldw); sps_count_launch(); }
  cudaMemsetAsync(X.part, 0, n * 5 * SPS_MAX_BAND * sizeof(long long), s);
  if (tc) st = sps_exact_tc_forward(t, ws, n, rows, s);          // (brackets its GEMM kernel for sps_profile itself)
  else {
    dim3 grid(T.n_wave_pad / XB_N, (unsigned)((n + XB_M - 1) / XB_M));
    sps_prof_begin(SPS_K_EXACT_FWD, s);
    exact_fwd_simt_kernel<<<grid, 256, 0, s>>>(T, n, rows, ws.rows, X.W, ldw, X.part); sps_count_launch();
    sps_prof_end(SPS_K_EXACT_FWD, s);
  }
  if (st != SPS_OK) return st;
  const unsigned wb = (unsigned)((n * 32 + 255) / 256);
  exact_mid_kernel<<<wb, 256, 0, s>>>(T, n, rows, gal_of_row, obs_flux, obs_sigma, flux_bar, want_grad, ws.rows, X.part, X.gbuf);
  sps_count_launch();
  if (!want_grad) return SPS_OK;
  if (tc) st = sps_exact_tc_backward(t, ws, n, rows, s);
  else {
    dim3 grid((ldw + XB_N - 1) / XB_N, (unsigned)((n + XB_M - 1) / XB_M));
    sps_prof_begin(SPS_K_EXACT_BWD, s);
    exact_bwd_simt_kernel<<<grid, 256, 0, s>>>(T, n, rows, ws.rows, X.gbuf, X.Wbar, ldw); sps_count_launch();
    sps_prof_end(SPS_K_EXACT_BWD, s);
  }
  if (st != SPS_OK) return st;
  exact_final_kernel<<<wb, 256, 0, s>>>(T, n, rows, ws.rows, X.Wbar, ldw); sps_count_launch();
  return SPS_OK;
}
