// sps_kernels.cu -- prologue (a0-a5), approximate-photometry contraction (a7, a9, a10) and
// epilogue (reverse of a0-a5 + prior) kernels.
#include <algorithm>
#include <cstddef>
#include "sps_rows.cuh"

#define WARPS_PER_BLOCK 8                       // rows per block of the small row kernels
#ifndef PRO_WARPS
#define PRO_WARPS 16                            // rows (warps) per prologue block
#endif
#ifndef EPI_WARPS_PER_BLOCK
#define EPI_WARPS_PER_BLOCK 4                   // rows (warps) per epilogue block
#endif
#ifndef PRO_MIN_BLOCKS
#define PRO_MIN_BLOCKS 2                        // resident blocks per SM the prologue / epilogue are compiled for
#endif
#ifndef EPI_MIN_BLOCKS
#define EPI_MIN_BLOCKS 8
#endif

// ---------------------------------------------------------------------------------------------
// Forward model of one row (one warp per parameter row): everything a0-a5 needs, held per lane.
// ---------------------------------------------------------------------------------------------
struct RowFwd {
  float th[SPS_NDIM];
  double t_obs_d, z_d;
  float dt_dz, Msum, Mf;
  AgeQuad Q;
  BurstQuad Bq;
  float m, dm_lz, dm_s;
};

template <bool WANT_GRAD>
__device__ __forceinline__ void row_forward(const TableDev& T, const PriorView& P, const float* __restrict__ row,
                                            bool unbounded, RowFwd& R) {
  load_params(row, unbounded, P, R.th, R.z_d);
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

// a0-a5.  With store_part the per-bin masses dM_i and their partials with respect to (tau, alpha, beta, t_obs) are
// kept in B.part for the epilogue, which then has no quadrature to redo.  One instantiation serves forward-only and
// gradient calls (the partials are computed either way), so that both give bit-identical weights and fluxes.
// Compiled for 48 resident warps per SM (40 registers, ~170 bytes of spills) rather than 32 (60 registers, none): measured
// 82.6 -> 77.3 us at 40,000 rows; 64 warps (32 registers) and 256-thread blocks at the same occupancy are slower.
// PW = rows (warps) per block: 16 when the kernel has the SMs to itself; 8 when the sampler overlaps two row groups, so
// that a block fits in the registers the persistent contraction CTA of the other group leaves free on an SM.
template <int PW>
__global__ void __launch_bounds__(32 * PW, 48 / PW)
prologue_kernel(TableDev T, PriorDev P, const float* __restrict__ theta, int64_t n, bool unbounded, bool store_part,
                const int* __restrict__ rows, RowBuffers B, int* __restrict__ hist) {
  constexpr bool WANT_GRAD = true;
  __shared__ float s_prior[7 * SPS_NDIM];
  const PriorView PV = stage_prior(P, s_prior);
  pdl_wait();                                                // theta, the z-cell counts and the row buffers belong to the kernels before
  const int64_t r = (int64_t)blockIdx.x * PW + (threadIdx.x >> 5);
  if (r >= n) return;
  const int64_t row = rows ? rows[r] : r;
  const int l = lane_id();
  RowFwd R;
  row_forward<WANT_GRAD>(T, PV, theta + row * SPS_NDIM, unbounded, R);
  const float Fb = R.th[4], inv_M = 1.f / R.Msum;
#pragma unroll
  for (int q = 0; q < SPS_AGE_PER_LANE; ++q) {
    const int i = l + 32 * q;
    B.a[row * ROW_A_STRIDE + i] = (i < T.n_age) ? (1.f - Fb) * R.Q.dM[q] * inv_M + Fb * R.Bq.P[q] : 0.f;  // Eq. (A6)
    if (store_part) {
      float* p = B.part + row * (ROW_PARTS * ROW_A_STRIDE) + i;
      p[0] = R.Q.dM[q]; p[ROW_A_STRIDE] = R.Q.g_tau[q]; p[2 * ROW_A_STRIDE] = R.Q.g_al[q];
      p[3 * ROW_A_STRIDE] = R.Q.g_be[q]; p[4 * ROW_A_STRIDE] = R.Q.g_t[q];
    }
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
    sc.Msum = R.Msum; sc.pad1 = R.th[7]; sc.pad2 = R.th[8];       // logZ, sigma_logZ for the non-separable contraction (R26)
    B.sc[row] = sc;
    if (hist) {                                             // z-cell histogram (and row list) for the approximate path's row grouping
      const int pos = atomicAdd(&hist[sc.zbin], 1);
      if (B.cell_list) B.cell_list[(int64_t)sc.zbin * B.cell_cap + pos] = (int)row;
    }
  }
}

// ---------------------------------------------------------------------------------------------
// Grouping of the rows of a call by z cell (counting sort; the histogram is taken by the prologue): rows of one cell share the two c_SSP arrays c_t, D_t
// (PAPER.md:87), so a CTA stages them in shared memory once for up to AC_ROWS_PER_CTA rows.
// bins[0][.] histogram, bins[1][.] first position of each cell in `order`, bins[2][.] first CTA of each cell,
// bins[3][.] scatter cursors.
// ---------------------------------------------------------------------------------------------
#ifndef AC_WARPS
#define AC_WARPS 16                              // warps per CTA
#endif
#ifndef AC_R
#define AC_R 4                                    // rows per warp, register-blocked (4 or 8)
#endif
#define AC_ROWS_PER_CTA (AC_WARPS * AC_R)

__global__ void __launch_bounds__(1024) approx_plan_kernel(int nb, int rows_per_item, int* __restrict__ bins) {
  __shared__ int s_rows[1024], s_ctas[1024];
  const int stride = nb + 2;
  int* hist = bins; int* row_start = bins + stride; int* cta_start = bins + 2 * stride; int* cursor = bins + 3 * stride;
  const int t = threadIdx.x;
  int carry_r = 0, carry_c = 0;
  for (int base = 0; base < nb; base += 1024) {
    const int b = base + t;
    const int cnt = b < nb ? hist[b] : 0, ctas = (cnt + rows_per_item - 1) / rows_per_item;
    s_rows[t] = cnt; s_ctas[t] = ctas;
    __syncthreads();
    for (int o = 1; o < 1024; o <<= 1) {
      const int a = t >= o ? s_rows[t - o] : 0, c = t >= o ? s_ctas[t - o] : 0;
      __syncthreads();
      s_rows[t] += a; s_ctas[t] += c;
      __syncthreads();
    }
    if (b < nb) { row_start[b] = carry_r + s_rows[t] - cnt; cursor[b] = carry_r + s_rows[t] - cnt; cta_start[b] = carry_c + s_ctas[t] - ctas; }
    carry_r += s_rows[1023]; carry_c += s_ctas[1023];
    __syncthreads();
  }
  if (t == 0) { row_start[nb] = carry_r; cta_start[nb] = carry_c; }
}
__global__ void approx_scatter_kernel(int64_t n, const int* __restrict__ rows, RowBuffers B, int* __restrict__ cursor, int* __restrict__ order) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  const int lane = threadIdx.x & 31;
  int row = -1, cell = -1 - lane;                            // idle lanes get distinct dummy keys
  if (i < n) { row = rows ? rows[i] : (int)i; cell = B.sc[row].zbin; }
  // chains of one galaxy sit in consecutive rows and mostly in one cell: one atomic per distinct cell per warp
  const unsigned peers = __match_any_sync(FULL_MASK, cell);
  const int leader = __ffs(peers) - 1;
  int base = 0;
  if (lane == leader && cell >= 0) base = atomicAdd(&cursor[cell], __popc(peers));
  base = __shfl_sync(FULL_MASK, base, leader);
  if (cell >= 0) order[base + __popc(peers & ((1u << lane) - 1u))] = row;
}

// The same with the cell offsets computed in place (n_z - 1 <= 1024): every block scans the histogram itself (4 cells per
// thread), block 0 publishes the row / item offsets for the contraction kernel, and the scatter cursors start at zero
// (cleared together with the histogram before the prologue).  One launch instead of two.
__global__ void __launch_bounds__(256) approx_scan_scatter_kernel(int64_t n, const int* __restrict__ rows, RowBuffers B, int nb,
                                                                  int rows_per_item, int* __restrict__ bins, int* __restrict__ order) {
  __shared__ int s_row[1024];
  __shared__ int s_wr[8], s_wc[8];
  const int t = threadIdx.x, lane = t & 31, wid = t >> 5, stride = nb + 2;
  int hq[4], cq[4], sum_r = 0, sum_c = 0;
#pragma unroll
  for (int k = 0; k < 4; ++k) {
    const int b = 4 * t + k;
    hq[k] = b < nb ? bins[b] : 0;
    cq[k] = (hq[k] + rows_per_item - 1) / rows_per_item;
    sum_r += hq[k]; sum_c += cq[k];
  }
  int inc_r = sum_r, inc_c = sum_c;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const int a = __shfl_up_sync(FULL_MASK, inc_r, o), c = __shfl_up_sync(FULL_MASK, inc_c, o);
    if (lane >= o) { inc_r += a; inc_c += c; }
  }
  if (lane == 31) { s_wr[wid] = inc_r; s_wc[wid] = inc_c; }
  __syncthreads();
  int base_r = inc_r - sum_r, base_c = inc_c - sum_c, tot_r = 0, tot_c = 0;
#pragma unroll
  for (int w = 0; w < 8; ++w) {
    if (w < wid) { base_r += s_wr[w]; base_c += s_wc[w]; }
    tot_r += s_wr[w]; tot_c += s_wc[w];
  }
#pragma unroll
  for (int k = 0; k < 4; ++k) {
    const int b = 4 * t + k;
    if (b < nb) {
      s_row[b] = base_r;
      if (blockIdx.x == 0) { bins[stride + b] = base_r; bins[2 * stride + b] = base_c; }
    }
    base_r += hq[k]; base_c += cq[k];
  }
  if (blockIdx.x == 0 && t == 0) { bins[stride + nb] = tot_r; bins[2 * stride + nb] = tot_c; }
  __syncthreads();
  int* cursor = bins + 3 * stride;
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  int row = -1, cell = -1 - lane;                            // idle lanes get distinct dummy keys
  if (i < n) { row = rows ? rows[i] : (int)i; cell = B.sc[row].zbin; }
  const unsigned peers = __match_any_sync(FULL_MASK, cell);
  const int leader = __ffs(peers) - 1;
  int base = 0;
  if (lane == leader && cell >= 0) base = s_row[cell] + atomicAdd(&cursor[cell], __popc(peers));
  base = __shfl_sync(FULL_MASK, base, leader);
  if (cell >= 0) order[base + __popc(peers & ((1u << lane) - 1u))] = row;
}

// ---------------------------------------------------------------------------------------------
// a7 + a9 + a10: approximate photometry (Eq. 6) fused with the Gaussian likelihood and the reverse
// pass over the c_SSP table.  One CTA per (z cell, chunk of 64 rows): the cell's two arrays c_t and D_t = c_{t+1} - c_t
// (106 KB at full size) are staged in shared memory; each warp owns AC_R rows and register-blocks over them, so every
// table word read from shared memory feeds AC_R FMAs (the 1 LDS : 2 FMA ratio of a row-at-a-time pass would leave the
// kernel shared-memory bound at ~1/4 of the FMA rate).
//   pass 1 (lane = 4 consecutive entries e = j*n_band + b of a table row):
//            Q^(s)_r,e = sum_i a_r,i c^(s)[i][e]          s = 0: c_t, s = 1: D_t
//   per row: S^(s)_b = sum_j m_j Q^(s)_{jb};  flux_b = F_att,b Mn [S^(0)_b + f S^(1)_b];  g_b = -(flux_b - d_b)/sigma_b^2
//            (or the caller's flux_bar);  direct bars of Mn, z, A_V, delta, F_floor;  m_bar_j
//   pass 2 (lane = age bins i = l, l+32, ...; table rows are an odd number of float4 apart: conflict free):
//            a_bar_r,i = sum_e v_r,e (c_t[i][e] + f_r D_t[i][e]),   v_r,e = g_b F_b Mn m_j
// ---------------------------------------------------------------------------------------------
struct ACWarp {
  float4 buf[128 * AC_R / 4];      // pass 1: a_T[i][r];  pass 2: v[e4][r] (float4 over 4 entries)
  float Qs[AC_R][2][128];          // Q^(0), Q^(1) of the warp's rows after pass 1
  float ms[AC_R][ROW_M_STRIDE];
  float sbar[AC_R][SPS_MAX_BAND];  // g_b F_b Mn
  int rowid[AC_R];
  float4 sc[AC_R][4];              // RowScalars of the warp's rows, fetched before pass 1
  float obs[AC_R][2][SPS_MAX_BAND];// (d_b, sigma_b) or (flux_bar_b, -) of the warp's rows
};

__device__ __forceinline__ void ac_wait(uint32_t bar, uint32_t parity) {
  uint32_t ok = 0;
  while (!ok)
    asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}" : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
}

// One work item: up to AC_ROWS_PER_CTA rows of one z cell; warp w owns rows r_begin + AC_R w .. + AC_R - 1.
__device__ __forceinline__ void ac_item(const TableDev& T, ACWarp& S, const float4* __restrict__ s0, const float4* __restrict__ s1,
                                        int r_begin, int r_end, const int* __restrict__ order, const int* __restrict__ gal_of_row,
                                        const float* __restrict__ obs_flux, const float* __restrict__ obs_sigma,
                                        const float* __restrict__ flux_bar, bool want_grad, const RowBuffers& B,
                                        uint32_t bar, uint32_t parity, bool need_wait) {
  const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
  const int r0 = r_begin + w * AC_R;
  const int cs4 = T.cs_stride >> 2;
  if (r0 >= r_end) { if (need_wait) ac_wait(bar, parity); return; }
  int row[AC_R];
#pragma unroll
  for (int r = 0; r < AC_R; ++r) row[r] = (r0 + r < r_end) ? order[r0 + r] : -1;
  // Request everything the item needs from global memory first (independent loads, all in flight together), then
  // stage it: weights transposed (a_T[i][r], lane = age bin), m, RowScalars and observations of the warp's rows.
  {
    float av[SPS_AGE_PER_LANE][AC_R], mv[AC_R], o0[AC_R], o1[AC_R];
#pragma unroll
    for (int q = 0; q < SPS_AGE_PER_LANE; ++q)
#pragma unroll
      for (int r = 0; r < AC_R; ++r) av[q][r] = row[r] >= 0 ? __ldg(B.a + (int64_t)row[r] * ROW_A_STRIDE + l + 32 * q) : 0.f;
#pragma unroll
    for (int r = 0; r < AC_R; ++r) {
      mv[r] = (row[r] >= 0 && l < ROW_M_STRIDE) ? __ldg(B.m + (int64_t)row[r] * ROW_M_STRIDE + l) : 0.f;
      o0[r] = o1[r] = 0.f;
      if (row[r] >= 0 && l < T.n_band) {
        if (flux_bar) o0[r] = __ldg(flux_bar + (int64_t)row[r] * T.n_band + l);
        else {
          const int64_t gal = gal_of_row ? __ldg(gal_of_row + row[r]) : row[r];
          o0[r] = __ldg(obs_flux + gal * T.n_band + l); o1[r] = __ldg(obs_sigma + gal * T.n_band + l);
        }
      }
    }
    const int rr = l >> 2, part = l & 3;                    // lane -> (row, quarter of its RowScalars)
    int my_row = -1;
#pragma unroll
    for (int r = 0; r < AC_R; ++r) if (r == rr) my_row = row[r];
    float4 scv = make_float4(0.f, 0.f, 0.f, 0.f);
    if (my_row >= 0) scv = reinterpret_cast<const float4*>(B.sc + my_row)[part];
    if (rr < AC_R) S.sc[rr][part] = scv;
#pragma unroll
    for (int q = 0; q < SPS_AGE_PER_LANE; ++q) {
#pragma unroll
      for (int h = 0; h < AC_R / 4; ++h)
        S.buf[(AC_R / 4) * (l + 32 * q) + h] = make_float4(av[q][4 * h], av[q][4 * h + 1], av[q][4 * h + 2], av[q][4 * h + 3]);
    }
#pragma unroll
    for (int r = 0; r < AC_R; ++r) {
      if (l < ROW_M_STRIDE) S.ms[r][l] = mv[r];
      if (l < SPS_MAX_BAND) { S.obs[r][0][l] = o0[r]; S.obs[r][1][l] = o1[r]; }
    }
  }
  __syncwarp();
  if (need_wait) ac_wait(bar, parity);
  const bool act = l < cs4;
  const int E = T.n_Z * T.n_band;
  // ---- pass 1 ----
  float4 q0[AC_R], q1[AC_R];
#pragma unroll
  for (int r = 0; r < AC_R; ++r) q0[r] = q1[r] = make_float4(0.f, 0.f, 0.f, 0.f);
  if (act) {
    const float4* c0p = s0 + l; const float4* c1p = s1 + l;
#pragma unroll 2
    for (int i = 0; i < T.n_age; ++i) {
      const float4 c0 = c0p[i * cs4], c1 = c1p[i * cs4];
      float a8[AC_R];
#pragma unroll
      for (int h = 0; h < AC_R / 4; ++h) {
        const float4 t4 = S.buf[(AC_R / 4) * i + h];
        a8[4 * h] = t4.x; a8[4 * h + 1] = t4.y; a8[4 * h + 2] = t4.z; a8[4 * h + 3] = t4.w;
      }
#pragma unroll
      for (int r = 0; r < AC_R; ++r) {
        q0[r].x = fmaf(a8[r], c0.x, q0[r].x); q0[r].y = fmaf(a8[r], c0.y, q0[r].y); q0[r].z = fmaf(a8[r], c0.z, q0[r].z); q0[r].w = fmaf(a8[r], c0.w, q0[r].w);
        q1[r].x = fmaf(a8[r], c1.x, q1[r].x); q1[r].y = fmaf(a8[r], c1.y, q1[r].y); q1[r].z = fmaf(a8[r], c1.z, q1[r].z); q1[r].w = fmaf(a8[r], c1.w, q1[r].w);
      }
    }
  }
  __syncwarp();                                             // a_T is dead: S.buf becomes the v buffer
  // ---- band step for the warp's rows: lane = (row 2k + l/16, band l%16), AC_R / 2 rounds ----
  //      fluxes, likelihood, direct bars (16-lane reductions), then m_bar (lane = (row, j)) and v (lane = 4 entries)
#pragma unroll
  for (int r = 0; r < AC_R; ++r) {
    if (act) { reinterpret_cast<float4*>(S.Qs[r][0])[l] = q0[r]; reinterpret_cast<float4*>(S.Qs[r][1])[l] = q1[r]; }
    if (l == 0) S.rowid[r] = row[r];
  }
  __syncwarp();
  {
    const int b = l & 15, hl = l >> 4;
    const bool isb = b < T.n_band;
#pragma unroll 1
    for (int k = 0; k < AC_R / 2; ++k) {
      const int r = 2 * k + hl;
      const int rw = S.rowid[r];
      const RowScalars& sc = *reinterpret_cast<const RowScalars*>(&S.sc[r][0]);
      const bool ok = isb && rw >= 0;
      const float f = sc.zfrac, Mn = sc.Mn, zp = 1.f + sc.z;
      float S0 = 0.f, S1 = 0.f, F = 1.f, F_av = 0.f, F_del = 0.f, F_fl = 0.f, F_lam = 0.f, lam_r = 1.f, g = 0.f, chi2 = 0.f;
      if (ok) {
        for (int j = 0; j < T.n_Z; ++j) { S0 = fmaf(S.ms[r][j], S.Qs[r][0][j * T.n_band + b], S0); S1 = fmaf(S.ms[r][j], S.Qs[r][1][j * T.n_band + b], S1); }
        const float izp = __fdividef(1.f, zp);
        lam_r = T.lam_eff[b] * izp;
        dust_at(lam_r, sc.AV, sc.delta, sc.Ffloor, F, F_av, F_del, F_fl, F_lam, T.model == SPS_MODEL_TINY5);
        const float flux = F * Mn * (S0 + f * S1);
        B.flux[(int64_t)rw * SPS_MAX_BAND + b] = flux;
        if (flux_bar) g = S.obs[r][0][b];
        else {
          const float d = S.obs[r][0][b], sg = S.obs[r][1][b];
          const float isg = __fdividef(1.f, sg);
          const float rr = (flux - d) * isg;
          chi2 = rr * rr;
          g = -rr * isg;
        }
      }
      const float Sint = S0 + f * S1;
      float v_mn = g * F * Sint, v_z = g * (F * Mn * S1 * T.inv_dz + Mn * Sint * F_lam * (-lam_r * __fdividef(1.f, zp)));
      float v_av = g * Mn * Sint * F_av, v_de = g * Mn * Sint * F_del, v_fl = g * Mn * Sint * F_fl;
#pragma unroll
      for (int o = 8; o > 0; o >>= 1) {
        chi2 += __shfl_xor_sync(FULL_MASK, chi2, o); v_mn += __shfl_xor_sync(FULL_MASK, v_mn, o); v_z += __shfl_xor_sync(FULL_MASK, v_z, o);
        v_av += __shfl_xor_sync(FULL_MASK, v_av, o); v_de += __shfl_xor_sync(FULL_MASK, v_de, o); v_fl += __shfl_xor_sync(FULL_MASK, v_fl, o);
      }
      if (b == 0 && rw >= 0) {
        RowScalars* out = B.sc + rw;
        out->logp_like = -0.5f * chi2;
        if (want_grad) { out->Mn_bar = v_mn; out->z_bar = v_z; out->AV_bar = v_av; out->delta_bar = v_de; out->Ffloor_bar = v_fl; }
      }
      S.sbar[r][b] = ok ? g * F * Mn : 0.f;
    }
  }
  if (!want_grad) return;
  __syncwarp();
  {
    const int j = l & 15, hl = l >> 4;
#pragma unroll 1
    for (int k = 0; k < AC_R / 2; ++k) {
      const int r = 2 * k + hl;
      const int rw = S.rowid[r];
      if (rw < 0) continue;
      const float f = reinterpret_cast<const RowScalars*>(&S.sc[r][0])->zfrac;
      float mb = 0.f;
      if (j < T.n_Z)
        for (int b = 0; b < T.n_band; ++b) mb = fmaf(S.sbar[r][b], S.Qs[r][0][j * T.n_band + b] + f * S.Qs[r][1][j * T.n_band + b], mb);
      B.m_bar[(int64_t)rw * ROW_M_STRIDE + j] = mb;
    }
  }
  float f8[AC_R];
  {
    int ej[4], eb[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) { const int e = min(4 * l + k, E - 1); ej[k] = e / T.n_band; eb[k] = e - ej[k] * T.n_band; }
#pragma unroll
    for (int r = 0; r < AC_R; ++r) {
      f8[r] = reinterpret_cast<const RowScalars*>(&S.sc[r][0])->zfrac;
      if (act) {
        float vv[4];
#pragma unroll
        for (int k = 0; k < 4; ++k) vv[k] = (4 * l + k < E && row[r] >= 0) ? S.sbar[r][eb[k]] * S.ms[r][ej[k]] : 0.f;
        S.buf[l * AC_R + r] = make_float4(vv[0], vv[1], vv[2], vv[3]);
      }
    }
  }
  __syncwarp();
  // ---- pass 2 ----
  float acc[SPS_AGE_PER_LANE][AC_R];
#pragma unroll
  for (int q = 0; q < SPS_AGE_PER_LANE; ++q)
#pragma unroll
    for (int r = 0; r < AC_R; ++r) acc[q][r] = 0.f;
  int irow[SPS_AGE_PER_LANE];
#pragma unroll
  for (int q = 0; q < SPS_AGE_PER_LANE; ++q) irow[q] = min(l + 32 * q, T.n_age - 1) * cs4;
  for (int e4 = 0; e4 < cs4; ++e4) {
    float4 v[AC_R];
#pragma unroll
    for (int r = 0; r < AC_R; ++r) v[r] = S.buf[e4 * AC_R + r];
#pragma unroll
    for (int q = 0; q < SPS_AGE_PER_LANE; ++q) {
      const float4 c0 = s0[irow[q] + e4], c1 = s1[irow[q] + e4];
#pragma unroll
      for (int r = 0; r < AC_R; ++r) {
        const float tx = fmaf(f8[r], c1.x, c0.x), ty = fmaf(f8[r], c1.y, c0.y), tz = fmaf(f8[r], c1.z, c0.z), tw = fmaf(f8[r], c1.w, c0.w);
        acc[q][r] = fmaf(v[r].x, tx, fmaf(v[r].y, ty, fmaf(v[r].z, tz, fmaf(v[r].w, tw, acc[q][r]))));
      }
    }
  }
#pragma unroll
  for (int r = 0; r < AC_R; ++r) {
    if (row[r] < 0) continue;
#pragma unroll
    for (int q = 0; q < SPS_AGE_PER_LANE; ++q) B.a_bar[(int64_t)row[r] * ROW_A_STRIDE + l + 32 * q] = (l + 32 * q < T.n_age) ? acc[q][r] : 0.f;
  }
}

// Persistent: one CTA per SM walks a contiguous range of the (cell-ordered) work items and reloads the two table
// arrays only when the cell changes, so the 106 KB staging cost is paid ~once per cell per CTA instead of once per item.
__global__ void __launch_bounds__(32 * AC_WARPS, 1)
approx_contract_kernel(TableDev T, int64_t n, const int* __restrict__ order, const int* __restrict__ bins,
                       const int* __restrict__ gal_of_row, const float* __restrict__ obs_flux, const float* __restrict__ obs_sigma,
                       const float* __restrict__ flux_bar, bool want_grad, RowBuffers B) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int nb = T.n_z - 1, stride = nb + 2;
  const int* row_start = bins + stride; const int* cta_start = bins + 2 * stride;
  const int total = cta_start[nb];
  const int per = total / (int)gridDim.x, rem = total % (int)gridDim.x;
  const int w_begin = (int)blockIdx.x * per + min((int)blockIdx.x, rem);
  const int w_end = w_begin + per + ((int)blockIdx.x < rem ? 1 : 0);
  if (w_begin >= w_end) return;
  const int cs4 = T.cs_stride >> 2;                         // float4 per table row (odd)
  const int slice4 = T.n_age * cs4;                         // float4 per array
  float4* s0 = reinterpret_cast<float4*>(smem_raw);
  float4* s1 = s0 + slice4;
  ACWarp* warps = reinterpret_cast<ACWarp*>(s0 + 2 * slice4 + 4);
  __shared__ __align__(8) unsigned long long load_bar;
  const uint32_t bar = (uint32_t)__cvta_generic_to_shared(&load_bar);
  if (threadIdx.x == 0) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(bar));
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  int lo = 0, hi = nb;
  while (hi - lo > 1) { const int mid = (lo + hi) >> 1; if (cta_start[mid] <= w_begin) lo = mid; else hi = mid; }
  int cell = lo, cur_cell = -1;
  uint32_t parity = 1;                                      // flipped before each load: the first one completes phase 0
  for (int w = w_begin; w < w_end; ++w) {
    while (cta_start[cell + 1] <= w) ++cell;
    const bool reload = cell != cur_cell;
    if (reload) {
      __syncthreads();                                      // every warp is done with the previous cell's arrays
      parity ^= 1u;
      cur_cell = cell;
      if (threadIdx.x == 0) {
        // one thread streams the cell's two arrays (contiguous in HBM/L2) into shared memory with bulk async copies
        const char* src = reinterpret_cast<const char*>(T.cssp + (int64_t)cell * 2 * T.n_age * T.cs_stride);
        const uint32_t bytes = (uint32_t)(2 * slice4) * 16u;
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
        const uint32_t dst = (uint32_t)__cvta_generic_to_shared(s0);
        for (uint32_t off = 0; off < bytes; off += 16384u) {
          const uint32_t len = min(16384u, bytes - off);
          asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                       ::"r"(dst + off), "l"(src + off), "r"(len), "r"(bar) : "memory");
        }
      }
    }
    const int r_begin = row_start[cell] + (w - cta_start[cell]) * AC_ROWS_PER_CTA;
    const int r_end = min(row_start[cell + 1], r_begin + AC_ROWS_PER_CTA);
    ac_item(T, warps[threadIdx.x >> 5], s0, s1, r_begin, r_end, order, gal_of_row, obs_flux, obs_sigma, flux_bar, want_grad, B, bar, parity, reload);
    __syncwarp();
  }
}

// ---------------------------------------------------------------------------------------------
// Reverse of a0-a5 (a10) + skew-normal prior (a9): one warp per row contracts the stored per-bin partials (B.part)
// with a_bar, m_bar, Mn_bar and the direct bars.  Only the cheap closed forms (C1, dt/dz, burst polynomial, MDF) are
// re-evaluated; no quadrature is redone.
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(32 * EPI_WARPS_PER_BLOCK, EPI_MIN_BLOCKS)
epilogue_kernel(TableDev T, PriorDev P, const float* theta, int64_t n, bool unbounded, bool with_prior,
                const int* __restrict__ rows, RowBuffers B, float* __restrict__ logp, float* __restrict__ grad, LeapfrogFuse lf) {
  __shared__ float s_prior[7 * SPS_NDIM];
  const PriorView PV = stage_prior(P, s_prior);
  pdl_wait();
  const int64_t r = (int64_t)blockIdx.x * EPI_WARPS_PER_BLOCK + (threadIdx.x >> 5);
  if (r >= n) return;
  const int64_t row = rows ? rows[r] : r;
  const int l = lane_id();
  const RowScalars sc = B.sc[row];
  if (!grad) {                                               // log-posterior only
    float lp = 0.f;
    if (with_prior && l < SPS_NDIM) { float dlp; log_skew_normal(theta[row * SPS_NDIM + l], PV.xi[l], PV.omega[l], PV.skew[l], lp, dlp); }
    lp = warp_sum(lp);
    if (l == 0 && logp) logp[row] = sc.logp_like + lp;
    return;
  }
  // all of the row's stored quantities are requested first: the kernel is a latency-bound stream over B.part
  float lf_eps = 0.f, lf_p = 0.f, lf_im = 0.f, lf_th = 0.f;     // operands of the fused leapfrog update, in flight from the start
  if (lf.p_w && l < SPS_NDIM) {
    const int64_t o = row * SPS_NDIM + l;
    lf_eps = lf.eps[row]; lf_p = lf.p_w[o]; lf_im = lf.inv_mass[o]; lf_th = lf.theta_w[o];
  }
  const float* part = B.part + row * (ROW_PARTS * ROW_A_STRIDE);
  float abar[SPS_AGE_PER_LANE], pr[ROW_PARTS][SPS_AGE_PER_LANE];
#pragma unroll
  for (int q = 0; q < SPS_AGE_PER_LANE; ++q) {
    abar[q] = B.a_bar[row * ROW_A_STRIDE + l + 32 * q];
#pragma unroll
    for (int k = 0; k < ROW_PARTS; ++k) pr[k][q] = part[k * ROW_A_STRIDE + l + 32 * q];
  }
  const float mb = (l < ROW_M_STRIDE) ? B.m_bar[row * ROW_M_STRIDE + l] : 0.f;
  // the direct bar of this lane's parameter, straight from the row's scalars (lane 0: Mn_bar, 9-11: dust bars, 12: z_bar)
  const int fld = l < 16 ? (int)((0x9CBA000000008ull >> (4 * l)) & 15ull) : 0;   // nibble l = the field of RowScalars lane l needs
  static_assert(offsetof(RowScalars, Mn_bar) == 32 && offsetof(RowScalars, z_bar) == 36 && offsetof(RowScalars, AV_bar) == 40 &&
                offsetof(RowScalars, Ffloor_bar) == 48, "RowScalars layout");
  const float direct = reinterpret_cast<const float*>(B.sc + row)[fld];
  // the prior term (a9) depends on the row's parameters only: evaluated while the loads above are in flight
  float lp = 0.f, dlp = 0.f;
  if (with_prior && l < SPS_NDIM) log_skew_normal(theta[row * SPS_NDIM + l], PV.xi[l], PV.omega[l], PV.skew[l], lp, dlp);
  float th_l, d1;                                             // lane p: bounded parameter p and d theta_p / d theta~_p
  load_param_lane(theta + row * SPS_NDIM, unbounded, PV, th_l, d1);
  const float Fb = __shfl_sync(FULL_MASK, th_l, 4), ltp = __shfl_sync(FULL_MASK, th_l, 5), ltm = __shfl_sync(FULL_MASK, th_l, 6);
  const float lz = __shfl_sync(FULL_MASK, th_l, 7), slz = __shfl_sync(FULL_MASK, th_l, 8);
  const float zp = 1.f + __shfl_sync(FULL_MASK, th_l, 12);
  const float dt_dz = -1.f / (zp * T.H0_gyr * sqrtf(T.Om * zp * zp * zp + T.OL));
  BurstQuad Bq;
  burst_bins(T, ltp, ltm, Bq);
  float m_unused, dm_lz, dm_s;
  met_bin(T, lz, slz, m_unused, dm_lz, dm_s);
  const float inv_M = 1.f / sc.Msum, Mf = sc.Mn * inv_M;
  float Ps[SPS_AGE_PER_LANE];
  // round 1 of warp sums: {dL/dF_burst (Eq. A6), sum a_bar P_smooth, burst-time sums}
  float r1[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
  for (int q = 0; q < SPS_AGE_PER_LANE; ++q) {
    Ps[q] = pr[0][q] * inv_M;
    r1[0] += abar[q] * (Bq.P[q] - Ps[q]);
    r1[1] += abar[q] * Ps[q];
    r1[2] += abar[q] * Bq.d_ltp[q];
    r1[3] += abar[q] * Bq.d_ltm[q];
  }
  const float R1 = warp_sum_multi<4>(r1);
  const float s_pp = __shfl_sync(FULL_MASK, R1, warp_multi_holder<4>(1));
  // dL/d(dM_i) = (1-Fb)/Msum (a_bar_i - sum_k a_bar_k Ps_k) + Mn_bar * Mf
  // round 2: {tau, alpha, beta, t_obs sums; MDF sums; prior}
  float r2[8] = {0.f, 0.f, 0.f, 0.f, mb * dm_lz, mb * dm_s, lp, 0.f};
  if (T.agez_gamma != 0.f && l == 0) { r2[4] += sc.pad1; r2[5] += sc.pad2; }   // R26: the bars through every age bin's MDF
  const float c1 = (1.f - Fb) * inv_M, c2 = sc.Mn_bar * Mf;
#pragma unroll
  for (int q = 0; q < SPS_AGE_PER_LANE; ++q) {
    const float dMb = (l + 32 * q < T.n_age) ? fmaf(c1, abar[q] - s_pp, c2) : 0.f;
    r2[0] += dMb * pr[1][q]; r2[1] += dMb * pr[2][q]; r2[2] += dMb * pr[3][q]; r2[3] += dMb * pr[4][q];
  }
  const float R2 = warp_sum_multi<8>(r2);
  // lane p fetches the sum its gradient component needs.  Round 2 holders: value k in lane 16 b2(k) + 8 b1(k) + 4 b0(k):
  // lane 1 <- tau (k 0), 2 <- alpha (1), 3 <- beta (2), 12 <- t_obs (3), 7 <- logZ (4), 8 <- sigma_logZ (5), 0 <- prior (6).
  // Round 1 holders: lane 4 <- F_burst (k 0: lane 0), 5 <- logT_peak (k 2: lane 16), 6 <- logT_max (k 3: lane 24).
  const int k2 = l < 16 ? (int)((0x3000540002106ull >> (4 * l)) & 15ull) : 0;      // nibble l = the round-2 value lane l needs
  const int k1 = l < 16 ? (int)((0x3200000ull >> (4 * l)) & 15ull) : 0;            // nibble l = the round-1 value lane l needs
  const float g2 = __shfl_sync(FULL_MASK, R2, warp_multi_holder<8>(k2));
  const float g1 = __shfl_sync(FULL_MASK, R1, warp_multi_holder<4>(k1));
  float g = g2;                                              // lanes 1, 2, 3, 7, 8
  if (l == 0) g = direct * sc.Mn * LN10F;
  else if (l == 4) g = g1;
  else if (l == 5 || l == 6) g = g1 * Fb;
  else if (l >= 9 && l <= 11) g = direct;
  else if (l == 12) g = fmaf(g2, dt_dz, direct);
  if (l < SPS_NDIM) {
    g = g * d1 + dlp;
    grad[row * SPS_NDIM + l] = g;
    if (lf.p_w) {                                            // fused leapfrog update (theta may alias lf.theta_w: read above, written here)
      const int64_t o = row * SPS_NDIM + l;
      const float pn = lf_p + lf_eps * g;
      lf.p_w[o] = pn;
      lf.theta_w[o] = lf_th + lf_eps * lf_im * pn;
    }
  }
  if (l == 0 && logp) logp[row] = sc.logp_like + g2;         // lane 0's fetch is the prior sum
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

void launch_prologue(const TableDev& T, const PriorDev& P, const float* theta, int64_t n, bool unbounded, bool want_grad,
                     const int* rows, RowBuffers B, bool with_hist, cudaStream_t s, bool small_blocks, bool zero_bins) {
  if (n <= 0) return;
  int* hist = nullptr;
  if (with_hist) { hist = B.bins; if (zero_bins) cudaMemsetAsync(B.bins, 0, 4 * (size_t)(T.n_z + 1) * sizeof(int), s); }   // histogram and scatter cursors
  sps_prof_begin(SPS_K_PROLOGUE, s);
  if (small_blocks) sps_launch(prologue_kernel<8>, dim3((unsigned)((n + 7) / 8)), dim3(256), 0, s, T, P, theta, n, unbounded, want_grad, rows, B, hist);
  else sps_launch(prologue_kernel<PRO_WARPS>, dim3((unsigned)((n + PRO_WARPS - 1) / PRO_WARPS)), dim3(32 * PRO_WARPS), 0, s, T, P, theta, n, unbounded, want_grad, rows, B, hist);
  sps_prof_end(SPS_K_PROLOGUE, s);
  sps_count_launch();
}

static size_t approx_smem_bytes(const TableDev& T) {
  return (size_t)2 * T.n_age * T.cs_stride * sizeof(float) + 64 + AC_WARPS * sizeof(ACWarp);
}
sps_status approx_contract_setup(const TableDev& T) {
  if (T.n_z - 1 > 1 << 20) { sps_set_error("n_z too large"); return SPS_ESHAPE; }
  const size_t bytes = approx_smem_bytes(T);
  if (bytes > 227 * 1024) {
    sps_set_error("table too large for the approximate path: the two c_SSP arrays of a z cell (2 x n_age x n_Z*n_band floats = %zu bytes) "
                  "plus %zu bytes of row staging must fit the 227 KB of shared memory of an SM", (size_t)2 * T.n_age * T.cs_stride * sizeof(float),
                  bytes - (size_t)2 * T.n_age * T.cs_stride * sizeof(float));
    return SPS_ESHAPE;
  }
  // the opt-in is per kernel, not per table: ask for the device maximum so that tables of different sizes can coexist
  int dev = 0, optin = 0;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
  cudaFuncAttributes fa;
  if (cudaFuncGetAttributes(&fa, approx_contract_kernel) == cudaSuccess) optin -= (int)fa.sharedSizeBytes; else cudaGetLastError();
  return sps_check_cuda(cudaFuncSetAttribute(approx_contract_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, std::max((int)bytes, optin)),
                        "approximate-path shared memory opt-in");
}

// rows of a call grouped by z cell (the histogram was taken by the prologue): cell offsets, item offsets, scatter
void approx_group_rows(const TableDev& T, int64_t n, const int* rows, RowBuffers B, int rows_per_item, cudaStream_t s) {
  const int nb = T.n_z - 1, stride = nb + 2;
  const unsigned eb = (unsigned)((n + 255) / 256);
  if (nb <= 1024) {
    approx_scan_scatter_kernel<<<eb, 256, 0, s>>>(n, rows, B, nb, rows_per_item, B.bins, B.order);
    sps_count_launch();
    return;
  }
  approx_plan_kernel<<<1, 1024, 0, s>>>(nb, rows_per_item, B.bins);
  approx_scatter_kernel<<<eb, 256, 0, s>>>(n, rows, B, B.bins + 3 * stride, B.order);
  sps_count_launch(2);
}

void launch_approx_contract(const TableDev& T, int sm_count, int64_t n, const int* rows, const int* gal_of_row,
                            const float* obs_flux, const float* obs_sigma, const float* flux_bar,
                            bool want_grad, RowBuffers B, cudaStream_t s) {
  if (n <= 0) return;
  const int nb = T.n_z - 1;
  approx_group_rows(T, n, rows, B, AC_ROWS_PER_CTA, s);
  const unsigned grid = (unsigned)std::min<int64_t>(sm_count, (n + AC_ROWS_PER_CTA - 1) / AC_ROWS_PER_CTA + nb);
  sps_prof_begin(SPS_K_APPROX, s);
  approx_contract_kernel<<<grid, 32 * AC_WARPS, approx_smem_bytes(T), s>>>(T, n, B.order, B.bins, gal_of_row, obs_flux, obs_sigma,
                                                                         flux_bar, want_grad, B);
  sps_prof_end(SPS_K_APPROX, s);
  sps_count_launch();
}
void launch_epilogue(const TableDev& T, const PriorDev& P, const float* theta, int64_t n, bool unbounded,
                     bool with_prior, const int* rows, RowBuffers B, float* logp, float* grad, LeapfrogFuse lf, cudaStream_t s) {
  if (n <= 0) return;
  sps_prof_begin(SPS_K_EPILOGUE, s);
  sps_launch(epilogue_kernel, dim3((unsigned)((n + EPI_WARPS_PER_BLOCK - 1) / EPI_WARPS_PER_BLOCK)), dim3(32 * EPI_WARPS_PER_BLOCK), 0, s, T, P, theta, n, unbounded, with_prior, rows, B, logp, grad, lf);
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
