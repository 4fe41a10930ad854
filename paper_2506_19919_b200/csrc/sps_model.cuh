// sps_model.cuh -- warp-level device functions of the SPS model: one warp owns one parameter row.
// Steps a0-a5 of the hot path (C1 unbounding, t_obs(z), smooth/burst age weights, MDF weights) and
// their reverse mode.  Lane l owns age bins l, l+32, l+64, l+96 and metallicity bin l.
#pragma once
#include "sps_common.cuh"

#define LN2F 0.69314718055994531f
#define LOG2EF 1.4426950408889634f
#define LN10F 2.3025850929940457f

// ---- a0: Eq. (C1) PAPER.md:429 -----------------------------------------------------------------
// Every lane returns all 13 bounded parameters (th); the slopes d theta / d theta~ are lane-local (load_param_lane).
// The redshift (lane 12) is also returned in double: t_obs(z) - age cancels for the oldest bins.
// The prior / bounds arrays of a launch, staged once per block in shared memory: lanes index them by parameter, and a
// lane-indexed read of the kernel-parameter (constant) bank is replayed once per distinct address.
struct PriorView { const float *y_lo, *y_hi, *k, *x0, *xi, *omega, *skew; };
__device__ __forceinline__ PriorView stage_prior(const PriorDev& P, float* s_prior) {
  static_assert(sizeof(PriorDev) == 7 * SPS_NDIM * sizeof(float), "PriorDev is seven float[SPS_NDIM] arrays");
  if (threadIdx.x < 7 * SPS_NDIM) s_prior[threadIdx.x] = reinterpret_cast<const float*>(&P)[threadIdx.x];
  __syncthreads();
  return PriorView{s_prior, s_prior + SPS_NDIM, s_prior + 2 * SPS_NDIM, s_prior + 3 * SPS_NDIM, s_prior + 4 * SPS_NDIM,
                   s_prior + 5 * SPS_NDIM, s_prior + 6 * SPS_NDIM};
}

// 1 / (1 + exp(-x)) in double at ~30 instructions (libdevice's exp and the division cost ~80): exp(-|x|) = 2^-n exp(-r) with
// |r| <= ln2 / 2 by a degree-10 Taylor polynomial (2e-13), the reciprocal by one Newton step from the fp32 one (4e-15).
__device__ __forceinline__ double sigmoid_d(double x) {
  const double a = fmin(fabs(x), 44.0);
  const double nd = rint(a * 1.4426950408889634);
  const double r = fma(nd, -1.9082149292705877e-10, fma(nd, -0.693147180369123816490, a));      // a - n ln2 (ln2 = hi + lo)
  double p = 2.755731922398589e-7;                                                                  // exp(-r): 1/10!, -1/9!, ...
  p = fma(p, r, -2.755731922398589e-6); p = fma(p, r, 2.48015873015873e-5); p = fma(p, r, -1.984126984126984e-4);
  p = fma(p, r, 1.388888888888889e-3); p = fma(p, r, -8.333333333333333e-3); p = fma(p, r, 4.166666666666666e-2);
  p = fma(p, r, -1.6666666666666666e-1); p = fma(p, r, 0.5); p = fma(p, r, -1.0); p = fma(p, r, 1.0);
  const double e = p * __hiloint2double((1023 - (int)nd) << 20, 0);
  const double d = 1.0 + e;
  const double y0 = (double)__frcp_rn((float)d);
  const double y = fma(y0, fma(-d, y0, 1.0), y0);                                                   // 1 / (1 + e^-|x|)
  return x >= 0.0 ? y : e * y;
}

template <bool NEED_ZD = true, class PR = PriorDev>
__device__ __forceinline__ void load_params(const float* __restrict__ row, bool unbounded, const PR& pr,
                                            float th[SPS_NDIM], double& z_d) {
  const int l = lane_id();
  float v = 0.f;
  double vd = 0.0;
  if (l < SPS_NDIM) {
    v = row[l];
    vd = (double)v;
    if (unbounded) {
      float s = 1.f / (1.f + expf(-pr.k[l] * (v - pr.x0[l])));
      float w = pr.y_hi[l] - pr.y_lo[l];
      if (NEED_ZD && l == SPS_NDIM - 1) {
        const double sd = sigmoid_d((double)pr.k[l] * ((double)v - (double)pr.x0[l]));
        vd = (double)pr.y_lo[l] + ((double)pr.y_hi[l] - (double)pr.y_lo[l]) * sd;
      }
      v = pr.y_lo[l] + w * s;
    }
  }
  z_d = NEED_ZD ? __shfl_sync(FULL_MASK, vd, SPS_NDIM - 1) : 0.0;
#pragma unroll
  for (int p = 0; p < SPS_NDIM; ++p) th[p] = __shfl_sync(FULL_MASK, v, p);
}

// The same for lane p < SPS_NDIM only: its own bounded parameter and slope (no broadcast; the reverse pass needs six of them).
template <class PR>
__device__ __forceinline__ void load_param_lane(const float* __restrict__ row, bool unbounded, const PR& pr, float& v, float& d) {
  const int l = lane_id();
  v = 0.f; d = 1.f;
  if (l < SPS_NDIM) {
    v = row[l];
    if (unbounded) {
      const float s = 1.f / (1.f + expf(-pr.k[l] * (v - pr.x0[l])));
      const float w = pr.y_hi[l] - pr.y_lo[l];
      v = pr.y_lo[l] + w * s;
      d = w * pr.k[l] * s * (1.f - s);
    }
  }
}

// ---- a1: age of the universe (R11), Gyr, and dt/dz ------------------------------------------------
__device__ __forceinline__ void cosmic_time(const TableDev& T, double z_d, double& t_d, float& dt_dz) {
  const double zpd = 1.0 + z_d;
  const double sz = (z_d - T.tz_lo) * T.tz_inv_h;
  if (T.tz_coef != nullptr && sz >= 0.0 && sz < (double)T.tz_n) {            // every lane of the warp holds the same z
    const int iz = (int)sz;
    const double u = 2.0 * (sz - (double)iz) - 1.0;
    const double* c = T.tz_coef + 6 * iz;
    t_d = fma(fma(fma(fma(fma(c[5], u, c[4]), u, c[3]), u, c[2]), u, c[1]), u, c[0]);
  } else {
    t_d = T.t_pref_d * asinh(T.t_arg_d * rsqrt(zpd * zpd * zpd));
  }
  const float zp = (float)zpd, zp3 = zp * zp * zp;
  dt_dz = -1.f / (zp * T.H0_gyr * sqrtf(T.Om * zp3 + T.OL));
}

// ---- a2: double power law, Eq. (A4) PAPER.md:346 ---------------------------------------------------
// f = 1/(x^alpha + x^-beta) at x = 2^lx2.  With A = f^2 x^alpha and B = f^2 x^-beta the partials are
//   t df/dt = -(alpha A - beta B) = -q,  df/dtau = q / tau,  df/dalpha = -A ln x,  df/dbeta = B ln x,
// so a quadrature accumulates sum w f, sum w A, sum w B, sum w A lx2, sum w B lx2 (and sum w A / t, sum w B / t for the
// t_obs partial) and combines them once per bin (SfrSums::finish) instead of forming q, fa, fb at every node.
struct SfrNode { float f, A, B, lx2; };
__device__ __forceinline__ SfrNode sfr_node(float lx2, float alpha, float beta) {
  const float xa = exp2f(fminf(alpha * lx2, 60.f));
  const float xb = exp2f(fminf(-beta * lx2, 60.f));
  SfrNode n;
  n.f = __fdividef(1.f, xa + xb);
  const float f2 = n.f * n.f;
  n.A = f2 * xa; n.B = f2 * xb; n.lx2 = lx2;
  return n;
}
struct SfrSums {
  float f = 0.f, A = 0.f, B = 0.f, Al = 0.f, Bl = 0.f, At = 0.f, Bt = 0.f;
  __device__ __forceinline__ void add(const SfrNode& n, float w) {
    f = fmaf(w, n.f, f);
    const float wA = w * n.A, wB = w * n.B;
    A += wA; B += wB; Al = fmaf(wA, n.lx2, Al); Bl = fmaf(wB, n.lx2, Bl);
  }
  __device__ __forceinline__ void add_t(const SfrNode& n, float w, float inv_t) {      // also the d/dt_obs sums (linear-t rules)
    f = fmaf(w, n.f, f);
    const float wA = w * n.A, wB = w * n.B;
    A += wA; B += wB; Al = fmaf(wA, n.lx2, Al); Bl = fmaf(wB, n.lx2, Bl);
    At = fmaf(wA, inv_t, At); Bt = fmaf(wB, inv_t, Bt);
  }
};
__device__ __forceinline__ float sfr_value(float t, float tau, float alpha, float beta) {
  if (!(t > 0.f)) return 0.f;
  float lx2 = __log2f(t / tau);
  return __fdividef(1.f, exp2f(fminf(alpha * lx2, 60.f)) + exp2f(fminf(-beta * lx2, 60.f)));
}

struct AgeQuad {                       // per lane: its (up to) 4 bins, for M_formed = 1
  float dM[SPS_AGE_PER_LANE];          // int_bin f dt            (Eq. A5 numerator)
  float g_tau[SPS_AGE_PER_LANE], g_al[SPS_AGE_PER_LANE], g_be[SPS_AGE_PER_LANE], g_t[SPS_AGE_PER_LANE];
};

// Gauss-Legendre nodes/weights on [-1,1]
__device__ __constant__ float GL2_X[2] = {-0.5773502691896257f, 0.5773502691896257f};
__device__ __constant__ float GL4_X[4] = {-0.8611363115940526f, -0.3399810435848563f, 0.3399810435848563f, 0.8611363115940526f};
__device__ __constant__ float GL4_W[4] = {0.3478548451374538f, 0.6521451548625461f, 0.6521451548625461f, 0.3478548451374538f};
__device__ __constant__ float GL8_X[8] = {-0.9602898564975363f, -0.7966664774136267f, -0.5255324099163290f, -0.1834346424956498f,
                                          0.1834346424956498f, 0.5255324099163290f, 0.7966664774136267f, 0.9602898564975363f};
__device__ __constant__ float GL8_W[8] = {0.1012285362903763f, 0.2223810344533745f, 0.3137066458778873f, 0.3626837833783620f,
                                          0.3626837833783620f, 0.3137066458778873f, 0.2223810344533745f, 0.1012285362903763f};

// Four values summed over the warp in 6 shuffles (instead of 4 x 5): the halves of the warp swap two of the four, then the
// quarters one of the two, then three plain steps.  Afterwards lane l holds the total of value (l >> 3) & 3.
__device__ __forceinline__ float warp_sum4(float v0, float v1, float v2, float v3) {
  const int l = lane_id();
  const bool h16 = l & 16, h8 = l & 8;
  float k0 = h16 ? v2 : v0, k1 = h16 ? v3 : v1;
  k0 += __shfl_xor_sync(FULL_MASK, h16 ? v0 : v2, 16);
  k1 += __shfl_xor_sync(FULL_MASK, h16 ? v1 : v3, 16);
  float k = h8 ? k1 : k0;
  k += __shfl_xor_sync(FULL_MASK, h8 ? k0 : k1, 8);
#pragma unroll
  for (int o = 4; o > 0; o >>= 1) k += __shfl_xor_sync(FULL_MASK, k, o);
  return k;
}

// Mass formed per age bin (Eq. A5; R5, R6 restated for fp32):
//  * bins whose span in ln t is small against the width 1/(alpha+beta) of the SFR turnover are
//    integrated by 2- or 4-point Gauss-Legendre in linear t with the tabulated bin width (no
//    t_obs - age cancellation in the width);
//  * the few old bins near age ~ t_obs (and the one that reaches t = 0) are integrated by the whole
//    warp: 8-point Gauss-Legendre panels in v = ln t, cut at ln t_hi - 16/(beta+1).
// t = t_obs - age in two-float arithmetic: t_obs = th + tl, edge = ah + al; (th - ah) is exact where the two are within a
// factor of two (the old bins, where the difference cancels), so t is within an ulp of the double difference everywhere.
template <bool WANT_GRAD>
__device__ __forceinline__ void smooth_bins(const TableDev& T, double t_obs_d, float tau, float alpha, float beta, AgeQuad& Q) {
  const int l = lane_id();
  const float l2tau = __log2f(tau);
  const float ab = alpha + beta;
  const float th = (float)t_obs_d, tl = (float)(t_obs_d - (double)th);
  float t_edge[SPS_AGE_PER_LANE + 1];       // t at the lower age edge of the lane's bins (= t_hi of the bin), clipped at 0
#pragma unroll
  for (int q = 0; q < SPS_AGE_PER_LANE; ++q) {
    const float2 e = T.A_edge_hl[l + 32 * q];
    t_edge[q] = fmaxf((th - e.x) + (tl - e.y), 0.f);
  }
  t_edge[SPS_AGE_PER_LANE] = 0.f;
  unsigned problem_mask[SPS_AGE_PER_LANE];
  float t_lo_q[SPS_AGE_PER_LANE], t_hi_q[SPS_AGE_PER_LANE];
#pragma unroll
  for (int q = 0; q < SPS_AGE_PER_LANE; ++q) {
    const int i = l + 32 * q;
    Q.dM[q] = Q.g_tau[q] = Q.g_al[q] = Q.g_be[q] = Q.g_t[q] = 0.f;
    // the bin's upper age edge is the lower edge of the next bin: lane + 1, or lane 0's next slot
    float t_lo = __shfl_down_sync(FULL_MASK, t_edge[q], 1);
    const float t_lo0 = __shfl_sync(FULL_MASK, t_edge[q + 1], 0);
    if (l == 31) t_lo = t_lo0;
    float t_hi = 0.f, half = 0.f, t_mid = 1.f;
    int kind = 0;                       // 0 empty, 1 GL2, 2 GL4, 3 warp-cooperative
    if (i < T.n_age && t_edge[q] > 0.f) {
      t_hi = t_edge[q];
      half = T.A_half[i];
      t_mid = t_hi - half;
      // half-width over the distance to the nearest singularity: the turnover poles at Im ln t = pi/(alpha+beta)
      // and the branch point of t^beta at t = 0
      const float s = (t_lo > 0.f) ? __fdividef(half, t_mid) * fmaxf(ab * 0.3183098861837907f, 1.f) : 1e9f;
      kind = (s < 0.06f) ? 1 : (s < 0.36f ? 2 : 3);
    } else t_lo = 0.f;
    t_lo_q[q] = t_lo; t_hi_q[q] = t_hi;
    problem_mask[q] = __ballot_sync(FULL_MASK, kind == 3);
    const bool any4 = __any_sync(FULL_MASK, kind == 2);
    if (kind == 1 || kind == 2) {
      SfrSums S;
      if (!any4) {
#pragma unroll
        for (int k = 0; k < 2; ++k) {
          const float t = t_mid + half * GL2_X[k];
          S.add_t(sfr_node(__log2f(t) - l2tau, alpha, beta), 1.f, __fdividef(1.f, t));
        }
      } else {
#pragma unroll
        for (int k = 0; k < 4; ++k) {
          const float t = t_mid + half * GL4_X[k];
          S.add_t(sfr_node(__log2f(t) - l2tau, alpha, beta), GL4_W[k], __fdividef(1.f, t));
        }
      }
      Q.dM[q] = half * S.f;
      if (WANT_GRAD) {
        Q.g_tau[q] = half * (alpha * S.A - beta * S.B) / tau;
        Q.g_al[q] = -half * LN2F * S.Al; Q.g_be[q] = half * LN2F * S.Bl;
        Q.g_t[q] = -half * (alpha * S.At - beta * S.Bt);
      }
    }
  }
  // warp-cooperative bins: 8-point Gauss-Legendre panels in v = ln t.
  //  * the one bin that reaches t = 0 spans many panels: all 32 lanes share its nodes;
  //  * the other old bins near t_obs need one or two panels each: four of them are integrated at once, 8 lanes per bin.
  const float ln_tau = l2tau * LN2F;
  const float w_target = fminf(fmaxf(6.5f / ab, 0.5f), 2.0f);
#pragma unroll
  for (int q = 0; q < SPS_AGE_PER_LANE; ++q) {
    unsigned m = problem_mask[q];
    const unsigned mz = __ballot_sync(FULL_MASK, t_hi_q[q] > 0.f && !(t_lo_q[q] > 0.f)) & m;     // the bin touching t = 0
    if (mz) {
      const int src = __ffs(mz) - 1;
      m &= ~mz;
      const float t_hi = __shfl_sync(FULL_MASK, t_hi_q[q], src);
      const float v_hi = __logf(t_hi);
      // below min(t_hi, tau) the integrand falls as t^(beta+1): cut 16/(beta+1) e-folds under that point (not under t_hi:
      // a coarse grid's oldest bin can reach far past the turnover, and most of its mass then sits near tau)
      const float v_lo = fminf(v_hi, ln_tau) - 16.f / (beta + 1.f);
      const float dv = v_hi - v_lo;
      const int n_pan = max(1, (int)ceilf(dv / w_target));
      const float wp = dv / (float)n_pan;
      SfrSums S;
      const float xk = 0.5f + 0.5f * GL8_X[l & 7], wk = 0.5f * wp * GL8_W[l & 7];
      for (int n = l; n < n_pan * 8; n += 32) {
        const float v = v_lo + ((float)(n >> 3) + xk) * wp;
        S.add(sfr_node((v - ln_tau) * LOG2EF, alpha, beta), wk * __expf(v));        // dt = t dv
      }
      const float s0 = warp_sum(S.f);
      // the four gradient sums in one pass: lane l ends up with the total of sum (l >> 3) & 3
      const float g = warp_sum4(alpha * S.A - beta * S.B, S.Al, S.Bl, 0.f);
      const float r1 = __shfl_sync(FULL_MASK, g, 0), r2 = __shfl_sync(FULL_MASK, g, 8), r3 = __shfl_sync(FULL_MASK, g, 16);
      if (l == src) {
        Q.dM[q] = s0;
        if (WANT_GRAD) { Q.g_tau[q] = r1 / tau; Q.g_al[q] = -LN2F * r2; Q.g_be[q] = LN2F * r3; Q.g_t[q] = sfr_value(t_hi, tau, alpha, beta); }   // Leibniz, f(0) = 0
      }
    }
    while (m) {
      int srcs[4];
#pragma unroll
      for (int j = 0; j < 4; ++j) { srcs[j] = m ? __ffs(m) - 1 : -1; m &= m - 1; }
      const int sg = l >> 3, k = l & 7;
      const int my_src = sg == 0 ? srcs[0] : (sg == 1 ? srcs[1] : (sg == 2 ? srcs[2] : srcs[3]));
      const bool have = my_src >= 0;
      const float t_hi = __shfl_sync(FULL_MASK, t_hi_q[q], have ? my_src : 0);
      const float t_lo = __shfl_sync(FULL_MASK, t_lo_q[q], have ? my_src : 0);
      const float v_hi = __logf(t_hi);
      const float v_lo = fmaxf(fminf(v_hi, ln_tau) - 16.f / (beta + 1.f), __logf(t_lo));
      const float dv = v_hi - v_lo;
      int n_pan = have ? max(1, (int)ceilf(dv / w_target)) : 0;
      const float wp = dv / (float)max(n_pan, 1);
      int n_max = max(n_pan, __shfl_xor_sync(FULL_MASK, n_pan, 8));
      n_max = max(n_max, __shfl_xor_sync(FULL_MASK, n_max, 16));
      SfrSums S;
      const float xk = 0.5f + 0.5f * GL8_X[k], wk = 0.5f * wp * GL8_W[k];
      for (int pan = 0; pan < n_max; ++pan) {
        if (pan < n_pan) {
          const float v = v_lo + ((float)pan + xk) * wp;
          S.add(sfr_node((v - ln_tau) * LOG2EF, alpha, beta), wk * __expf(v));
        }
      }
      float s0 = S.f, s1 = alpha * S.A - beta * S.B, s2 = -LN2F * S.Al, s3 = LN2F * S.Bl;
#pragma unroll
      for (int o = 4; o > 0; o >>= 1) {
        s0 += __shfl_xor_sync(FULL_MASK, s0, o);
        if (WANT_GRAD) { s1 += __shfl_xor_sync(FULL_MASK, s1, o); s2 += __shfl_xor_sync(FULL_MASK, s2, o); s3 += __shfl_xor_sync(FULL_MASK, s3, o); }
      }
      // hand each result to the lane that owns the bin
      const int rank = l == srcs[0] ? 0 : (l == srcs[1] ? 1 : (l == srcs[2] ? 2 : (l == srcs[3] ? 3 : -1)));
      const int from = 8 * max(rank, 0);
      const float r0 = __shfl_sync(FULL_MASK, s0, from);
      float r1 = 0, r2 = 0, r3 = 0;
      if (WANT_GRAD) { r1 = __shfl_sync(FULL_MASK, s1, from); r2 = __shfl_sync(FULL_MASK, s2, from); r3 = __shfl_sync(FULL_MASK, s3, from); }
      if (rank >= 0) {
        Q.dM[q] = r0;
        if (WANT_GRAD) {
          Q.g_tau[q] = r1 / tau; Q.g_al[q] = r2; Q.g_be[q] = r3;
          Q.g_t[q] = sfr_value(t_hi_q[q], tau, alpha, beta) - sfr_value(t_lo_q[q], tau, alpha, beta);   // Leibniz
        }
      }
    }
  }
}

// ---- a3: triweight burst, Eq. (A6)-(A7) PAPER.md:358-372 (R7: CDF differences over the age-bin edges) ----
// P_i = int_{y_lo}^{y_hi} (35/32)(1-y^2)^3 dy with y = clip((e - logT_peak)/(logT_max - logT_peak), -1, 1);
// the integrand is a degree-6 polynomial, so 4-point Gauss-Legendre is exact and free of cancellation.
__device__ __forceinline__ float tri_pdf_y(float y) { float u = 1.f - y * y; return (35.f / 32.f) * u * u * u; }

struct BurstQuad { float P[SPS_AGE_PER_LANE], d_ltp[SPS_AGE_PER_LANE], d_ltm[SPS_AGE_PER_LANE]; };

__device__ __forceinline__ void burst_bins(const TableDev& T, float ltp, float ltm, BurstQuad& B) {
  const int l = lane_id();
  const float inv_s3 = 1.f / (ltm - ltp);
  // Every bin edge is evaluated once, by the lane that owns the bin above it: y clipped to [-1, 1] and the density there
  // (zero at the clips); a bin takes its upper edge from the owner of the next bin (lane + 1, or lane 0's next slot).
  // Slots past the grid sit at the upper clip, so their bins come out as zero without a branch.
  float y[SPS_AGE_PER_LANE + 1], p[SPS_AGE_PER_LANE + 1];
#pragma unroll
  for (int q = 0; q < SPS_AGE_PER_LANE; ++q) {
    const int i = l + 32 * q;
    const float e = (i <= T.n_age) ? T.e_edge[i] : 1e30f;
    y[q] = fminf(fmaxf((e - ltp) * inv_s3, -1.f), 1.f);
    p[q] = tri_pdf_y(y[q]);
  }
  y[SPS_AGE_PER_LANE] = 1.f; p[SPS_AGE_PER_LANE] = 0.f;
  const float x1 = 0.8611363115940526f, x2 = 0.3399810435848563f, w1 = 0.3478548451374538f, w2 = 0.6521451548625461f;
#pragma unroll
  for (int q = 0; q < SPS_AGE_PER_LANE; ++q) {
    float yb = __shfl_down_sync(FULL_MASK, y[q], 1), pb = __shfl_down_sync(FULL_MASK, p[q], 1);
    const float y0 = __shfl_sync(FULL_MASK, y[q + 1], 0), p0 = __shfl_sync(FULL_MASK, p[q + 1], 0);
    if (l == 31) { yb = y0; pb = p0; }
    const float ya = y[q], pa = p[q];
    const float half = 0.5f * (yb - ya), mid = 0.5f * (yb + ya), h1 = half * x1, h2 = half * x2;
    // 4-point Gauss-Legendre on the symmetric node pairs mid +- h1, mid +- h2
    float u1 = fmaf(-(mid - h1), mid - h1, 1.f), u2 = fmaf(-(mid + h1), mid + h1, 1.f);
    float u3 = fmaf(-(mid - h2), mid - h2, 1.f), u4 = fmaf(-(mid + h2), mid + h2, 1.f);
    const float s = w1 * (u1 * u1 * u1 + u2 * u2 * u2) + w2 * (u3 * u3 * u3 + u4 * u4 * u4);
    B.P[q] = (35.f / 32.f) * half * s;
    // dy/dlogT_peak = (y-1)/s3, dy/dlogT_max = -y/s3
    B.d_ltp[q] = (pb * (yb - 1.f) - pa * (ya - 1.f)) * inv_s3;
    B.d_ltm[q] = (-pb * yb + pa * ya) * inv_s3;
  }
}

// ---- a4: lognormal MDF PAPER.md:378 (R9).  Lane j < n_Z owns metallicity bin j. -------------------
__device__ __forceinline__ void met_bin(const TableDev& T, float lz, float s, float& m, float& d_lz, float& d_s) {
  const int j = lane_id();
  const float inv_s = 1.f / s;
  const bool has_lo = j > 0 && j < T.n_Z, has_hi = j < T.n_Z - 1;
  // lane k < n_Z - 1 evaluates bin edge k once (erfc of |u| and the normal density); bin j takes its lower edge from lane j - 1
  const float ub = has_hi ? (T.g_mid[j] - lz) * inv_s : 1e30f;
  const float r2 = 0.7071067811865476f, c = 0.3989422804014327f;
  const float eb = has_hi ? erfcf(fabsf(ub) * r2) : 0.f;
  const float pb = has_hi ? c * expf(-0.5f * ub * ub) : 0.f;
  float ua = __shfl_up_sync(FULL_MASK, ub, 1), ea = __shfl_up_sync(FULL_MASK, eb, 1), pa = __shfl_up_sync(FULL_MASK, pb, 1);
  if (!has_lo) { ua = -1e30f; ea = 0.f; pa = 0.f; }
  m = d_lz = d_s = 0.f;
  if (j < T.n_Z) {
    // normal-CDF difference through the tail that keeps relative accuracy
    if (ua > 0.f) m = 0.5f * (ea - eb);
    else if (ub < 0.f) m = 0.5f * (eb - ea);
    else m = 1.f - 0.5f * (eb + ea);
    d_lz = -(pb - pa) * inv_s;
    d_s = -(pb * (has_hi ? ub : 0.f) - pa * (has_lo ? ua : 0.f)) * inv_s;
  }
}

// The same MDF for one median, serially in one thread (non-separable weights, R26: every age bin has its own median):
// m[j], dm/dmedian, dm/dsigma for j < n_Z.
__device__ __forceinline__ void mdf_row(const TableDev& T, float mu, float s, float* __restrict__ m, float* __restrict__ d_mu, float* __restrict__ d_s) {
  const float inv_s = 1.f / s, r2 = 0.7071067811865476f, c = 0.3989422804014327f;
  float ua = -1e30f, ea = 0.f, pa = 0.f;                    // lower edge of bin 0: -infinity
  for (int j = 0; j < T.n_Z; ++j) {
    const bool has_hi = j < T.n_Z - 1;
    const float ub = has_hi ? (T.g_mid[j] - mu) * inv_s : 1e30f;
    const float eb = has_hi ? erfcf(fabsf(ub) * r2) : 0.f;
    const float pb = has_hi ? c * expf(-0.5f * ub * ub) : 0.f;
    float mj;
    if (ua > 0.f) mj = 0.5f * (ea - eb);
    else if (ub < 0.f) mj = 0.5f * (eb - ea);
    else mj = 1.f - 0.5f * (eb + ea);
    m[j] = mj;
    d_mu[j] = -(pb - pa) * inv_s;
    d_s[j] = -(pb * (has_hi ? ub : 0.f) - pa * (j > 0 ? ua : 0.f)) * inv_s;
    ua = ub; ea = eb; pa = pb;
  }
}

// ---- a8: dust, Eq. (A8)-(A9) PAPER.md:386-392 (R10) at an arbitrary rest wavelength (approximate path) ----
#define CALZ_SWITCH_INV_UM 1.2809053864877329f
// `screen` (SPS_MODEL_TINY5): k0 = 4.05 and no bump, which with delta = -0.7, F_floor = 0 and A_V = 1.0857 tau_V is the
// power-law screen exp(-tau_V (lambda/5500)^-0.7).
__device__ __forceinline__ void dust_at(float lam, float AV, float delta, float Ffl,
                                        float& F, float& F_av, float& F_del, float& F_fl, float& F_lam, bool screen = false) {
  const float ilam = __fdividef(1.f, lam);                  // one approximate reciprocal (1 ulp) serves every division by lambda
  const float u = 1.0e4f * ilam;
  float k0, dk_du;
  if (screen) { k0 = 4.05f; dk_du = 0.f; }
  else if (u > CALZ_SWITCH_INV_UM) {
    k0 = 2.659f * (-2.156f + u * (1.509f + u * (-0.198f + u * 0.011f))) + 4.05f;
    dk_du = 2.659f * (1.509f + u * (-0.396f + u * 0.033f));
  } else {
    k0 = 2.659f * (-1.857f + 1.040f * u) + 4.05f;
    dk_du = 2.659f * 1.040f;
  }
  float dk0 = dk_du * (-u * ilam);
  if (!(k0 > 0.f)) { k0 = 0.f; dk0 = 0.f; }
  const float l0 = 2175.f, w = 350.f;
  const float n = (lam * w) * (lam * w);
  const float dl = lam * lam - l0 * l0;
  const float den = dl * dl + n;
  const float dn = 2.f * lam * w * w;
  const float dd = 4.f * lam * dl + dn;
  const float iden = __fdividef(1.f, den);
  const float dr = screen ? 0.f : n * iden, ddr = screen ? 0.f : (dn * den - n * dd) * iden * iden;
  const float l2r = log2f(lam * (1.f / 5500.f));
  const float pw = exp2f(delta * l2r);
  const float Eb = 0.85f - 1.9f * delta;
  const float br = k0 * pw + Eb * dr;
  float A = AV * (1.f / 4.05f) * br;
  float A_av = br * (1.f / 4.05f);
  float A_del = AV * (1.f / 4.05f) * (k0 * pw * l2r * LN2F - 1.9f * dr);     // (TINY5 never uses the delta, F_floor, lambda partials)
  float A_lam = AV * (1.f / 4.05f) * (dk0 * pw + k0 * delta * pw * ilam + Eb * ddr);
  if (!(A > 0.f)) { A = 0.f; A_av = A_del = A_lam = 0.f; }
  const float Tt = exp2f(-0.4f * 3.321928094887362f * A);
  const float dF_dA = -(1.f - Ffl) * 0.4f * LN10F * Tt;
  F = Ffl + (1.f - Ffl) * Tt;
  F_av = dF_dA * A_av; F_del = dF_dA * A_del; F_fl = 1.f - Tt; F_lam = dF_dA * A_lam;
}

// ---- a9 (prior part): log skew-normal, Eq. (C2), and d/dtheta~ ---------------------------
__device__ __forceinline__ void log_skew_normal(float x, float xi, float om, float s, float& lp, float& dlp) {
  const float u = (x - xi) / om;
  const float a = s * u;
  // log Phi(a) through erfc (scaled form for the far lower tail)
  const float r2 = 0.7071067811865476f;
  float logPhi, ratio;   // ratio = phi(a)/Phi(a)
  const float Phi = 0.5f * erfcf(-a * r2);
  if (a > -5.f) {
    logPhi = logf(Phi);
    ratio = 0.3989422804014327f * expf(-0.5f * a * a) / Phi;
  } else {               // asymptotic: Phi(a) ~ phi(a)/(-a) (1 - 1/a^2 + 3/a^4)
    const float ia2 = 1.f / (a * a);
    const float corr = 1.f - ia2 + 3.f * ia2 * ia2;
    logPhi = -0.5f * a * a - 0.9189385332046727f - logf(-a) + logf(corr);
    ratio = -a / corr;
  }
  lp = 0.6931471805599453f - logf(om) - 0.9189385332046727f - 0.5f * u * u + logPhi;
  dlp = (-u + s * ratio) / om;
}
