// sps_common.cuh -- shared declarations of the CUDA path (sm_100a only).
// No code is shared with oracle/ ; formulas are restated from PAPER.md (line numbers cited) and
// the DESIGN.md readings R#.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include "../../include/sps.h"

#define SPS_MAX_AGE 128
#define SPS_MAX_Z 16
#define SPS_MAX_BAND 16
#define SPS_AGE_PER_LANE 4          // ceil(SPS_MAX_AGE / 32)
#define FULL_MASK 0xffffffffu
#define SPS_FTAB_BINS 1024          // index bins per tabulated filter
#define SPS_FTAB_MAX_KNOTS 4096     // knots per tabulated filter

// Tabulated filter curves (R4: linear interpolation between knots, zero outside the support).  A lookup finds the
// segment through a uniform index over the band's support (first[b][bin] = the segment holding the bin's left end) and
// then walks right while lambda is past the segment's end.
struct FilterTab {
  const float4* knots;        // [n_knot] {w, t, slope to the next knot, w_next}; a band's last knot: slope 0, w_next = +huge
  const int* first;           // [n_band][SPS_FTAB_BINS]
  float lo[SPS_MAX_BAND], hi[SPS_MAX_BAND], inv_d[SPS_MAX_BAND];
  int last[SPS_MAX_BAND];     // the band's last segment (index of the knot before its last knot)
};

// ---------------------------------------------------------------------------------------------
// device-side view of a table (passed to kernels by value; arrays live in device memory)
// ---------------------------------------------------------------------------------------------
struct TableDev {
  int model, n_dim;                            // SPS_MODEL_*; number of sampled parameters
  int filt_tab;                                // 1: tabulated filters (ft), 0: Gaussian (filt_mu, filt_sigma)
  float agez_gamma;                            // R26: d(median logZ) / d(log10 age); 0 = separable weights
  const float* gauss;                          // SPS_MODEL_GAUSS_TEST: [13] mu then [13][13] precision (row stride 13)
  FilterTab ft;
  int n_age, n_Z, n_wave, n_band, n_z, K;     // K = n_age * n_Z
  int n_wave_pad;                              // n_wave rounded up for the tensor-core tiles
  int cs_stride;                               // floats between consecutive ages in a c_SSP slice (n_Z*n_band padded)
  // age grid (R5): A[i] lower age edge of bin i in Gyr (A[0] = 0, A[n_age] = +huge)
  const double* A_edge_d;   // [n_age+1] the same in double: t_obs - A is formed in double (old bins cancel)
  const double* A_mid_d;    // [n_age]
  const float2* A_edge_hl;  // [128] the edges as float pairs (hi, lo = double - hi; entries past n_age: +huge): t_obs - A in two-float arithmetic
  const float* A_edge;      // [n_age+1]
  const float* A_mid;       // [n_age]   (A[i]+A[i+1])/2   (last: unused)
  const float* A_half;      // [n_age]   (A[i+1]-A[i])/2   (last: +huge)
  const float* e_edge;      // [n_age+1] log10(age/yr) of the edges (-huge, ..., +huge)
  const float* g_mid;       // [n_Z-1]   log10 Z bin edges (midpoints)
  const float* la9;         // [n_age]   log10(age_i / yr) - 9 (R26: the MDF median of age bin i is logZ + agez_gamma la9[i])
  // wavelength grid and per-wavelength constants (exact path)
  const float* wave;        // [n_wave_pad] Angstrom (padding: copies of the last value)
  const float* dlam;        // [n_wave_pad] trapezoid weights (R4), 0 in the padding
  const float* k0;          // [n_wave_pad] Calzetti k0(lambda) (R10)
  const float* drude;       // [n_wave_pad] Drude profile (R10)
  const float* l2r;         // [n_wave_pad] log2(lambda / 5500 A)
  const float* ssp;         // [K][n_wave_pad] fp32
  // filters
  float filt_mu[SPS_MAX_BAND], filt_sigma[SPS_MAX_BAND], lam_eff[SPS_MAX_BAND];
  // c_SSP lookup table (Eq. 7): [n_z][2][n_age][cs_stride]: per z slice the values c_t and the increments
  // c_{t+1} - c_t; entry (j*n_band + b) inside a row
  const float* cssp;
  float z_min, dz, inv_dz;
  // cosmology (R11): t = t_pref * asinh(t_arg * (1+z)^-1.5)  [Gyr];  H0 in 1/Gyr
  float t_pref, t_arg, H0_gyr, Om, OL;
  double t_pref_d, t_arg_d;
  // the same function as piecewise degree-5 polynomials in double over the z grid's range (tz_n intervals, local variable
  // u in [-1, 1], coefficients c0..c5; interpolated at Chebyshev nodes at table creation: relative error < 1e-15), so that a
  // row costs five double FMAs instead of a double-precision asinh; outside the range the closed form is evaluated
  const double* tz_coef;    // [tz_n][6] or null
  double tz_lo, tz_inv_h;
  int tz_n;
  float log10_mass_unit;
  // exact path: bound of a band sum per unit M_star (largest bolometric integral of an SSP x largest transmission) and the
  // headroom bits of the z partial (sps_exact.cuh: fixed-point band sums)
  float part_bound; int part_shift_z;
};

struct PriorDev {
  float y_lo[SPS_NDIM], y_hi[SPS_NDIM], k[SPS_NDIM], x0[SPS_NDIM];
  float xi[SPS_NDIM], omega[SPS_NDIM], skew[SPS_NDIM];
};

// Per-row intermediate record exchanged between the prologue, contraction and epilogue kernels.
// All sizes padded so rows are 16-byte aligned.
#define ROW_A_STRIDE 128      // a_i / a_bar_i
#define ROW_M_STRIDE 16       // m_j / m_bar_j
struct RowScalars {           // 16 floats
  float Mn;                   // M_star / mass_unit
  float z;                    // bounded redshift
  float zfrac;                // position inside the z cell [0,1)
  int   zbin;                 // lower z-grid index
  float AV, delta, Ffloor;    // bounded dust parameters
  float logp_like;            // filled by the contraction: -1/2 chi^2
  float Mn_bar;               // d logL / d Mn
  float z_bar;                // direct d logL / d z (table interpolation + dust at lambda_eff/(1+z) or filter shift)
  float AV_bar, delta_bar, Ffloor_bar;
  float Msum;                 // int_0^t_obs f dt for M_formed = 1 (Eq. A3), kept for the reverse pass
  float pad1, pad2;           // non-separable weights (R26): logZ, sigma_logZ from the prologue; the contraction replaces them
                              // by d logL / d logZ, d logL / d sigma_logZ (through every age bin's MDF) for the epilogue
};

// ---------------------------------------------------------------------------------------------
// small device helpers
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ float warp_sum(float v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(FULL_MASK, v, o);
  return v;
}

__device__ __forceinline__ int lane_id() { return threadIdx.x & 31; }

// Warp sums of N = 4 or 8 per-lane values at once: every exchange step halves the number of values a lane carries
// (N + log2(32) - 1 shuffles instead of 5 N).  On return lane l holds the complete sum of value
// k(l) = 4 b4 + 2 b3 + b2 (N = 8) or 2 b4 + b3 (N = 4), b_i = bit i of l: value k is held by lane warp_multi_holder<N>(k).
template <int N> __device__ __forceinline__ float warp_sum_multi(float (&v)[N]) {
  static_assert(N == 4 || N == 8, "4 or 8 values");
  const int l = threadIdx.x & 31;
  int o = 16;
#pragma unroll
  for (int n = N / 2; n >= 1; n >>= 1, o >>= 1) {
    const bool up = (l & o) != 0;
#pragma unroll
    for (int k = 0; k < n; ++k) {
      const float send = up ? v[k] : v[k + n], keep = up ? v[k + n] : v[k];
      v[k] = keep + __shfl_xor_sync(FULL_MASK, send, o);
    }
  }
#pragma unroll
  for (; o > 0; o >>= 1) v[0] += __shfl_xor_sync(FULL_MASK, v[0], o);
  return v[0];
}
template <int N> __device__ __forceinline__ constexpr int warp_multi_holder(int k) {
  return N == 8 ? 16 * ((k >> 2) & 1) + 8 * ((k >> 1) & 1) + 4 * (k & 1) : 16 * ((k >> 1) & 1) + 8 * (k & 1);
}

// T_b(lambda_obs) and dT_b/dlambda_obs of a tabulated filter
__device__ __forceinline__ void filter_tab_eval(const FilterTab& F, int b, float lam, float& Tv, float& dT) {
  Tv = 0.f; dT = 0.f;
  if (!(lam >= F.lo[b]) || !(lam <= F.hi[b])) return;
  const int bin = min((int)((lam - F.lo[b]) * F.inv_d[b]), SPS_FTAB_BINS - 1);
  int seg = __ldg(F.first + b * SPS_FTAB_BINS + bin);
  float4 k = __ldg(F.knots + seg);
  while (lam >= k.w && seg < F.last[b]) { ++seg; k = __ldg(F.knots + seg); }
  Tv = fmaf(lam - k.x, k.z, k.y); dT = k.z;
}

// launch counter (host side)
extern "C" int64_t sps_launch_count(void);
void sps_count_launch(int n = 1);
bool sps_prof_enabled();

// Programmatic dependent launch (griddepcontrol): a kernel launched with sps_launch() may start while the kernel before it
// in the stream is still draining; it must not touch that kernel's results before pdl_wait() (which returns once the
// preceding grid has completed and its writes are visible).  pdl_launch_dependents() would let the NEXT kernel's blocks be
// scheduled as soon as every block of this grid has issued it; no kernel here calls it (measured at 40,000 rows: early-
// resident blocks of the next kernel cost more than they save: contraction +7 us, prologue 0, epilogue -1), so a
// dependent kernel's launch overlaps the tail of the one before and its blocks start as the last ones exit.
// Both are no-ops under a plain launch.
#ifdef __CUDACC__
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
#endif
void sps_prof_begin(int id, cudaStream_t s);
void sps_prof_end(int id, cudaStream_t s);
void sps_set_error(const char* fmt, ...);
sps_status sps_check_cuda(cudaError_t e, const char* what);
