// sps_exact.cuh -- shared declarations of the exact-path kernels.
#pragma once
#include "sps_internal.h"

// Table-constant state of the exact path (built by sps_create_table, immutable afterwards).
struct ExactState {
  int ldw;         // K padded: row pitch of W / Wbar
  bool use_tc;     // tcgen05 kernels available for this table shape
  void* tc;        // sps_exact_tc.cu: split SSP tables, their TMA maps, filter constants
};

// ---- band sums as fixed-point integers ----------------------------------------------------------------------------
// A row's five band sums (flux and its direct partials w.r.t. A_V, delta, F_floor, z) are accumulated across wavelength
// tiles by many warps.  They are added as 64-bit integers (value * 2^k rounded), so the result does not depend on the
// order of the additions or on which rows share a tile: exact-path fluxes are bit-reproducible.  Every sum c is bounded
// by 2^PART_SHIFT[c] * Mn * T.part_bound (weights sum to one, F_att <= 1, T_b <= max transmission), so the scale
// 2^(61 - shift_c) / pow2ceil(Mn part_bound) cannot overflow, and it resolves 2^-41 or better of Mn part_bound.
__device__ __forceinline__ float part_scale(float Mn, float part_bound, int shift) {
  const int E = min(max((int)((__float_as_uint(Mn * part_bound) >> 23) & 0xffu), 64), 250);      // biased exponent
  return __uint_as_float((uint32_t)min(max(314 - shift - E, 1), 254) << 23);
}
__device__ __forceinline__ void part_add(long long* p, float v, float scale) {
  if (v != 0.f) atomicAdd(reinterpret_cast<unsigned long long*>(p), (unsigned long long)__float2ll_rn(v * scale));
}
__device__ __forceinline__ float part_read(const long long* p, float scale) { return (float)((double)(*p) / (double)scale); }
#define PART_SHIFT_FLUX 0
#define PART_SHIFT_AV 10
#define PART_SHIFT_DELTA 14
#define PART_SHIFT_FFLOOR 0
// (the z partial's shift is a table constant: TableDev.part_shift_z)

// tcgen05 path (sps_exact_tc.cu)
sps_status sps_exact_tc_setup(sps_table* t, int precision);
void sps_exact_tc_teardown(sps_table* t);
sps_status sps_exact_tc_ensure(const sps_table* t, ExactScratch& X, int64_t cap);
void sps_exact_tc_free_scratch(ExactScratch& X);
sps_status sps_exact_tc_forward(const sps_table* t, Workspace& ws, int64_t n, const int* rows, cudaStream_t s);
sps_status sps_exact_tc_backward(const sps_table* t, Workspace& ws, int64_t n, const int* rows, cudaStream_t s);
