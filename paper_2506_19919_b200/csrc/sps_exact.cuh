// sps_exact.cuh -- shared declarations of the exact-path kernels.
#pragma once
#include "sps_internal.h"

struct ExactState {
  float* W;        // [cap][ldw]  forward operand  W = Mn a (x) m
  float* Wbar;     // [cap][ldw]  reverse result
  float* part;     // [cap][5][SPS_MAX_BAND] band sums: flux and its direct partials (A_V, delta, F_floor, z)
  float* gbuf;     // [cap][SPS_MAX_BAND]    d logL / d flux_b
  int64_t cap;
  int ldw;         // K padded to a multiple of 32
  bool use_tc;     // tcgen05 kernels available for this table shape
  void* tc;        // sps_exact_tc.cu state (tensor maps, split tables)
};
