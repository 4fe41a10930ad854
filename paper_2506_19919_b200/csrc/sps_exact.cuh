// sps_exact.cuh -- shared declarations of the exact-path kernels.
#pragma once
#include "sps_internal.h"

struct ExactState {
  float* W;        // [cap][ldw]  forward operand  W = Mn a (x) m
  float* Wbar;     // [cap][ldw]  reverse result
  float* part;     // [cap][5][SPS_MAX_BAND] band sums: flux and its direct partials (A_V, delta, F_floor, z)
  float* gbuf;     // [cap][SPS_MAX_BAND]    d logL / d flux_b
  int* sorted;     // [cap] rows of the current call ordered by redshift
  int* zhist;      // [2][1024] counting-sort histogram / cursors
  int64_t cap;
  int ldw;         // K padded to a multiple of 32
  bool use_tc;     // tcgen05 kernels available for this table shape
  void* tc;        // sps_exact_tc.cu state (tensor maps, split tables)
};

// tcgen05 path (sps_exact_tc.cu)
sps_status sps_exact_tc_setup(sps_table* t, int precision);
void sps_exact_tc_teardown(sps_table* t);
sps_status sps_exact_tc_ensure(sps_table* t, int64_t cap);
sps_status sps_exact_tc_forward(sps_table* t, int64_t n, const int* rows, cudaStream_t s);
sps_status sps_exact_tc_backward(sps_table* t, int64_t n, const int* rows, cudaStream_t s);
