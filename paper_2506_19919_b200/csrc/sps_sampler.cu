// sps_sampler.cu -- counter-based RNG, leapfrog, HMC / NUTS engine.  [RNG only for now]
#include "sps_internal.h"
#include "sps_philox.cuh"

__global__ void philox_words_kernel(uint32_t k0, uint32_t k1, uint32_t first_chain, uint32_t transition, uint32_t purpose,
                                    uint32_t index, int64_t n, uint32_t* out) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  uint4 w = philox4x32_10(make_uint4(first_chain + (uint32_t)i, transition, purpose, index), make_uint2(k0, k1));
  reinterpret_cast<uint4*>(out)[i] = w;
}

extern "C" sps_status sps_philox_words(uint64_t seed, uint32_t first_chain, uint32_t transition, uint32_t purpose,
                                       uint32_t index, int64_t n, uint32_t* out, void* stream) {
  if (!out || n < 0) { sps_set_error("sps_philox_words: bad argument"); return SPS_EINVAL; }
  if (n == 0) return SPS_OK;
  sps_status st = sps_require_device(); if (st != SPS_OK) return st;
  philox_words_kernel<<<(unsigned)((n + 255) / 256), 256, 0, (cudaStream_t)stream>>>((uint32_t)seed, (uint32_t)(seed >> 32), first_chain,
                                                                                 transition, purpose, index, n, out);
  sps_count_launch();
  return sps_check_cuda(cudaGetLastError(), "philox launch");
}
