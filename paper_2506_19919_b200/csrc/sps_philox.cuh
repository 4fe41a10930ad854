// sps_philox.cuh -- Philox4x32-10 counter-based generator (Salmon et al. 2011; R16).
// counter = (chain, transition, purpose, index), key = 64-bit seed.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

enum { RNG_MOMENTUM = 0, RNG_ACCEPT = 1, RNG_DIRECTION = 2, RNG_LEAF = 3, RNG_SUBTREE = 4, RNG_INIT = 5 };

__device__ __forceinline__ uint4 philox4x32_10(uint4 c, uint2 k) {
#pragma unroll
  for (int r = 0; r < 10; ++r) {
    const uint32_t hi0 = __umulhi(0xD2511F53u, c.x), lo0 = 0xD2511F53u * c.x;
    const uint32_t hi1 = __umulhi(0xCD9E8D57u, c.z), lo1 = 0xCD9E8D57u * c.z;
    c = make_uint4(hi1 ^ c.y ^ k.x, lo1, hi0 ^ c.w ^ k.y, lo0);
    k.x += 0x9E3779B9u; k.y += 0xBB67AE85u;
  }
  return c;
}
// u = ((x >> 8) + 0.5) 2^-24 : exact in fp32, never 0 or 1
__device__ __forceinline__ float philox_u01(uint32_t x) { return ((float)(x >> 8) + 0.5f) * 5.9604644775390625e-8f; }

// four standard normals from one counter block: Box-Muller on (u0,u1) and (u2,u3)
__device__ __forceinline__ float4 philox_normal4(uint4 c, uint2 k) {
  const uint4 w = philox4x32_10(c, k);
  const float r0 = sqrtf(-2.f * logf(philox_u01(w.x))), r1 = sqrtf(-2.f * logf(philox_u01(w.z)));
  float s0, c0, s1, c1;
  sincospif(2.f * philox_u01(w.y), &s0, &c0);
  sincospif(2.f * philox_u01(w.w), &s1, &c1);
  return make_float4(r0 * c0, r0 * s0, r1 * c1, r1 * s1);
}
