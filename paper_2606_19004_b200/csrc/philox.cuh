// philox.cuh - device functions of K1 shared by noise.cu (initial latents) and sde.cu (per-step noise):
// Philox4x32-10 and Box-Muller exactly as DESIGN.md S1-S2 state them.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

__device__ __forceinline__ uint4 philox4x32_10(uint4 c, uint2 k) {
#pragma unroll
  for (int r = 0; r < 10; ++r) {
    if (r > 0) { k.x += 0x9E3779B9u; k.y += 0xBB67AE85u; }
    uint32_t lo0 = 0xD2511F53u * c.x, hi0 = __umulhi(0xD2511F53u, c.x);
    uint32_t lo1 = 0xCD9E8D57u * c.z, hi1 = __umulhi(0xCD9E8D57u, c.z);
    c = make_uint4(hi1 ^ c.y ^ k.x, lo1, hi0 ^ c.w ^ k.y, lo0);
  }
  return c;
}

__device__ __forceinline__ float2 box_muller(uint32_t wa, uint32_t wb) {
  float u1 = (float)((wa >> 8) + 1u) * 5.9604644775390625e-08f;   // 2^-24, exact
  float u2x2 = (float)(wb >> 8) * 1.1920928955078125e-07f;        // 2*u2 = (wb>>8) * 2^-23, exact
  float rho = sqrtf(-2.0f * logf(u1));
  float s, c;
  sincospif(u2x2, &s, &c);                                        // angle 2*pi*u2 without rounding 2*pi*u2
  return make_float2(rho * c, rho * s);
}

