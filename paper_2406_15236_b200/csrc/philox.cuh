// Philox-4x32-10 counter-based generator for the CUDA path (host + device).
// Stream layout: key = (seed_lo, seed_hi), counter = (index, sub, step, tag).
// The CPU oracle re-types the same definition on its own; nothing here is shared with it.
#pragma once
#include <stdint.h>

namespace mpc {

enum : uint32_t { TAG_SHIFT = 0, TAG_AXIS = 1, TAG_MBS = 2, TAG_AT = 3, TAG_WALL = 4, TAG_PHANTOM = 5 };

struct Block4 { uint32_t a, b, c, d; };

__host__ __device__ __forceinline__ uint32_t mul_hi32(uint32_t x, uint32_t y) {
#ifdef __CUDA_ARCH__
  return __umulhi(x, y);
#else
  return (uint32_t)(((unsigned long long)x * (unsigned long long)y) >> 32);
#endif
}

__host__ __device__ __forceinline__ Block4 philox(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                                  uint32_t k0, uint32_t k1) {
#pragma unroll
  for (int round = 0; round < 10; ++round) {
    const uint32_t h0 = mul_hi32(0xD2511F53u, c0), l0 = 0xD2511F53u * c0;
    const uint32_t h1 = mul_hi32(0xCD9E8D57u, c2), l1 = 0xCD9E8D57u * c2;
    const uint32_t y0 = h1 ^ c1 ^ k0, y2 = h0 ^ c3 ^ k1;
    c0 = y0; c1 = l1; c2 = y2; c3 = l0;
    k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
  }
  return Block4{c0, c1, c2, c3};
}

// Same generator with the ten round keys precomputed (round r uses key + r * bump): one 3-input
// LOP3 per output word and no key arithmetic in the loop. rk = { k0_0..k0_9, k1_0..k1_9 }.
__host__ __device__ __forceinline__ void philox_round_keys(uint32_t k0, uint32_t k1, uint32_t (&rk)[20]) {
  for (int r = 0; r < 10; ++r) { rk[r] = k0 + (uint32_t)r * 0x9E3779B9u; rk[10 + r] = k1 + (uint32_t)r * 0xBB67AE85u; }
}
__host__ __device__ __forceinline__ Block4 philox_rk(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                                     const uint32_t (&rk)[20]) {
#pragma unroll
  for (int round = 0; round < 10; ++round) {
    const uint32_t h0 = mul_hi32(0xD2511F53u, c0), l0 = 0xD2511F53u * c0;
    const uint32_t h1 = mul_hi32(0xCD9E8D57u, c2), l1 = 0xCD9E8D57u * c2;
    const uint32_t y0 = h1 ^ c1 ^ rk[round], y2 = h0 ^ c3 ^ rk[10 + round];
    c0 = y0; c1 = l1; c2 = y2; c3 = l0;
  }
  return Block4{c0, c1, c2, c3};
}

// top 24 bits -> [0,1) and (0,1]; both conversions are exact in fp32
__host__ __device__ __forceinline__ float u01_co(uint32_t w) { return (float)(w >> 8) * 5.9604644775390625e-08f; }
__host__ __device__ __forceinline__ float u01_oc(uint32_t w) { return (float)((w >> 8) + 1u) * 5.9604644775390625e-08f; }

#ifdef __CUDACC__
// three standard normals from one block (Box-Muller on word pairs (a,b) and (c,d))
__device__ __forceinline__ void normals3(const Block4& o, float& g0, float& g1, float& g2) {
  const float r0 = sqrtf(-2.0f * logf(u01_oc(o.a)));
  const float r1 = sqrtf(-2.0f * logf(u01_oc(o.c)));
  float s0, c0, c1;
  sincospif(2.0f * u01_co(o.b), &s0, &c0);
  c1 = cospif(2.0f * u01_co(o.d));
  g0 = r0 * c0; g1 = r0 * s0; g2 = r1 * c1;
}
#endif

}  // namespace mpc
