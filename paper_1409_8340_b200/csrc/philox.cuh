// Philox4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11, Sec. 3.3), counter-based, in registers.
// The paper names no generator; BASELINE.json fixes Philox; readings S11' / S13 fix the
// counter/key assignment: key = (seed_lo, seed_hi), counter = (m_lo, m_hi, step, stream) with a
// global site index m; stream 0 = Langevin noise (ONE call per site pair: m = the even site, words
// (x0, x1) -> even site, (x2, x3) -> odd site), stream 1 = initial condition (one call per site).
#pragma once
#include <stdint.h>

struct PhiloxOut { uint32_t x0, x1, x2, x3; };

__device__ __forceinline__ PhiloxOut philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                                   uint32_t k0, uint32_t k1) {
  const uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u;   // round multipliers
  const uint32_t W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;   // Weyl key increments
#pragma unroll
  for (int r = 0; r < 10; ++r) {
    const uint32_t hi0 = __umulhi(M0, c0), lo0 = M0 * c0;
    const uint32_t hi1 = __umulhi(M1, c2), lo1 = M1 * c2;
    const uint32_t n0 = hi1 ^ c1 ^ k0, n2 = hi0 ^ c3 ^ k1;
    c0 = n0; c1 = lo1; c2 = n2; c3 = lo0;
    k0 += W0; k1 += W1;
  }
  PhiloxOut o; o.x0 = c0; o.x1 = c1; o.x2 = c2; o.x3 = c3;
  return o;
}

// uint32 -> uniform in (-1, 1): ((x >> 9) + 0.5) 2^-22 - 1, an odd multiple of 2^-23: exact in fp32 (S11).
__device__ __forceinline__ float u32_to_pm1(uint32_t x) {
  return (float)(int)((x >> 9) * 2u + 1u - (1u << 23)) * (1.0f / 8388608.0f);
}
// uint32 -> uniform in (0, 1): ((x >> 9) + 0.5) 2^-23 (S13), as a double.
__device__ __forceinline__ double u32_to_01(uint32_t x) {
  return ((double)(x >> 9) + 0.5) * (1.0 / 8388608.0);
}

// Langevin words of ONE site (reading S11'): the call of its pair, the words picked by the parity of m.  For kernels
// that own one site per thread; the marching kernels own whole pairs and use all four words of a call.
__device__ __forceinline__ void langevin_words(unsigned long long m, uint32_t step, uint32_t k0, uint32_t k1,
                                               uint32_t &re, uint32_t &im) {
  const unsigned long long me = m & ~1ull;
  const PhiloxOut p = philox4x32_10((uint32_t)me, (uint32_t)(me >> 32), step, 0u, k0, k1);
  re = (m & 1ull) ? p.x2 : p.x0;
  im = (m & 1ull) ? p.x3 : p.x1;
}
