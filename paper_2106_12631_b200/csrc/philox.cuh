// philox.cuh — Philox4x32-10 on the device (step A1) and the u32 -> uniform map (step A2).
// PAPER.md:78/:108 (§3/§4: random numbers, "four per external particle")
// (reproducibility); generator fixed by BASELINE.json north_star (reading R1).  Round function:
// Salmon et al., SC'11.  Counter/key mapping R2, uniform map R3.
#pragma once
#include <stdint.h>
#include "cx.cuh"

namespace mg {

struct u32x4 { uint32_t x, y, z, w; };

// counter (c0,c1,c2,c3), key (k0,k1); ten rounds, key bumped by the Weyl constants between rounds.
__device__ __forceinline__ u32x4 philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                               uint32_t k0, uint32_t k1) {
  constexpr uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u, W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;
#pragma unroll
  for (int r = 0; r < 10; ++r) {
    const uint32_t hi0 = __umulhi(M0, c0), lo0 = M0 * c0;
    const uint32_t hi1 = __umulhi(M1, c2), lo1 = M1 * c2;
    c0 = hi1 ^ c1 ^ k0;
    c1 = lo1;
    c2 = hi0 ^ c3 ^ k1;
    c3 = lo0;
    k0 += W0;  // the bump after the last round is dead code and is removed by the compiler
    k1 += W1;
  }
  return u32x4{c0, c1, c2, c3};
}

// R2: key = seed, counter = (event_lo, event_hi, i_final, 0); `event` is the GLOBAL event index.
__device__ __forceinline__ u32x4 philox_event_particle(uint64_t seed, uint64_t event, uint32_t i_final) {
  return philox4x32_10((uint32_t)event, (uint32_t)(event >> 32), i_final, 0u,
                       (uint32_t)seed, (uint32_t)(seed >> 32));
}

// R3, exact in both precisions (no rounding anywhere):
//   FP64: (x + 0.5) * 2^-32.  Built without an int->double conversion: the double with bit pattern
//         0x43300000:x is 2^52 + x; (that - 2^52) * 2^-32 + 2^-33.
//   FP32: ((x>>9) + 0.5) * 2^-23.  The float 0x3F800000 | (x>>9) is 1 + (x>>9) 2^-23; subtracting
//         (1 - 2^-24) is exact (Sterbenz) and gives ((x>>9) + 0.5) 2^-23.
template <class T> __device__ __forceinline__ T u32_to_uniform(uint32_t x);
template <> __device__ __forceinline__ double u32_to_uniform<double>(uint32_t x) {
  const double d = __hiloint2double(0x43300000, (int)x) - 4503599627370496.0;
  return fma(d, 2.3283064365386963e-10 /* 2^-32 */, 1.1641532182693481e-10 /* 2^-33 */);
}
template <> __device__ __forceinline__ float u32_to_uniform<float>(uint32_t x) {
  return __uint_as_float(0x3F800000u | (x >> 9)) - 0.99999994f /* 1 - 2^-24 */;
}

}  // namespace mg
