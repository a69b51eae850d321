// ORACLE — test infrastructure only.  Plain, slow, scalar CPU code written from the paper
// (arXiv 2106.12631, /root/reference/PAPER.md) and the public definitions it cites.  Shares no
// code with the CUDA path; only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
// --impl reference legs may use anything under oracle/.
//
// Philox4x32-10 counter-based generator and the u32 -> uniform map.
//
// Serves PAPER.md:78 / PAPER.md:108 (§3, §4: "generating all relevant random numbers (four per
// external particle) ... using the cuRAND library") and PAPER.md:80 (§3: the same sequence on CPU
// and GPU, bit-wise reproducible).  The paper does not name the generator; BASELINE.json's
// north_star fixes it to Philox (reading R1 in DESIGN.md).  The round function below is the
// public Random123 definition (Salmon, Moraes, Dror, Shaw, SC'11, "Parallel random numbers: as
// easy as 1, 2, 3"), written out step by step.
#pragma once
#include <cstdint>

namespace oracle {

// One Philox4x32 round:   (c0,c1,c2,c3) -> (hi(M1*c2)^c1^k0, lo(M1*c2), hi(M0*c0)^c3^k1, lo(M0*c0)).
inline void philox_round(uint32_t c[4], const uint32_t k[2]) {
  const uint64_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u;
  const uint64_t p0 = M0 * (uint64_t)c[0];
  const uint64_t p1 = M1 * (uint64_t)c[2];
  const uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
  const uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
  const uint32_t n0 = hi1 ^ c[1] ^ k[0];
  const uint32_t n1 = lo1;
  const uint32_t n2 = hi0 ^ c[3] ^ k[1];
  const uint32_t n3 = lo0;
  c[0] = n0; c[1] = n1; c[2] = n2; c[3] = n3;
}

// Ten rounds; the key is bumped by the Weyl constants after every round except the last.
inline void philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
  const uint32_t W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;
  uint32_t c[4] = {ctr[0], ctr[1], ctr[2], ctr[3]};
  uint32_t k[2] = {key[0], key[1]};
  for (int r = 0; r < 10; ++r) {
    philox_round(c, k);
    if (r != 9) { k[0] += W0; k[1] += W1; }
  }
  for (int i = 0; i < 4; ++i) out[i] = c[i];
}

// Reading R2: key = (seed_lo32, seed_hi32), counter = (event_lo32, event_hi32,
// i_final, 0) with `event` the GLOBAL event index; the four words are rho_1..rho_4 of that
// final-state particle ("four per external particle"; R4: only final particles need them).
inline void philox_event_particle(uint64_t seed, uint64_t event, uint32_t i_final, uint32_t out[4]) {
  const uint32_t ctr[4] = {(uint32_t)event, (uint32_t)(event >> 32), i_final, 0u};
  const uint32_t key[2] = {(uint32_t)seed, (uint32_t)(seed >> 32)};
  philox4x32_10(ctr, key, out);
}

// Reading R3: FP64  rho = (x + 0.5) * 2^-32 ;  FP32  rho = ((x >> 9) + 0.5) * 2^-23.
// Both are exact (no rounding) and lie strictly inside (0,1).
inline double u32_to_uniform_f64(uint32_t x) { return ((double)x + 0.5) * (1.0 / 4294967296.0); }
inline float u32_to_uniform_f32(uint32_t x) { return ((float)(x >> 9) + 0.5f) * (1.0f / 8388608.0f); }

}  // namespace oracle
