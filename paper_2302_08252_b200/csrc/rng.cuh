// Counter-based random numbers of the transport step (DESIGN.md rules R1-R3).
//
// BASELINE.json north_star: "draws the same Philox-4x32 random streams keyed by (track id, step,
// draw index)".  The paper's tracks carry a large stateful `RngState` (Fig. 3) and it
// observes that "photon physics requires far less random numbers"; a counter-based
// generator turns that observation into saved work: a block is only evaluated when a draw of it is
// consumed, and no generator state is ever loaded or stored.
#pragma once
#include <cstdint>

namespace adept {

// R1: Philox-4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11).  One 128-bit block per call.
__device__ __forceinline__ uint4 philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                               uint32_t k0, uint32_t k1) {
  constexpr uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u;
  constexpr uint32_t W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;
#pragma unroll
  for (int r = 0; r < 10; ++r) {
    const uint32_t hi0 = __umulhi(M0, c0), lo0 = M0 * c0;
    const uint32_t hi1 = __umulhi(M1, c2), lo1 = M1 * c2;
    c0 = hi1 ^ c1 ^ k0;
    c1 = lo1;
    c2 = hi0 ^ c3 ^ k1;
    c3 = lo0;
    k0 += W0;
    k1 += W1;
  }
  return make_uint4(c0, c1, c2, c3);
}

// R3: 32 random bits -> odd multiple of 2^-24 in (0, 1); exact, never 0 or 1.
__device__ __forceinline__ float u01(uint32_t x) {
  return static_cast<float>(2u * (x >> 9) + 1u) * 5.9604644775390625e-08f;
}

// R2: the stream of one track at one step.  key = track id, counter = (step, call, 0, 0).
//   call 0: words 0..2 re-sample nial[0..2]
//   call 1: word 0 energy sample, 1 Compton azimuth, 2 annihilation cos(theta), 3 annihilation azimuth
//   call 2: child ids, ordinal 0 = (x, y), ordinal 1 = (z, w)
struct Stream {
  uint32_t id_lo, id_hi, step;
  __device__ __forceinline__ uint4 call(uint32_t c) const {
    return philox4x32_10(step, c, 0u, 0u, id_lo, id_hi);
  }
};

// R4: id of the primary with global index p under a context seed.
__device__ __forceinline__ uint2 primary_id(unsigned long long p, unsigned long long seed) {
  const uint4 w = philox4x32_10(static_cast<uint32_t>(p), static_cast<uint32_t>(p >> 32), 0u, 0x5052494Du,
                                static_cast<uint32_t>(seed), static_cast<uint32_t>(seed >> 32));
  return make_uint2(w.x, w.y);
}

}  // namespace adept
