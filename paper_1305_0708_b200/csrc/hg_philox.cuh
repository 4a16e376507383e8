// hg_philox.cuh -- counter-based uniforms for the phase-space generator (step a1).
//
// Role of List 1 `xorshift.cu` (Appendix B): one independent stream of doubles per
// phase-space point.  The paper seeds a per-thread xorshift128 from (thread, iteration); BASELINE.json
// mandates a counter-based Philox instead, so a point's numbers depend only on (seed, event index) and a
// batch can be split or replayed at will (reading SURVEY.md 8c-A15):
//     key     = (seed_lo, seed_hi)
//     counter = (event_lo, event_hi, block j, process id)
//     draw d  = words (2d mod 4, 2d+1 mod 4) of block floor(d/2):  lo, hi
//     u       = ((hi >> 6) * 2^26 + (lo >> 6) + 1/2) * 2^-52   in the open interval (0,1)
// Philox4x32-10 is the published algorithm of Salmon et al. (multipliers 0xD2511F53 / 0xCD9E8D57, Weyl
// increments 0x9E3779B9 / 0xBB67AE85, ten rounds).
#pragma once
#include <stdint.h>

#include "hg_cx.cuh"

namespace hg {

struct U4 {
  uint32_t x, y, z, w;
};

HG_HD void mulhilo(uint32_t a, uint32_t b, uint32_t& hi, uint32_t& lo) {
#if defined(__CUDA_ARCH__)
  hi = __umulhi(a, b);
  lo = a * b;
#else
  uint64_t p = (uint64_t)a * (uint64_t)b;
  hi = (uint32_t)(p >> 32);
  lo = (uint32_t)p;
#endif
}

HG_HD U4 philox4x32_10(U4 c, uint32_t k0, uint32_t k1) {
#pragma unroll
  for (int r = 0; r < 10; ++r) {
    uint32_t hi0, lo0, hi1, lo1;
    mulhilo(0xD2511F53u, c.x, hi0, lo0);
    mulhilo(0xCD9E8D57u, c.z, hi1, lo1);
    U4 n;
    n.x = hi1 ^ c.y ^ k0;
    n.y = lo1;
    n.z = hi0 ^ c.w ^ k1;
    n.w = lo0;
    c = n;
    k0 += 0x9E3779B9u;
    k1 += 0xBB67AE85u;
  }
  return c;
}

HG_HD double u52(uint32_t lo, uint32_t hi) {
  // exact in fp64: the mantissa is < 2^52, +1/2 keeps it representable, the scale is a power of two
  uint64_t m = ((uint64_t)(hi >> 6) << 26) + (uint64_t)(lo >> 6);
  return ((double)m + 0.5) * 2.220446049250313e-16;  // 2^-52
}

// Fills u[0..ND) with the draws of one event.
template <int ND>
HG_HD void draw_uniforms(uint64_t seed, uint64_t event, uint32_t pid, double* u) {
  const uint32_t k0 = (uint32_t)seed, k1 = (uint32_t)(seed >> 32);
#pragma unroll
  for (int j = 0; j < (ND + 1) / 2; ++j) {
    U4 c;
    c.x = (uint32_t)event;
    c.y = (uint32_t)(event >> 32);
    c.z = (uint32_t)j;
    c.w = pid;
    U4 r = philox4x32_10(c, k0, k1);
    u[2 * j] = u52(r.x, r.y);
    if (2 * j + 1 < ND) u[2 * j + 1] = u52(r.z, r.w);
  }
}

}  // namespace hg
