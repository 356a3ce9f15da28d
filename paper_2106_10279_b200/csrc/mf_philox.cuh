// mf_philox.cuh — step a1/a2 of the hot path: counter-based random numbers.
//
// Philox4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11; named by BASELINE.json north_star; PAPER.md L61 says
// only "generation of random numbers").  Stream layout (R1): key = (seed lo, seed hi),
// counter = (event lo, event hi, iteration, block).  Block b yields VEGAS dimensions 2b and 2b+1;
// block 0xFFFFFFFF yields the accept draw of the unweighting stage.
#pragma once
#include "mf_common.cuh"

namespace mf {

struct U4 { uint32_t x, y, z, w; };

MF_HD void mulhilo(uint32_t a, uint32_t b, uint32_t& hi, uint32_t& lo) {
#if defined(__CUDA_ARCH__)
  lo = a * b;
  hi = __umulhi(a, b);
#else
  uint64_t p = (uint64_t)a * (uint64_t)b;
  lo = (uint32_t)p;
  hi = (uint32_t)(p >> 32);
#endif
}

MF_HD U4 philox4x32_10(U4 c, uint32_t k0, uint32_t k1) {
#pragma unroll
  for (int r = 0; r < 10; ++r) {
    uint32_t h0, l0, h1, l1;
    mulhilo(0xD2511F53u, c.x, h0, l0);
    mulhilo(0xCD9E8D57u, c.z, h1, l1);
    U4 n;
    n.x = h1 ^ c.y ^ k0;
    n.y = l1;
    n.z = h0 ^ c.w ^ k1;
    n.w = l0;
    c = n;
    k0 += 0x9E3779B9u;  // Weyl bumps; the one after round 10 is unused
    k1 += 0xBB67AE85u;
  }
  return c;
}

MF_HD U4 philox_block(uint64_t seed, uint32_t iteration, uint64_t event, uint32_t block) {
  U4 c;
  c.x = (uint32_t)event;
  c.y = (uint32_t)(event >> 32);
  c.z = iteration;
  c.w = block;
  return philox4x32_10(c, (uint32_t)seed, (uint32_t)(seed >> 32));
}

// Two words -> uniform in (0,1) (R2): 52-bit mantissa m = hi*2^20 | lo>>12, u = (2m+1) 2^-53.
// Exact in binary64: no rounding anywhere, so CPU and GPU agree bit for bit.
MF_HD double uniform52(uint32_t hi, uint32_t lo) {
  uint64_t m = ((uint64_t)hi << 20) | (uint64_t)(lo >> 12);
  return (double)(long long)(2 * m + 1) * 0x1.0p-53;
}

}  // namespace mf
