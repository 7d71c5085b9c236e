// philox.cuh -- counter-based Philox4x32-10 (Salmon et al., SC'11) for the heatbath and the hot start.
// Mandated by BASELINE.json north_star in place of the paper's stateful PRNGCL generators:
// a counter-based stream keeps the paper's guarantee that one seed reproduces the run while
// making every (site, sub-step, draw) independent of thread count and launch shape.
// Keying (reading R7):  key = (seed lo, seed hi);  ctr = (lex site, sweep counter,
//   mu | parity<<4 | subgroup<<5 | hit<<8 | domain<<24,  draw).   domain 0 = heatbath, 1 = hot start.
#pragma once
#include <stdint.h>

namespace qcd {

struct Philox4 {
  uint32_t x, y, z, w;
};

__host__ __device__ __forceinline__ Philox4 philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t k0, uint32_t k1) {
  const uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u;
#pragma unroll
  for (int r = 0; r < 10; ++r) {
    const uint64_t p0 = (uint64_t)M0 * c0;
    const uint64_t p1 = (uint64_t)M1 * c2;
    const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
    const uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
    c1 = (uint32_t)p1;
    c3 = (uint32_t)p0;
    c0 = n0;
    c2 = n2;
    k0 += 0x9E3779B9u;
    k1 += 0xBB67AE85u;
  }
  Philox4 o; o.x = c0; o.y = c1; o.z = c2; o.w = c3;
  return o;
}

// The 20 round keys k0 + r W0, k1 + r W1 of a launch, computed once on the host: in the kernels they are constant-bank
// operands of the round's exclusive-or, where the per-call form above spends ~20 integer instructions on the schedule.
struct PhiloxKeys {
  uint32_t k[20];
};
inline PhiloxKeys philox_round_keys(uint32_t k0, uint32_t k1) {
  PhiloxKeys rk;
  for (int r = 0; r < 10; ++r) {
    rk.k[2 * r] = k0; rk.k[2 * r + 1] = k1;
    k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
  }
  return rk;
}
__device__ __forceinline__ Philox4 philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, const PhiloxKeys& rk) {
  const uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u;
#pragma unroll
  for (int r = 0; r < 10; ++r) {
    const uint64_t p0 = (uint64_t)M0 * c0;
    const uint64_t p1 = (uint64_t)M1 * c2;
    const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ rk.k[2 * r];
    const uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ rk.k[2 * r + 1];
    c1 = (uint32_t)p1;
    c3 = (uint32_t)p0;
    c0 = n0;
    c2 = n2;
  }
  Philox4 o; o.x = c0; o.y = c1; o.z = c2; o.w = c3;
  return o;
}

__host__ __device__ __forceinline__ uint32_t philox_c2(int mu, int parity, int sg, int hit, int domain) {
  return (uint32_t)mu | ((uint32_t)parity << 4) | ((uint32_t)sg << 5) | ((uint32_t)hit << 8) | ((uint32_t)domain << 24);
}

// word -> uniform strictly inside (0,1), exactly representable in the target precision (reading R8)
__device__ __forceinline__ double uniform64(uint32_t w) { return ((double)w + 0.5) * 2.3283064365386963e-10; }          // 2^-32
__device__ __forceinline__ double uniform23(uint32_t w) { return ((double)(w >> 9) + 0.5) * 1.1920928955078125e-07; }   // 2^-23
// the same fp32-mode uniform computed in float without an integer conversion: 1.m with m = w >> 9 is 1 + (w>>9) 2^-23,
// and subtracting 1 - 2^-24 gives (2 (w>>9) + 1) 2^-24, which has 24 significant bits: the subtraction is exact
__device__ __forceinline__ float uniform23f(uint32_t w) { return __uint_as_float(0x3F800000u | (w >> 9)) - 0.99999994f; }
template <typename R> __device__ __forceinline__ R uniform_real(uint32_t w);
template <> __device__ __forceinline__ float uniform_real<float>(uint32_t w) { return uniform23f(w); }
template <> __device__ __forceinline__ double uniform_real<double>(uint32_t w) { return uniform64(w); }
template <typename R> __device__ __forceinline__ double uniform_for(uint32_t w);
template <> __device__ __forceinline__ double uniform_for<float>(uint32_t w) { return uniform23(w); }
template <> __device__ __forceinline__ double uniform_for<double>(uint32_t w) { return uniform64(w); }

}  // namespace qcd
