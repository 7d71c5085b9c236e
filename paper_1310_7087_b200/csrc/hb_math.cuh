// hb_math.cuh -- double-precision elementary functions of the Kennedy-Pendleton heatbath, specialised to their actual
// arguments: uniforms (w + 1/2) 2^-32 built from one 32-bit Philox word (reading R8) and radicands / divisors that are
// positive normal numbers.
//
// Why (profiles/r2_a_launches_and_ncu.md): the fp64 heatbath kernel spent ~1500 of its ~4800 instructions per link in the
// library's log / cospi / sincospi / sqrt / rsqrt -- 104 per log, 48 per cospi, 72 per sincospi, 25 per sqrt, each with
// special-case paths (denormals, infinities, huge arguments) that cannot occur here and that keep the compiler from
// interleaving the 15 independent evaluations of a link.  The forms below are branch-free and do the argument reduction
// in INTEGER arithmetic on the Philox word, where it is exact:
//     ln u             u = n 2^-33, n = 2w+1 odd:  n = 2^e m, m in [sqrt(1/2), sqrt 2);  ln m = 2 atanh(s), s = (m-1)/(m+1)
//     cos^2(2 pi u)    period 1/2 and even about 1/4: folded on the integer n to +-cos(pi t), t in (0, 1/2)
//     sin, cos(2 pi u) quadrant and octant from the top bits of n, t in (0, 1/4]
// All polynomials are plain Taylor series (coefficient tables below, each stating its formula), truncated where the
// remainder is below 1e-17.  Errors, measured by tests/test_hb_math.py (this header compiled for the host, against libm
// in long double over 10^6 random words and +-2000 words around every fold point): ln u 2.5e-15 absolute (|ln u| <= 22.9,
// i.e. 0.7 units in the last place of the result), cos^2 / sin / cos 2e-16 absolute, sqrt / rsqrt / rcp 1.4e-16
// relative; the same bounds on the device through qcd_debug_hb_math (`test_heatbath_functions_on_the_device_against_libm`).
// The link tolerance against the fp64 oracle is 1e-12, and an accept decision changes only if its margin is
// below these errors (probability ~1e-15 per trial).
#pragma once
#include <stdint.h>

#ifdef __CUDACC__
#define HBM_FN __host__ __device__ __forceinline__
#else
#include <cmath>
#include <cstring>
#define HBM_FN inline
#endif

namespace qcd {
namespace hbm {

// ---- bit access and ~20-bit hardware seeds (device: MUFU.RCP64H / MUFU.RSQ64H; host: float arithmetic, 24 bits, so the
// host evaluation of the same refinement steps is representative)
HBM_FN int hi32(double x) {
#ifdef __CUDA_ARCH__
  return __double2hiint(x);
#else
  uint64_t u; memcpy(&u, &x, 8); return (int)(u >> 32);
#endif
}
HBM_FN int lo32(double x) {
#ifdef __CUDA_ARCH__
  return __double2loint(x);
#else
  uint64_t u; memcpy(&u, &x, 8); return (int)(u & 0xffffffffu);
#endif
}
HBM_FN double make_double(int hi, int lo) {
#ifdef __CUDA_ARCH__
  return __hiloint2double(hi, lo);
#else
  uint64_t u = ((uint64_t)(uint32_t)hi << 32) | (uint32_t)lo; double x; memcpy(&x, &u, 8); return x;
#endif
}
HBM_FN double seed_rcp(double d) {
#ifdef __CUDA_ARCH__
  double r; asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(d)); return r;
#else
  // 20 leading bits, like the hardware seed
  return make_double(hi32((double)(1.0f / (float)d)) , 0);
#endif
}
HBM_FN double seed_rsqrt(double d) {
#ifdef __CUDA_ARCH__
  double r; asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(d)); return r;
#else
  return make_double(hi32(1.0 / std::sqrt(d)), 0);
#endif
}
HBM_FN double fma_(double a, double b, double c) {
#ifdef __CUDA_ARCH__
  return __fma_rn(a, b, c);
#else
  return std::fma(a, b, c);
#endif
}

// ---- Taylor coefficients.  On the device they live in the constant bank, where a DFMA reads them as an operand (as
// literals every coefficient costs two uniform-register moves).
#define HBM_ATANH_TABLE {1.0 / 3.0, 1.0 / 5.0, 1.0 / 7.0, 1.0 / 9.0, 1.0 / 11.0, 1.0 / 13.0, 1.0 / 15.0, 1.0 / 17.0, 1.0 / 19.0}
// (-1)^j pi^(2j) / (2j)!, j = 1 .. 11
#define HBM_COS_TABLE                                                                                                       \
  {-4.93480220054467900e+00, 4.05871212641676848e+00, -1.33526276885458950e+00, 2.35330630358893206e-01,                    \
   -2.58068913900140612e-02, 1.92957430940392314e-03, -1.04638104924845705e-04, 4.30306958703294729e-06,                    \
   -1.38789524622137714e-07, 3.60473079746250112e-09, -7.70070713060135385e-11}
// (-1)^j pi^(2j+1) / (2j+1)!, j = 0 .. 8
#define HBM_SIN_TABLE                                                                                                       \
  {3.14159265358979312e+00, -5.16771278004997026e+00, 2.55016403987734552e+00, -5.99264529320792105e-01,                    \
   8.21458866111282326e-02, -7.37043094571435044e-03, 4.66302805767612554e-04, -2.19153534478302173e-05,                    \
   7.95205400147551261e-07}
#ifdef __CUDACC__
static __constant__ double c_atanh[9] = HBM_ATANH_TABLE;
static __constant__ double c_cos[11] = HBM_COS_TABLE;
static __constant__ double c_sin[9] = HBM_SIN_TABLE;
#endif
static const double h_atanh[9] = HBM_ATANH_TABLE;
static const double h_cos[11] = HBM_COS_TABLE;
static const double h_sin[9] = HBM_SIN_TABLE;
#ifdef __CUDA_ARCH__
#define HBM_ATANH(i) c_atanh[i]
#define HBM_COS(i) c_cos[i]
#define HBM_SIN(i) c_sin[i]
#else
#define HBM_ATANH(i) h_atanh[i]
#define HBM_COS(i) h_cos[i]
#define HBM_SIN(i) h_sin[i]
#endif

// 1/d, d normal and positive: seed (20 bits), two Newton steps (-> 40 -> 80 bits)
HBM_FN double rcp(double d) {
  double r = seed_rcp(d);
  double e = fma_(-d, r, 1.0);
  r = fma_(r, e, r);
  e = fma_(-d, r, 1.0);
  return fma_(r, e, r);
}
// x^-1/2, x normal and positive: seed, two Newton steps y += y (1/2 - x y^2 / 2)
HBM_FN double rsqrt(double x) {
  double y = seed_rsqrt(x);
  double e = fma_(-x * y, 0.5 * y, 0.5);
  y = fma_(y, e, y);
  e = fma_(-x * y, 0.5 * y, 0.5);
  y = fma_(y, e, y);
  e = fma_(-x * y, 0.5 * y, 0.5);
  return fma_(y, e, y);
}
// sqrt(x), x >= 0 (below 1e-300: 0): coupled iteration g -> sqrt x, h -> 1 / (2 sqrt x), then one correction of g
HBM_FN double sqrt_pos(double x) {
  const bool ok = x > 1e-300;
  const double xs = ok ? x : 1.0;
  const double y = seed_rsqrt(xs);
  double g = xs * y, h = 0.5 * y;
  double e = fma_(-g, h, 0.5);
  g = fma_(g, e, g); h = fma_(h, e, h);
  e = fma_(-g, h, 0.5);
  g = fma_(g, e, g); h = fma_(h, e, h);
  g = fma_(fma_(-g, g, xs), h, g);                         // g += (x - g^2) / (2 g)
  return ok ? g : 0.0;
}

// ---- ln((w + 1/2) 2^-32)
HBM_FN double log_uniform32(uint32_t w) {
  const double x = fma_((double)w, 2.0, 1.0);            // n = 2w+1, exact
  int hi = hi32(x);
  int e = (hi >> 20) - 1023;
  hi = (hi & 0x000fffff) | 0x3ff00000;                     // m in [1, 2)
  const int up = hi > 0x3ff6a09e ? 1 : 0;                  // m above sqrt 2 (to its 20 leading bits): halve it
  hi -= up << 20;
  e += up;
  const double m = make_double(hi, lo32(x));
  const double f = m - 1.0;                                // exact; f in [-0.2929, 0.4143)
  const double d = 2.0 + f;
  const double r = rcp(d);
  double s = f * r;
  s = fma_(fma_(-d, s, f), r, s);                          // s = f / d, correctly rounded or one ulp off
  const double z = s * s;                                  // z <= 0.02944
  // 2 atanh(s) = 2 s (1 + z/3 + z^2/5 + ... + z^9/19); remainder 2 s z^10 / 21 < 1e-17
  double p = HBM_ATANH(8);
#pragma unroll
  for (int i = 7; i >= 0; --i) p = fma_(p, z, HBM_ATANH(i));
  const double s2 = s + s;
  const double lnm = fma_(s2, p * z, s2);
  return fma_((double)(e - 33), 0.69314718055994531, lnm);   // + (e - 33) ln 2
}

// cos(pi t), t in [0, 1/2]: sum_j (-1)^j pi^(2j)/(2j)! t^(2j), j <= 11; remainder (pi/2)^24/24! < 1e-19
HBM_FN double cospi_series_half(double t) {
  const double z = t * t;
  double p = HBM_COS(10);                                  // j = 11
#pragma unroll
  for (int i = 9; i >= 0; --i) p = fma_(p, z, HBM_COS(i));
  return fma_(p, z, 1.0);
}

// cos^2(2 pi u), u = (w + 1/2) 2^-32 = n 2^-33.  cos^2 = (1 + cos(4 pi u)) / 2 and 4 pi u = 2 pi k / 2^32 with
// k = n mod 2^32 (odd); cos(2 pi - x) = cos x folds k to (0, 2^31), cos(pi - x) = -cos x to (0, 2^30): k stays odd, so
// no fold point is ever hit and every step is exact.
HBM_FN double cos2_2pi_uniform32(uint32_t w) {
  uint32_t k = (w << 1) | 1u;
  k = (k & 0x80000000u) ? (0u - k) : k;                    // k in (0, 2^31)
  const bool neg = (k & 0x40000000u) != 0;
  k = neg ? (0x80000000u - k) : k;                         // k in (0, 2^30)
  const double t = (double)k * 4.656612873077392578125e-10;   // k 2^-31: cos(pi t), t in (0, 1/2)
  const double c = cospi_series_half(t);
  return fma_(neg ? -0.5 : 0.5, c, 0.5);
}

// sin(2 pi u) and cos(2 pi u), u = n 2^-33: the angle is (pi/2)(q + r 2^-31), q = n >> 31 the quadrant, r = n mod 2^31
// (odd); inside the quadrant sin(pi/2 - x) = cos x folds r to (0, 2^30].  t = r 2^-32 in (0, 1/4].
//   sin(pi t) = t sum_j (-1)^j pi^(2j+1)/(2j+1)! t^(2j), j <= 8   (remainder (pi/4)^19/19! < 1e-19)
//   cos(pi t) =   sum_j (-1)^j pi^(2j)/(2j)! t^(2j),     j <= 8   (remainder (pi/4)^18/18! < 3e-18)
HBM_FN void sincos_2pi_uniform32(uint32_t w, double* sn, double* cs) {
  const uint32_t q = w >> 30;
  uint32_t r = ((w << 1) | 1u) & 0x7fffffffu;
  const bool swap = r > 0x40000000u;
  r = swap ? (0x80000000u - r) : r;
  const double t = (double)r * 2.3283064365386962890625e-10;  // r 2^-32
  const double z = t * t;
  double ps = HBM_SIN(8), pc = HBM_COS(7);                 // j = 8 in both series
#pragma unroll
  for (int i = 7; i >= 0; --i) ps = fma_(ps, z, HBM_SIN(i));
#pragma unroll
  for (int i = 6; i >= 0; --i) pc = fma_(pc, z, HBM_COS(i));
  const double s0 = ps * t;
  const double c0 = fma_(pc, z, 1.0);
  const double sq = swap ? c0 : s0, cq = swap ? s0 : c0;  // sin, cos of the angle inside the quadrant
  // quadrant: 0 (s, c)   1 (c, -s)   2 (-s, -c)   3 (-c, s)
  const double a = (q & 1u) ? cq : sq, b = (q & 1u) ? sq : cq;
  *sn = (q & 2u) ? -a : a;
  *cs = (q == 1u || q == 2u) ? -b : b;
}

}  // namespace hbm
}  // namespace qcd
