// Host evaluation of paper_1310_7087_b200/csrc/hb_math.cuh (the header compiles for the host as plain C++) against libm in
// long double: the error bounds its comment states.  Built and run by tests/test_hb_math.py; prints one line of maxima.
#include "../paper_1310_7087_b200/csrc/hb_math.cuh"
#include <cmath>
#include <cstdio>
#include <random>
using namespace qcd::hbm;

int main() {
  std::mt19937_64 rng(20241105);
  long double e_log = 0, e_c2 = 0, e_s = 0, e_c = 0, e_sq = 0, e_rs = 0, e_rc = 0;
  const long double PI = 3.14159265358979323846264338327950288L;
  auto check = [&](uint32_t w) {
    const long double u = ((long double)w + 0.5L) / 4294967296.0L;
    const long double c = cosl(2 * PI * u);
    long double d = fabsl((long double)log_uniform32(w) - logl(u));
    if (d > e_log) e_log = d;
    d = fabsl((long double)cos2_2pi_uniform32(w) - c * c);
    if (d > e_c2) e_c2 = d;
    double sn, cs;
    sincos_2pi_uniform32(w, &sn, &cs);
    d = fabsl((long double)sn - sinl(2 * PI * u));
    if (d > e_s) e_s = d;
    d = fabsl((long double)cs - c);
    if (d > e_c) e_c = d;
  };
  // every fold point of the integer reductions, both ends of the range, the sqrt(2) switch of the logarithm
  const uint32_t edges[] = {0x00000000u, 0x1fffffffu, 0x20000000u, 0x3fffffffu, 0x40000000u, 0x5fffffffu, 0x60000000u, 0x7fffffffu,
                            0x80000000u, 0x9fffffffu, 0xa0000000u, 0xbfffffffu, 0xc0000000u, 0xdfffffffu, 0xe0000000u, 0xffffffffu,
                            0x5a827999u, 0xb504f333u, 0x6a09e667u, 0x2d413cccu};
  for (uint32_t e : edges)
    for (int k = -2000; k <= 2000; ++k) check(e + (uint32_t)k);
  for (int i = 0; i < 1000000; ++i) check((uint32_t)rng());
  for (int i = 0; i < 1000000; ++i) {
    const double x = ldexp(1.0 + (double)(rng() >> 11) * 0x1p-53, (int)(rng() % 100) - 80);   // 2^-80 .. 2^20
    const long double s = sqrtl((long double)x);
    long double a = fabsl((long double)sqrt_pos(x) - s) / s;
    if (a > e_sq) e_sq = a;
    a = fabsl((long double)rsqrt(x) * s - 1);
    if (a > e_rs) e_rs = a;
    a = fabsl((long double)rcp(x) * (long double)x - 1);
    if (a > e_rc) e_rc = a;
  }
  printf("%.6Le %.6Le %.6Le %.6Le %.6Le %.6Le %.6Le %.17g %.17g\n", e_log, e_c2, e_s, e_c, e_sq, e_rs, e_rc, sqrt_pos(0.0), sqrt_pos(1e-310));
  return 0;
}
