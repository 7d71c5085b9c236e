// sun_math.cuh -- register-resident SU(3) (3x3 complex) and SU(2) (quaternion) algebra for the update and
// measurement kernels.  Conventions follow DESIGN.md readings R3 (subgroup order), R6 (Gram-Schmidt) and the
// quaternion <-> matrix map  a = (a0,a1,a2,a3) <-> [[a0+i a3, a2+i a1],[-a2+i a1, a0-i a3]].
#pragma once
#include "common.cuh"

namespace qcd {

template <typename R> struct Cx { R re, im; };

template <typename R> __device__ __forceinline__ Cx<R> cx(R re, R im) { Cx<R> c; c.re = re; c.im = im; return c; }
// acc += a*b
template <typename R> __device__ __forceinline__ void cmad(Cx<R>& acc, const Cx<R>& a, const Cx<R>& b) {
  acc.re = q_fma(a.re, b.re, acc.re); acc.re = q_fma(-a.im, b.im, acc.re);
  acc.im = q_fma(a.re, b.im, acc.im); acc.im = q_fma(a.im, b.re, acc.im);
}
// acc += a*conj(b)
template <typename R> __device__ __forceinline__ void cmad_conj(Cx<R>& acc, const Cx<R>& a, const Cx<R>& b) {
  acc.re = q_fma(a.re, b.re, acc.re); acc.re = q_fma(a.im, b.im, acc.re);
  acc.im = q_fma(a.im, b.re, acc.im); acc.im = q_fma(-a.re, b.im, acc.im);
}
// acc += conj(a)*b
template <typename R> __device__ __forceinline__ void cmad_conja(Cx<R>& acc, const Cx<R>& a, const Cx<R>& b) {
  acc.re = q_fma(a.re, b.re, acc.re); acc.re = q_fma(a.im, b.im, acc.re);
  acc.im = q_fma(a.re, b.im, acc.im); acc.im = q_fma(-a.im, b.re, acc.im);
}
template <typename R> __device__ __forceinline__ Cx<R> cmul(const Cx<R>& a, const Cx<R>& b) {
  return cx<R>(a.re * b.re - a.im * b.im, a.re * b.im + a.im * b.re);
}

template <typename R> struct M3 { Cx<R> e[3][3]; };

// row 2 = conj(row0 x row1)   (valid for SU(3): third-row reconstruction of the 12-real compression)
template <typename R> __device__ __forceinline__ void m3_complete_row2(M3<R>& a) {
#pragma unroll
  for (int c = 0; c < 3; ++c) {
    const int c1 = (c + 1) % 3, c2 = (c + 2) % 3;
    // conj(a0[c1]*a1[c2] - a0[c2]*a1[c1])
    R re = a.e[0][c1].re * a.e[1][c2].re - a.e[0][c1].im * a.e[1][c2].im - a.e[0][c2].re * a.e[1][c1].re + a.e[0][c2].im * a.e[1][c1].im;
    R im = a.e[0][c1].re * a.e[1][c2].im + a.e[0][c1].im * a.e[1][c2].re - a.e[0][c2].re * a.e[1][c1].im - a.e[0][c2].im * a.e[1][c1].re;
    a.e[2][c].re = re; a.e[2][c].im = -im;
  }
}

// rows [0,NR) of  acc += a*b
template <typename R, int NR> __device__ __forceinline__ void m3_mad_nn(M3<R>& acc, const M3<R>& a, const M3<R>& b) {
#pragma unroll
  for (int i = 0; i < NR; ++i)
#pragma unroll
    for (int j = 0; j < 3; ++j)
#pragma unroll
      for (int k = 0; k < 3; ++k) cmad(acc.e[i][j], a.e[i][k], b.e[k][j]);
}
// rows [0,NR) of acc += a * b^dagger      (needs rows [0,NR) of a and ALL rows of b)
template <typename R, int NR> __device__ __forceinline__ void m3_mad_nd(M3<R>& acc, const M3<R>& a, const M3<R>& b) {
#pragma unroll
  for (int i = 0; i < NR; ++i)
#pragma unroll
    for (int j = 0; j < 3; ++j)
#pragma unroll
      for (int k = 0; k < 3; ++k) cmad_conj(acc.e[i][j], a.e[i][k], b.e[j][k]);
}
// rows [0,NR) of acc += a^dagger * b      (needs ALL rows of a and b)
template <typename R, int NR> __device__ __forceinline__ void m3_mad_dn(M3<R>& acc, const M3<R>& a, const M3<R>& b) {
#pragma unroll
  for (int i = 0; i < NR; ++i)
#pragma unroll
    for (int j = 0; j < 3; ++j)
#pragma unroll
      for (int k = 0; k < 3; ++k) cmad_conja(acc.e[i][j], a.e[k][i], b.e[k][j]);
}
template <typename R> __device__ __forceinline__ void m3_zero(M3<R>& a) {
#pragma unroll
  for (int i = 0; i < 3; ++i)
#pragma unroll
    for (int j = 0; j < 3; ++j) a.e[i][j] = cx<R>(R(0), R(0));
}

// Gram-Schmidt on rows 0,1; row 2 = conj(row0 x row1)  (reading R6)
template <typename R> __device__ __forceinline__ void m3_reunitarise(M3<R>& u) {
  R n0 = R(0);
#pragma unroll
  for (int c = 0; c < 3; ++c) n0 += u.e[0][c].re * u.e[0][c].re + u.e[0][c].im * u.e[0][c].im;
  R s0 = q_rsqrt(n0);
#pragma unroll
  for (int c = 0; c < 3; ++c) { u.e[0][c].re *= s0; u.e[0][c].im *= s0; }
  Cx<R> d = cx<R>(R(0), R(0));
#pragma unroll
  for (int c = 0; c < 3; ++c) cmad_conja(d, u.e[0][c], u.e[1][c]);   // d = sum conj(r0) r1
#pragma unroll
  for (int c = 0; c < 3; ++c) {
    u.e[1][c].re -= d.re * u.e[0][c].re - d.im * u.e[0][c].im;
    u.e[1][c].im -= d.re * u.e[0][c].im + d.im * u.e[0][c].re;
  }
  R n1 = R(0);
#pragma unroll
  for (int c = 0; c < 3; ++c) n1 += u.e[1][c].re * u.e[1][c].re + u.e[1][c].im * u.e[1][c].im;
  R s1 = q_rsqrt(n1);
#pragma unroll
  for (int c = 0; c < 3; ++c) { u.e[1][c].re *= s1; u.e[1][c].im *= s1; }
  m3_complete_row2(u);
}

// reals <-> matrix (row-major, re then im); NREAL = 12 fills rows 0,1 only
template <typename R, int NREAL> __device__ __forceinline__ void m3_from_reals(M3<R>& u, const R* r) {
#pragma unroll
  for (int e = 0; e < NREAL / 2; ++e) { u.e[e / 3][e % 3].re = r[2 * e]; u.e[e / 3][e % 3].im = r[2 * e + 1]; }
}
template <typename R, int NREAL> __device__ __forceinline__ void m3_to_reals(const M3<R>& u, R* r) {
#pragma unroll
  for (int e = 0; e < NREAL / 2; ++e) { r[2 * e] = u.e[e / 3][e % 3].re; r[2 * e + 1] = u.e[e / 3][e % 3].im; }
}

// ------------------------------------------------------------------ quaternions (SU(2))
template <typename R> struct Q4 { R a0, a1, a2, a3; };
template <typename R> __device__ __forceinline__ Q4<R> q4(R a0, R a1, R a2, R a3) { Q4<R> q; q.a0 = a0; q.a1 = a1; q.a2 = a2; q.a3 = a3; return q; }
// (a.b)_0 = a0 b0 - a.b ;  vec(a.b) = a0 b + b0 a - a x b
template <typename R> __device__ __forceinline__ Q4<R> q4_mul(const Q4<R>& a, const Q4<R>& b) {
  Q4<R> r;
  r.a0 = a.a0 * b.a0 - a.a1 * b.a1 - a.a2 * b.a2 - a.a3 * b.a3;
  r.a1 = a.a0 * b.a1 + b.a0 * a.a1 - (a.a2 * b.a3 - a.a3 * b.a2);
  r.a2 = a.a0 * b.a2 + b.a0 * a.a2 - (a.a3 * b.a1 - a.a1 * b.a3);
  r.a3 = a.a0 * b.a3 + b.a0 * a.a3 - (a.a1 * b.a2 - a.a2 * b.a1);
  return r;
}
template <typename R> __device__ __forceinline__ Q4<R> q4_conj(const Q4<R>& a) { return q4<R>(a.a0, -a.a1, -a.a2, -a.a3); }
template <typename R> __device__ __forceinline__ Q4<R> q4_add(const Q4<R>& a, const Q4<R>& b) {
  return q4<R>(a.a0 + b.a0, a.a1 + b.a1, a.a2 + b.a2, a.a3 + b.a3);
}

}  // namespace qcd
