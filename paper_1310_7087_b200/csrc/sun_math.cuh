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

// ---- complex dot products, the unit every 3x3 product here is made of
//   cdot3<MODE>(acc, a0,a1,a2, b0,b1,b2):  acc += sum_k op(a_k, b_k),   NN: a*b   ND: a*conj(b)   DN: conj(a)*b
//   cdot2<MODE>: the same over two terms, result returned (not accumulated)
enum { CD_NN = 0, CD_ND = 1, CD_DN = 2 };
template <int MODE, typename R>
__device__ __forceinline__ void cdot3(Cx<R>& acc, const Cx<R>& a0, const Cx<R>& a1, const Cx<R>& a2, const Cx<R>& b0, const Cx<R>& b1,
                                      const Cx<R>& b2) {
  if (MODE == CD_NN) { cmad(acc, a0, b0); cmad(acc, a1, b1); cmad(acc, a2, b2); }
  else if (MODE == CD_ND) { cmad_conj(acc, a0, b0); cmad_conj(acc, a1, b1); cmad_conj(acc, a2, b2); }
  else { cmad_conja(acc, a0, b0); cmad_conja(acc, a1, b1); cmad_conja(acc, a2, b2); }
}
template <typename R> __device__ __forceinline__ Cx<R> cdot2_nn(const Cx<R>& a0, const Cx<R>& a1, const Cx<R>& b0, const Cx<R>& b1) {
  Cx<R> r = cmul(a0, b0);
  cmad(r, a1, b1);
  return r;
}

// fp32: the packed FP32x2 pipe of sm_100 (FFMA2 / FMUL2 work on an aligned register pair; ptxas folds the scalar broadcast
// (a.re, a.re) and the swap (b.im, b.re) into operand modifiers, but not a sign on one half).  So the real-part and
// imaginary-part coefficients are summed in two packed accumulators
//     T1 = sum_k a_k.re * (b_k.re, b_k.im)        T2 = sum_k a_k.im * (b_k.im, b_k.re)
// and the signs are applied once per dot product:  NN (T1.x - T2.x, T1.y + T2.y)   ND (T1.x + T2.x, T2.y - T1.y)
// DN (T1.x + T2.x, T1.y - T2.y):  8 issue slots per 3-term dot product instead of 12.
__device__ __forceinline__ float2 f2_bcast(float x) { return make_float2(x, x); }
__device__ __forceinline__ float2 f2_of(const Cx<float>& c) { return make_float2(c.re, c.im); }
__device__ __forceinline__ float2 f2_swap(const Cx<float>& c) { return make_float2(c.im, c.re); }
// Sign application of a packed complex product in ONE issue slot: an FFMA2 with the constant pair (-1, +1) or (+1, -1)
// instead of two scalar FADDs.  t * (+-1) + u is exact, so the results are bit-identical; 8 % fewer instructions per
// link, the same FMA-pipe cycles (measured: -5 % in a register-resident microbenchmark, neutral in the update kernels).
//   NN (t1.x - t2.x, t1.y + t2.y)    ND (t1.x + t2.x, t2.y - t1.y)    DN (t1.x + t2.x, t1.y - t2.y)
template <int MODE> __device__ __forceinline__ Cx<float> f2_signs(const float2& t1, const float2& t2) {
  const float2 S = make_float2(-1.0f, 1.0f), Sn = make_float2(1.0f, -1.0f);
  const float2 v = (MODE == 0) ? __ffma2_rn(t2, S, t1) : (MODE == 1) ? __ffma2_rn(t1, Sn, t2) : __ffma2_rn(t2, Sn, t1);
  Cx<float> r; r.re = v.x; r.im = v.y;
  return r;
}
template <int MODE>
__device__ __forceinline__ void cdot3(Cx<float>& acc, const Cx<float>& a0, const Cx<float>& a1, const Cx<float>& a2, const Cx<float>& b0,
                                      const Cx<float>& b1, const Cx<float>& b2) {
  float2 t1 = make_float2(acc.re, MODE == CD_ND ? -acc.im : acc.im);
  t1 = __ffma2_rn(f2_bcast(a0.re), f2_of(b0), t1);
  t1 = __ffma2_rn(f2_bcast(a1.re), f2_of(b1), t1);
  t1 = __ffma2_rn(f2_bcast(a2.re), f2_of(b2), t1);
  float2 t2 = __fmul2_rn(f2_bcast(a0.im), f2_swap(b0));
  t2 = __ffma2_rn(f2_bcast(a1.im), f2_swap(b1), t2);
  t2 = __ffma2_rn(f2_bcast(a2.im), f2_swap(b2), t2);
  acc = f2_signs<MODE>(t1, t2);
}
__device__ __forceinline__ Cx<float> cdot2_nn(const Cx<float>& a0, const Cx<float>& a1, const Cx<float>& b0, const Cx<float>& b1) {
  float2 t1 = __fmul2_rn(f2_bcast(a0.re), f2_of(b0));
  t1 = __ffma2_rn(f2_bcast(a1.re), f2_of(b1), t1);
  float2 t2 = __fmul2_rn(f2_bcast(a0.im), f2_swap(b0));
  t2 = __ffma2_rn(f2_bcast(a1.im), f2_swap(b1), t2);
  return f2_signs<CD_NN>(t1, t2);
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

// fp32: each component conj(p*q - r*s) as two packed accumulators, 6 issue slots instead of 8
__device__ __forceinline__ void m3_complete_row2(M3<float>& a) {
#pragma unroll
  for (int c = 0; c < 3; ++c) {
    const int c1 = (c + 1) % 3, c2 = (c + 2) % 3;
    const Cx<float>&p = a.e[0][c1], &q = a.e[1][c2], &r = a.e[0][c2], &s = a.e[1][c1];
    float2 t1 = __fmul2_rn(f2_bcast(p.re), f2_of(q));
    t1 = __ffma2_rn(f2_bcast(-r.re), f2_of(s), t1);
    float2 t2 = __fmul2_rn(f2_bcast(p.im), f2_swap(q));
    t2 = __ffma2_rn(f2_bcast(-r.im), f2_swap(s), t2);
    const float2 v = __ffma2_rn(t1, make_float2(1.0f, -1.0f), make_float2(-t2.x, -t2.y));   // (t1.x - t2.x, -t1.y - t2.y)
    a.e[2][c].re = v.x;
    a.e[2][c].im = v.y;
  }
}

// ---- staple accumulation with the third row summed in its unreduced form.
// Every staple S is in SU(3), so its row 2 is conj(S0 x S1); the sum A = sum S needs the sum of those rows.  Instead of
// rebuilding row 2 of each staple and adding it (per component: the cross product, its sign combination, an add), the
// products of the cross product are accumulated over the staples directly:
//   generic:  A[2][c] += conj(S[0][c1] S[1][c2] - S[0][c2] S[1][c1])        8 multiply-adds per component, nothing else
//   float:    two packed running sums per component; the sign combination is applied ONCE per link (finish)
// finish() ADDS the accumulated row to A's row 2 (which may already hold directly accumulated contributions).
template <typename R> struct Row2Sum {
  __device__ __forceinline__ void zero() {}
  __device__ __forceinline__ void add(M3<R>& A, const M3<R>& S) {
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      const int c1 = (c + 1) % 3, c2 = (c + 2) % 3;
      const Cx<R>&p = S.e[0][c1], &q = S.e[1][c2], &r = S.e[0][c2], &s = S.e[1][c1];
      R re = A.e[2][c].re, im = A.e[2][c].im;
      re = q_fma(p.re, q.re, re); re = q_fma(-p.im, q.im, re); re = q_fma(-r.re, s.re, re); re = q_fma(r.im, s.im, re);
      im = q_fma(-p.re, q.im, im); im = q_fma(-p.im, q.re, im); im = q_fma(r.re, s.im, im); im = q_fma(r.im, s.re, im);
      A.e[2][c].re = re; A.e[2][c].im = im;
    }
  }
  __device__ __forceinline__ void finish(M3<R>&) const {}
};
template <> struct Row2Sum<float> {
  float2 t1[3], t2[3];
  __device__ __forceinline__ void zero() {
#pragma unroll
    for (int c = 0; c < 3; ++c) { t1[c] = make_float2(0.0f, 0.0f); t2[c] = make_float2(0.0f, 0.0f); }
  }
  __device__ __forceinline__ void add(M3<float>&, const M3<float>& S) {
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      const int c1 = (c + 1) % 3, c2 = (c + 2) % 3;
      const Cx<float>&p = S.e[0][c1], &q = S.e[1][c2], &r = S.e[0][c2], &s = S.e[1][c1];
      t1[c] = __ffma2_rn(f2_bcast(p.re), f2_of(q), t1[c]);
      t1[c] = __ffma2_rn(f2_bcast(-r.re), f2_of(s), t1[c]);
      t2[c] = __ffma2_rn(f2_bcast(p.im), f2_swap(q), t2[c]);
      t2[c] = __ffma2_rn(f2_bcast(-r.im), f2_swap(s), t2[c]);
    }
  }
  __device__ __forceinline__ void finish(M3<float>& A) const {
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      float2 v = __ffma2_rn(t1[c], make_float2(1.0f, -1.0f), make_float2(-t2[c].x, -t2[c].y));   // (t1.x - t2.x, -t1.y - t2.y)
      v = __fadd2_rn(v, f2_of(A.e[2][c]));
      A.e[2][c].re = v.x; A.e[2][c].im = v.y;
    }
  }
};
// rows 0,1 of a += rows 0,1 of s
__device__ __forceinline__ void m3_add_rows01(M3<float>& a, const M3<float>& s) {
#pragma unroll
  for (int r = 0; r < 2; ++r)
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      const float2 v = __fadd2_rn(f2_of(a.e[r][c]), f2_of(s.e[r][c]));
      a.e[r][c].re = v.x; a.e[r][c].im = v.y;
    }
}
template <typename R> __device__ __forceinline__ void m3_add_rows01(M3<R>& a, const M3<R>& s) {
#pragma unroll
  for (int r = 0; r < 2; ++r)
#pragma unroll
    for (int c = 0; c < 3; ++c) { a.e[r][c].re += s.e[r][c].re; a.e[r][c].im += s.e[r][c].im; }
}

// The three product shapes, rows [0,NR) of acc += op(a) op(b), written as outer-product accumulation over k: the six
// consecutive multiply-adds that follow share the scalar a.re (then a.im) in the same operand slot, which lets the
// register-operand reuse cache serve it (the FP32 pipe is bounded by register-file reads).
//   SA, SB select the element of a / b:  nn: a[i][k] b[k][j]   nd: a[i][k] conj(b[j][k])   dn: conj(a[k][i]) b[k][j]
template <int NR, int MODE, typename R> __device__ __forceinline__ void m3_mad(M3<R>& acc, const M3<R>& a, const M3<R>& b) {
#pragma unroll
  for (int k = 0; k < 3; ++k)
#pragma unroll
    for (int i = 0; i < NR; ++i) {
      const Cx<R> x = (MODE == CD_DN) ? a.e[k][i] : a.e[i][k];
      const R are = x.re, aim = (MODE == CD_DN) ? -x.im : x.im;
#pragma unroll
      for (int j = 0; j < 3; ++j) {
        const Cx<R> y = (MODE == CD_ND) ? b.e[j][k] : b.e[k][j];
        const R bim = (MODE == CD_ND) ? -y.im : y.im;
        acc.e[i][j].re = q_fma(are, y.re, acc.e[i][j].re);
        acc.e[i][j].im = q_fma(are, bim, acc.e[i][j].im);
      }
#pragma unroll
      for (int j = 0; j < 3; ++j) {
        const Cx<R> y = (MODE == CD_ND) ? b.e[j][k] : b.e[k][j];
        const R bim = (MODE == CD_ND) ? -y.im : y.im;
        acc.e[i][j].re = q_fma(-aim, bim, acc.e[i][j].re);
        acc.e[i][j].im = q_fma(aim, y.re, acc.e[i][j].im);
      }
    }
}
// fp32 packed: per (i,j) two accumulators T1 += a.re * (b.re, b.im), T2 += a.im * (b.im, b.re), same k-outer order
template <int NR, int MODE> __device__ __forceinline__ void m3_mad(M3<float>& acc, const M3<float>& a, const M3<float>& b) {
  float2 t1[NR][3], t2[NR][3];
#pragma unroll
  for (int i = 0; i < NR; ++i)
#pragma unroll
    for (int j = 0; j < 3; ++j) t1[i][j] = make_float2(acc.e[i][j].re, MODE == CD_ND ? -acc.e[i][j].im : acc.e[i][j].im);
#pragma unroll
  for (int k = 0; k < 3; ++k)
#pragma unroll
    for (int i = 0; i < NR; ++i) {
      const Cx<float> x = (MODE == CD_DN) ? a.e[k][i] : a.e[i][k];
#pragma unroll
      for (int j = 0; j < 3; ++j) {
        const Cx<float> y = (MODE == CD_ND) ? b.e[j][k] : b.e[k][j];
        t1[i][j] = __ffma2_rn(f2_bcast(x.re), f2_of(y), t1[i][j]);
      }
#pragma unroll
      for (int j = 0; j < 3; ++j) {
        const Cx<float> y = (MODE == CD_ND) ? b.e[j][k] : b.e[k][j];
        t2[i][j] = (k == 0) ? __fmul2_rn(f2_bcast(x.im), f2_swap(y)) : __ffma2_rn(f2_bcast(x.im), f2_swap(y), t2[i][j]);
      }
    }
#pragma unroll
  for (int i = 0; i < NR; ++i)
#pragma unroll
    for (int j = 0; j < 3; ++j) {
      acc.e[i][j] = f2_signs<MODE>(t1[i][j], t2[i][j]);
    }
}
template <typename R, int NR> __device__ __forceinline__ void m3_mad_nn(M3<R>& acc, const M3<R>& a, const M3<R>& b) { m3_mad<NR, CD_NN>(acc, a, b); }
// rows [0,NR) of acc += a * b^dagger      (needs rows [0,NR) of a and ALL rows of b)
template <typename R, int NR> __device__ __forceinline__ void m3_mad_nd(M3<R>& acc, const M3<R>& a, const M3<R>& b) { m3_mad<NR, CD_ND>(acc, a, b); }
// rows [0,NR) of acc += a^dagger * b      (needs ALL rows of a and b)
template <typename R, int NR> __device__ __forceinline__ void m3_mad_dn(M3<R>& acc, const M3<R>& a, const M3<R>& b) { m3_mad<NR, CD_DN>(acc, a, b); }
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

// fp32: the same steps on the packed pipe (32 issue slots instead of 60)
__device__ __forceinline__ void m3_reunitarise(M3<float>& u) {
  auto norm2 = [&](int r) {
    float2 t = __fmul2_rn(f2_of(u.e[r][0]), f2_of(u.e[r][0]));
    t = __ffma2_rn(f2_of(u.e[r][1]), f2_of(u.e[r][1]), t);
    t = __ffma2_rn(f2_of(u.e[r][2]), f2_of(u.e[r][2]), t);
    return t.x + t.y;
  };
  auto scale = [&](int r, float sc) {
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      const float2 v = __fmul2_rn(f2_bcast(sc), f2_of(u.e[r][c]));
      u.e[r][c].re = v.x; u.e[r][c].im = v.y;
    }
  };
  scale(0, q_rsqrt(norm2(0)));
  Cx<float> d = cx<float>(0.0f, 0.0f);
  cdot3<CD_DN>(d, u.e[0][0], u.e[0][1], u.e[0][2], u.e[1][0], u.e[1][1], u.e[1][2]);   // d = sum conj(r0) r1
#pragma unroll
  for (int c = 0; c < 3; ++c) {                                    // r1 -= d r0
    const float2 t1 = __ffma2_rn(f2_bcast(-d.re), f2_of(u.e[0][c]), f2_of(u.e[1][c]));
    const float2 t2 = __fmul2_rn(f2_bcast(d.im), f2_swap(u.e[0][c]));
    const float2 v = __ffma2_rn(t2, make_float2(1.0f, -1.0f), t1);   // (t1.x + d.im r0.im, t1.y - d.im r0.re)
    u.e[1][c].re = v.x; u.e[1][c].im = v.y;
  }
  scale(1, q_rsqrt(norm2(1)));
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
