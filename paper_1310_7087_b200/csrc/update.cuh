// update.cuh -- the hot path: one (parity, mu) sub-step of the checkerboard sweep, one thread per link.
//   staple sum (2(D-1) staples, optional abelian field factor)  -> SURVEY 8(a)-3, 8(a)-4; PAPER.md:108 (checkerboard)
//   Cabibbo-Marinari over SU(2) subgroups: Kennedy-Pendleton heatbath ("(pseudo)heat-bath", NHIT trial cap,
//   PAPER.md:108, :134) or overrelaxation (BASELINE.json north_star)                       -> 8(a)-5, 8(a)-6
//   reunitarise + store ("reunitarization")                                   -> 8(a)-7
// A sub-step writes only U_mu on parity p and reads it only at the thread's own site, so it is race-free.
#pragma once
#include "common.cuh"
#include "philox.cuh"
#include "sun_math.cuh"

namespace qcd {

struct FieldArgs {   // F = diag(exp(i theta_c)) on plane (mu,nu), mu<nu; cos/sin precomputed on the host in double
  int mu, nu;
  double c[3], s[3];
};

struct UpdateArgs {
  double beta;
  int parity, mu, hit, max_trials;
  uint32_t sweep, key0, key1;
  uint8_t* trials;   // NULL or [lex][3] debug trial codes
  FieldArgs f;
};

// ------------------------------------------------------------------ Kennedy-Pendleton draw of g0 (reading R5)
// The accept decision is taken in double in both precisions so that it agrees with the fp64 oracle whenever
// alpha agrees; the uniforms are exactly representable in the storage precision (R8).
template <typename R>
__device__ __forceinline__ bool kp_draw(double alpha, uint32_t lex, const UpdateArgs& a, int sg, double& g0, int& code) {
  const uint32_t c2 = philox_c2(a.mu, a.parity, sg, a.hit, 0);
  const double inv_alpha = 1.0 / alpha;
  for (int t = 0; t < a.max_trials; ++t) {
    const Philox4 w = philox4x32_10(lex, a.sweep, c2, 1u + (uint32_t)t, a.key0, a.key1);
    const double r1 = uniform_for<R>(w.x), r2 = uniform_for<R>(w.y), r3 = uniform_for<R>(w.z), r4 = uniform_for<R>(w.w);
    const double c = cospi(2.0 * r2);
    const double delta = -(log(r1) + c * c * log(r3)) * inv_alpha;
    if (r4 * r4 <= 1.0 - 0.5 * delta) { g0 = 1.0 - delta; code = t + 1; return true; }
  }
  code = 0x80 | a.max_trials;
  return false;
}

// quaternion a of the subgroup update from the projected v = proj(W) (not normalised), k2 = |v|^2
template <typename R, int KIND, int NC>
__device__ __forceinline__ bool subgroup_quaternion(const Q4<R>& v, R k2, uint32_t lex, const UpdateArgs& a, int sg, Q4<R>& out, int& code) {
  if (KIND == 1) {
    // overrelaxation: a = (vt^dagger)^2 = (v0^2 - |vec v|^2, -2 v0 vec v) / k^2
    const R inv = q_rcp(k2);
    const R vv = v.a1 * v.a1 + v.a2 * v.a2 + v.a3 * v.a3;
    const R m2 = R(-2) * v.a0 * inv;
    out = q4<R>((v.a0 * v.a0 - vv) * inv, m2 * v.a1, m2 * v.a2, m2 * v.a3);
    return true;
  } else {
    const R rk = q_rsqrt(k2);
    const R k = k2 * rk;
    const double alpha = 2.0 * a.beta * (double)k / (double)NC;
    double g0d;
    if (!kp_draw<R>(alpha, lex, a, sg, g0d, code)) return false;
    const Philox4 w = philox4x32_10(lex, a.sweep, philox_c2(a.mu, a.parity, sg, a.hit, 0), 0u, a.key0, a.key1);
    const R u1 = (R)uniform_for<R>(w.x), u2 = (R)uniform_for<R>(w.y);
    const R g0 = (R)g0d;
    const R ct = R(1) - R(2) * u1;
    const R st = q_sqrt(R(1) - ct * ct);
    R sphi, cphi;
    q_sincospi(R(2) * u2, &sphi, &cphi);
    const R rr = q_sqrt(fmax(R(0), R(1) - g0 * g0));
    const Q4<R> g = q4<R>(g0, rr * st * cphi, rr * st * sphi, rr * ct);
    const Q4<R> vtc = q4<R>(v.a0 * rk, -v.a1 * rk, -v.a2 * rk, -v.a3 * rk);   // vt^dagger
    out = q4_mul(g, vtc);
    return true;
  }
}

template <typename R> struct Tiny;
template <> struct Tiny<float> { static __device__ __forceinline__ float k2() { return 1e-20f; } };
template <> struct Tiny<double> { static __device__ __forceinline__ double k2() { return 1e-30; } };

// =====================================================================================
// SU(3)
// =====================================================================================
template <typename R, bool COMP> struct Su3Store { static constexpr int NREAL = COMP ? 12 : 18; };

// load a link; ROW2: make sure row 2 is valid (reconstructed when compressed)
template <typename R, bool COMP, bool NC, bool ROW2>
__device__ __forceinline__ void su3_load(M3<R>& u, const typename PlaneTraits<R, (COMP ? 12 : 18)>::Vec* __restrict__ links,
                                         const Geom& g, size_t base, uint32_t h) {
  constexpr int NREAL = COMP ? 12 : 18;
  R r[NREAL];
  load_reals<R, NREAL, NC>(links, g, base, h, r);
  m3_from_reals<R, NREAL>(u, r);
  if (COMP && ROW2) m3_complete_row2(u);
}

// one Cabibbo-Marinari subgroup hit on rows (I,J) of U given the staple sum A
template <typename R, int KIND, int I, int J>
__device__ __forceinline__ void su3_subgroup_hit(M3<R>& U, const M3<R>& A, uint32_t lex, const UpdateArgs& a, int sg, int& code) {
  Cx<R> wii = cx<R>(0, 0), wij = cx<R>(0, 0), wji = cx<R>(0, 0), wjj = cx<R>(0, 0);
#pragma unroll
  for (int k = 0; k < 3; ++k) {
    cmad(wii, U.e[I][k], A.e[k][I]); cmad(wij, U.e[I][k], A.e[k][J]);
    cmad(wji, U.e[J][k], A.e[k][I]); cmad(wjj, U.e[J][k], A.e[k][J]);
  }
  Q4<R> v;
  v.a0 = R(0.5) * (wii.re + wjj.re);
  v.a1 = R(0.5) * (wij.im + wji.im);
  v.a2 = R(0.5) * (wij.re - wji.re);
  v.a3 = R(0.5) * (wii.im - wjj.im);
  const R k2 = v.a0 * v.a0 + v.a1 * v.a1 + v.a2 * v.a2 + v.a3 * v.a3;
  code = 0;
  if (k2 < Tiny<R>::k2()) return;                    // reading R4
  Q4<R> q;
  if (!subgroup_quaternion<R, KIND, 3>(v, k2, lex, a, sg, q, code)) return;
  const Cx<R> aii = cx<R>(q.a0, q.a3), aij = cx<R>(q.a2, q.a1), aji = cx<R>(-q.a2, q.a1), ajj = cx<R>(q.a0, -q.a3);
#pragma unroll
  for (int c = 0; c < 3; ++c) {
    const Cx<R> ui = U.e[I][c], uj = U.e[J][c];
    Cx<R> ni = cmul(aii, ui); cmad(ni, aij, uj);
    Cx<R> nj = cmul(aji, ui); cmad(nj, ajj, uj);
    U.e[I][c] = ni; U.e[J][c] = nj;
  }
}

// scale column c of m by exp(+-i theta_c)
template <typename R> __device__ __forceinline__ void su3_scale_cols(M3<R>& m, const FieldArgs& f, bool conj) {
#pragma unroll
  for (int c = 0; c < 3; ++c) {
    const Cx<R> ph = cx<R>((R)f.c[c], conj ? -(R)f.s[c] : (R)f.s[c]);
#pragma unroll
    for (int i = 0; i < 3; ++i) m.e[i][c] = cmul(m.e[i][c], ph);
  }
}
template <typename R> __device__ __forceinline__ void su3_scale_rows(M3<R>& m, const FieldArgs& f, bool conj) {
#pragma unroll
  for (int r = 0; r < 3; ++r) {
    const Cx<R> ph = cx<R>((R)f.c[r], conj ? -(R)f.s[r] : (R)f.s[r]);
#pragma unroll
    for (int j = 0; j < 3; ++j) m.e[r][j] = cmul(m.e[r][j], ph);
  }
}

template <typename R, int D, bool COMP, int KIND, bool FIELD>
__global__ void __launch_bounds__(128)
su3_update_kernel(Geom g, typename PlaneTraits<R, (COMP ? 12 : 18)>::Vec* links, UpdateArgs a) {
  typedef PlaneTraits<R, (COMP ? 12 : 18)> T;
  constexpr int NREAL = COMP ? 12 : 18;
  const uint32_t h = blockIdx.x * blockDim.x + threadIdx.x;
  if (h >= g.Vh) return;
  const int p = a.parity, mu = a.mu, q = 1 - p;
  const SiteCoord sc = decode_site(g, h, p);
  int fmu, bmu;
  nbr_offsets(g, sc, mu, fmu, bmu);

  M3<R> A;
  m3_zero(A);
  const typename T::Vec* __restrict__ ro = links;   // neighbour arrays are never written in this sub-step
#pragma unroll
  for (int i = 0; i < D - 1; ++i) {
    const int nu = i + (i >= mu ? 1 : 0);
    int fnu, bnu;
    nbr_offsets(g, sc, nu, fnu, bnu);
    int fsign = 0;   // +1: field role "first direction" (F on upper, F^+ in lower); -1: "second direction"
    if (FIELD) fsign = (mu == a.f.mu && nu == a.f.nu) ? 1 : (mu == a.f.nu && nu == a.f.mu) ? -1 : 0;
    {
      // upper staple  U_nu(x+mu) U_mu(x+nu)^+ U_nu(x)^+ = U1 (U3 U2)^+
      M3<R> U1, U2, U3, X, S;
      su3_load<R, COMP, true, !COMP>(U1, ro, g, array_base<T::NP>(g, D, q, nu), h + fmu);
      su3_load<R, COMP, true, true>(U2, ro, g, array_base<T::NP>(g, D, q, mu), h + fnu);
      su3_load<R, COMP, true, !COMP>(U3, ro, g, array_base<T::NP>(g, D, p, nu), h);
      m3_zero(X);
      if (COMP) {
        m3_mad_nn<R, 2>(X, U3, U2); m3_complete_row2(X);
        if (FIELD && fsign != 0) {
          m3_zero(S); m3_mad_nd<R, 2>(S, U1, X); m3_complete_row2(S);
          su3_scale_cols(S, a.f, fsign < 0);
#pragma unroll
          for (int r = 0; r < 3; ++r)
#pragma unroll
            for (int c = 0; c < 3; ++c) { A.e[r][c].re += S.e[r][c].re; A.e[r][c].im += S.e[r][c].im; }
        } else {
          m3_zero(S); m3_mad_nd<R, 2>(S, U1, X); m3_complete_row2(S);
#pragma unroll
          for (int r = 0; r < 3; ++r)
#pragma unroll
            for (int c = 0; c < 3; ++c) { A.e[r][c].re += S.e[r][c].re; A.e[r][c].im += S.e[r][c].im; }
        }
      } else {
        m3_mad_nn<R, 3>(X, U3, U2);
        if (FIELD && fsign != 0) {
          m3_zero(S); m3_mad_nd<R, 3>(S, U1, X);
          su3_scale_cols(S, a.f, fsign < 0);
#pragma unroll
          for (int r = 0; r < 3; ++r)
#pragma unroll
            for (int c = 0; c < 3; ++c) { A.e[r][c].re += S.e[r][c].re; A.e[r][c].im += S.e[r][c].im; }
        } else {
          m3_mad_nd<R, 3>(A, U1, X);
        }
      }
    }
    {
      // lower staple  U_nu(x+mu-nu)^+ U_mu(x-nu)^+ [F^+|F] U_nu(x-nu) = (U2 U1)^+ [F^+|F] U3
      M3<R> U1, U2, U3, Y;
      su3_load<R, COMP, true, true>(U1, ro, g, array_base<T::NP>(g, D, p, nu), h + fmu + bnu);
      su3_load<R, COMP, true, !COMP>(U2, ro, g, array_base<T::NP>(g, D, q, mu), h + bnu);
      su3_load<R, COMP, true, true>(U3, ro, g, array_base<T::NP>(g, D, q, nu), h + bnu);
      if (FIELD && fsign != 0) su3_scale_rows(U3, a.f, fsign > 0);   // first direction: F^+ U3 ; second: F U3
      m3_zero(Y);
      if (COMP) {
        M3<R> S;
        m3_mad_nn<R, 2>(Y, U2, U1); m3_complete_row2(Y);
        m3_zero(S); m3_mad_dn<R, 2>(S, Y, U3); m3_complete_row2(S);
#pragma unroll
        for (int r = 0; r < 3; ++r)
#pragma unroll
          for (int c = 0; c < 3; ++c) { A.e[r][c].re += S.e[r][c].re; A.e[r][c].im += S.e[r][c].im; }
      } else {
        m3_mad_nn<R, 3>(Y, U2, U1);
        m3_mad_dn<R, 3>(A, Y, U3);
      }
    }
  }

  // own link (plain load: this array is written by this kernel, each thread only its own element)
  M3<R> U;
  const size_t own = array_base<T::NP>(g, D, p, mu);
  su3_load<R, COMP, false, true>(U, links, g, own, h);

  const uint32_t lex = 2u * h + (uint32_t)sc.s;
  int c0, c1, c2;
  su3_subgroup_hit<R, KIND, 0, 1>(U, A, lex, a, 0, c0);
  su3_subgroup_hit<R, KIND, 0, 2>(U, A, lex, a, 1, c1);
  su3_subgroup_hit<R, KIND, 1, 2>(U, A, lex, a, 2, c2);
  m3_reunitarise(U);

  R r[NREAL];
  m3_to_reals<R, NREAL>(U, r);
  store_reals<R, NREAL>(links, g, own, h, r);
  if (KIND == 0 && a.trials) {
    a.trials[(size_t)lex * 3 + 0] = (uint8_t)c0; a.trials[(size_t)lex * 3 + 1] = (uint8_t)c1; a.trials[(size_t)lex * 3 + 2] = (uint8_t)c2;
  }
}

// =====================================================================================
// SU(2): links are unit quaternions; staples and updates stay in the quaternion algebra.
// The field factor F = diag(e^{i th}, e^{-i th}) is the quaternion (cos th, 0, 0, sin th).
// =====================================================================================
template <typename R, bool NC>
__device__ __forceinline__ Q4<R> su2_load(const typename PlaneTraits<R, 4>::Vec* __restrict__ links, const Geom& g, size_t base, uint32_t h) {
  R r[4];
  load_reals<R, 4, NC>(links, g, base, h, r);
  return q4<R>(r[0], r[1], r[2], r[3]);
}

template <typename R, int D, int KIND, bool FIELD>
__global__ void __launch_bounds__(256)
su2_update_kernel(Geom g, typename PlaneTraits<R, 4>::Vec* links, UpdateArgs a) {
  typedef PlaneTraits<R, 4> T;
  const uint32_t h = blockIdx.x * blockDim.x + threadIdx.x;
  if (h >= g.Vh) return;
  const int p = a.parity, mu = a.mu, q = 1 - p;
  const SiteCoord sc = decode_site(g, h, p);
  int fmu, bmu;
  nbr_offsets(g, sc, mu, fmu, bmu);
  const typename T::Vec* __restrict__ ro = links;
  Q4<R> A = q4<R>(0, 0, 0, 0);
#pragma unroll
  for (int i = 0; i < D - 1; ++i) {
    const int nu = i + (i >= mu ? 1 : 0);
    int fnu, bnu;
    nbr_offsets(g, sc, nu, fnu, bnu);
    int fsign = 0;
    if (FIELD) fsign = (mu == a.f.mu && nu == a.f.nu) ? 1 : (mu == a.f.nu && nu == a.f.mu) ? -1 : 0;
    const Q4<R> F = q4<R>((R)a.f.c[0], R(0), R(0), (R)a.f.s[0]);
    {
      const Q4<R> U1 = su2_load<R, true>(ro, g, array_base<T::NP>(g, D, q, nu), h + fmu);
      const Q4<R> U2 = su2_load<R, true>(ro, g, array_base<T::NP>(g, D, q, mu), h + fnu);
      const Q4<R> U3 = su2_load<R, true>(ro, g, array_base<T::NP>(g, D, p, nu), h);
      Q4<R> S = q4_mul(q4_mul(U1, q4_conj(U2)), q4_conj(U3));
      if (FIELD && fsign != 0) S = q4_mul(S, fsign > 0 ? F : q4_conj(F));
      A = q4_add(A, S);
    }
    {
      const Q4<R> U1 = su2_load<R, true>(ro, g, array_base<T::NP>(g, D, p, nu), h + fmu + bnu);
      const Q4<R> U2 = su2_load<R, true>(ro, g, array_base<T::NP>(g, D, q, mu), h + bnu);
      Q4<R> U3 = su2_load<R, true>(ro, g, array_base<T::NP>(g, D, q, nu), h + bnu);
      if (FIELD && fsign != 0) U3 = q4_mul(fsign > 0 ? q4_conj(F) : F, U3);
      const Q4<R> S = q4_mul(q4_mul(q4_conj(U1), q4_conj(U2)), U3);
      A = q4_add(A, S);
    }
  }
  const size_t own = array_base<T::NP>(g, D, p, mu);
  Q4<R> U = su2_load<R, false>(links, g, own, h);
  const uint32_t lex = 2u * h + (uint32_t)sc.s;
  const Q4<R> v = q4_mul(U, A);                       // proj(W) = W itself in the quaternion algebra
  const R k2 = v.a0 * v.a0 + v.a1 * v.a1 + v.a2 * v.a2 + v.a3 * v.a3;
  int code = 0;
  if (!(k2 < Tiny<R>::k2())) {
    Q4<R> qa;
    if (subgroup_quaternion<R, KIND, 2>(v, k2, lex, a, 0, qa, code)) U = q4_mul(qa, U);
  }
  const R n = q_rsqrt(U.a0 * U.a0 + U.a1 * U.a1 + U.a2 * U.a2 + U.a3 * U.a3);
  R r[4] = {U.a0 * n, U.a1 * n, U.a2 * n, U.a3 * n};
  store_reals<R, 4>(links, g, own, h, r);
  if (KIND == 0 && a.trials) {
    a.trials[(size_t)lex * 3 + 0] = (uint8_t)code; a.trials[(size_t)lex * 3 + 1] = 0; a.trials[(size_t)lex * 3 + 2] = 0;
  }
}

}  // namespace qcd
