// update.cuh -- the hot path: one (parity, mu) sub-step of the checkerboard sweep, one thread per link.
//   staple sum (2(D-1) staples, optional abelian field factor)  -> SURVEY 8(a)-3, 8(a)-4; PAPER.md:108 (checkerboard)
//   Cabibbo-Marinari over SU(2) subgroups: Kennedy-Pendleton heatbath ("(pseudo)heat-bath", NHIT trial cap,
//   PAPER.md:108, :134) or overrelaxation (BASELINE.json north_star)                       -> 8(a)-5, 8(a)-6
//   reunitarise + store ("reunitarization")                                   -> 8(a)-7
// A sub-step writes only U_mu on parity p and reads it only at the thread's own site, so it is race-free.
//
// Data movement: the 6(D-1) neighbour links and the own link of a thread are consumed in a
// fixed order; they are fetched by cp.async (LDGSTS, 16 B per plane) into a per-thread ring of K link slots in shared
// memory, K-1 links ahead of the arithmetic, so the loads of the next staples are in flight while the current 3x3 products
// run and no registers are held by data that is not being multiplied yet.  Every thread reads back only the slots it
// filled itself, so the ring needs no block barrier.  mu is a template parameter: every array base, neighbour direction
// and field role is resolved at compile time.
#pragma once
#include <type_traits>

#include "common.cuh"
#include "philox.cuh"
#include "sun_math.cuh"

namespace qcd {

struct FieldArgs {   // F = diag(exp(i theta_c)) on plane (mu,nu), mu<nu; cos/sin precomputed on the host in double
  int mu, nu;
  double c[3], s[3];
};

// Boundary layers of a part written straight into its neighbours' memory by the update kernel itself (the single-process
// driver of a divided lattice, qcd_split_*: "exchanging values of boundary sites", here without a separate
// exchange step).  A thread whose site lies in the part's first (last) own layer stores its new link a second time, into
// the previous (next) part's copy of that layer -- local memory or a peer GPU's over NVLink.  The destination part may
// have another extent, so its half-index is rebuilt from the coordinates with the destination's extents.
struct HaloPush {
  int on;            // 0: no neighbours to serve
  int last;          // the part's last own layer (first = 0)
  int layer[2];      // destination layer in the previous / next part
  int L1[2], L2[2];  // extents 1 and 2 of the previous / next part's local lattice (only the split extent differs)
  void* base[2];     // start of the (parity, mu) array being written in the previous / next part
};

struct UpdateArgs {
  double beta;
  double inv_c;      // N / (2 beta): delta = E / alpha = E * inv_c / k   (host-computed; inf when beta = 0 -> every trial fails)
  int parity, mu, hit, max_trials;
  int prev_parity, prev_mu;   // the kernel launched just before this one on the stream: an update kernel (its output array
                              // (prev_parity, prev_mu) is the only one that may not be read before griddepcontrol.wait),
                              // -1: a kernel that writes no links, -2: a kernel that writes all of them (init, set_links)
  uint32_t sweep, key0, key1;
  PhiloxKeys rk;     // the round keys of (key0, key1), host-computed (philox.cuh)
  uint8_t* trials;   // NULL or [lex][3] debug trial codes
  // fused plaquette measurement (MEAS kernels, see meas_store below): per-warp partial sums of Re Tr[U' A_nu] for the
  // staple directions nu < mu go to meas[meas_plane[nu] * meas_stride + global warp index]
  double* meas;
  uint32_t meas_stride;
  int meas_plane[3];
  TileMap tm;        // thread -> site mapping of the SU(3) kernels (set by the launcher)
  // start of every (parity, direction) array, computed by the launcher: pbase[nu] = U_nu on the parity being updated,
  // qbase[nu] = U_nu on the other parity.  In the kernels they are constant-bank loads; computed there, (p D + nu) * arr is
  // a 64-bit multiply-add per array on the FMA pipe.
  const void* pbase[4];
  const void* qbase[4];
  HaloPush hp;
  int rev;           // 1: the CTAs visit their boxes in descending order.  Consecutive launches of a sweep alternate, so that a
                     // launch starts on the part of the lattice the previous one touched last and finds it in the L2
                     // (the 32^4 lattices are 1.6 / 4.8 times the 126 MB L2: in the same order nothing survives a launch)
  int use_bulk;      // host side only: QCD_OPT_BULK_COPY (update_bulk.cuh instead of the tiled kernel where it applies)
  FieldArgs f;
};

// ------------------------------------------------------------------ fused plaquette measurement
// In the LAST pass of a sweep the sub-step (parity 1, mu) leaves every plaquette of the planes (nu, mu), nu < mu, in its
// final state: the links U_nu (nu < mu) and U_mu on parity 0 were updated earlier in the pass, U_mu on parity 1 is being
// written, and no later sub-step touches a link of these planes.  Each such plaquette contains exactly one U_mu link on an
// odd site (U_mu(x) and U_mu(x + nu) have opposite parities), so it is seen exactly once, by that link's thread, as a term
// of Re Tr[U'_mu(x) A_nu(x)], A_nu = the two staples of direction nu (with the field factor: the dressed plaquette of
// reading R10).  The kernels keep the cumulative staple sums after the first directions, take Re Tr with the NEW link,
// difference them per direction in double and reduce per warp (shuffles, fixed order: deterministic); a second kernel sums
// the per-warp partials.  The three launches (1, mu >= 1) of the last pass thus measure all D(D-1)/2 planes: the "working
// sweep" of PAPER.md:134 without a separate pass over the links.
// logical block index of a CTA: the launch order is reversed when a.rev is set; everything a CTA does (sites, measurement
// slots) follows the logical index, so results do not depend on the order
__device__ __forceinline__ uint32_t logical_block(const UpdateArgs& a) { return a.rev ? gridDim.x - 1u - blockIdx.x : blockIdx.x; }
// second store of a boundary link into the neighbouring part(s) (HaloPush); r = the reals just stored at the own site
template <typename R, int NREAL>
__device__ __forceinline__ void halo_push_store(const UpdateArgs& a, const Geom& g, const SiteCoord& sc, const R* r) {
  typedef typename PlaneTraits<R, NREAL>::Vec Vec;
  if (!a.hp.on) return;
  const int xs = g.sd == 1 ? sc.x1 : g.sd == 2 ? sc.x2 : sc.x3;
#pragma unroll
  for (int t = 0; t < 2; ++t) {
    if (xs != (t == 0 ? 0 : a.hp.last)) continue;
    int y1 = sc.x1, y2 = sc.x2, y3 = sc.x3;
    if (g.sd == 1) y1 = a.hp.layer[t]; else if (g.sd == 2) y2 = a.hp.layer[t]; else y3 = a.hp.layer[t];
    const uint32_t hh = (uint32_t)(((y3 * a.hp.L2[t] + y2) * a.hp.L1[t] + y1) * g.Lh0 + sc.j);
    store_reals<R, NREAL>((Vec*)a.hp.base[t], g, 0, hh, r);
  }
}
template <int NREC> __device__ __forceinline__ void meas_store(const UpdateArgs& a, const double (&t)[NREC]) {
  const uint32_t w = (logical_block(a) * blockDim.x + threadIdx.x) >> 5;
#pragma unroll
  for (int j = 0; j < NREC; ++j) {
    double x = t[j];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) x += __shfl_down_sync(0xffffffffu, x, o);
    if ((threadIdx.x & 31) == 0) a.meas[(size_t)a.meas_plane[j] * a.meas_stride + w] = x;
  }
}
// Re Tr[U S]
template <typename R> __device__ __forceinline__ R m3_retr(const M3<R>& U, const M3<R>& S) {
  R t = R(0);
#pragma unroll
  for (int i = 0; i < 3; ++i)
#pragma unroll
    for (int j = 0; j < 3; ++j) t += U.e[i][j].re * S.e[j][i].re - U.e[i][j].im * S.e[j][i].im;
  return t;
}

// ------------------------------------------------------------------ compile-time loops and cp.async
template <int I, int N, typename F> __device__ __forceinline__ void static_for(F&& f) {
  if constexpr (I < N) {
    f(std::integral_constant<int, I>{});
    static_for<I + 1, N>(f);
  }
}

// .cg: the copy bypasses L1 (measured: with .ca the L1, shrunk by the ring's shared memory, thrashes and costs an extra
// pass through the L1 data path -- 202 us instead of 133 us for the fp64 overrelaxation kernel at 32^4)
template <int BYTES> __device__ __forceinline__ void cp_async_vec(void* smem_dst, const void* gmem_src) {
  static_assert(BYTES == 8 || BYTES == 16, "plane vectors are 8 or 16 bytes");
  const unsigned s = (unsigned)__cvta_generic_to_shared(smem_dst);
  if constexpr (BYTES == 16) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(s), "l"(gmem_src) : "memory");
  } else {                                                          // 8-byte vectors (fp32 x18): .cg needs 16 bytes
    asm volatile("cp.async.ca.shared.global [%0], [%1], %2;\n" ::"r"(s), "l"(gmem_src), "n"(BYTES) : "memory");
  }
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::: "memory"); }
template <int N> __device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;\n" ::"n"(N) : "memory"); }

// ------------------------------------------------------------------ Kennedy-Pendleton heatbath (reading R5)
// One trial:  delta = -(ln r1 + cos^2(2 pi r2) ln r3) / alpha,  accept iff r4^2 <= 1 - delta/2,  g0 = 1 - delta.
// Everything but the division by alpha depends on the random numbers only, so it is split off:
//   E = -(ln r1 + cos^2(2 pi r2) ln r3),  w = r4^2            (KpRand, from Philox draw 1+t)
//   n = unit vector (st cos phi, st sin phi, ct)              (hb_direction, from Philox draw 0)
// and evaluated for trial 0 of all subgroups at the start of the kernel, while the first links are in flight.
// The accept decision is the fp64 one in both precisions, so that it agrees with the fp64 oracle whenever alpha agrees;
// the uniforms are exactly representable in the storage precision (R8).
template <typename R> struct HbDraw { R E, w, n1, n2, n3; };

template <typename R> struct KpRand;
template <> struct KpRand<double> {
  // branch-free forms on the Philox words themselves (hb_math.cuh): ln r1, cos^2(2 pi r2), ln r3 to ~5e-16 absolute
  static __device__ __forceinline__ void run(const Philox4& x, double& E, double& w) {
    const double r4 = uniform64(x.w);
    E = -(hbm::log_uniform32(x.x) + hbm::cos2_2pi_uniform32(x.y) * hbm::log_uniform32(x.z));
    w = r4 * r4;
  }
};
// fp32: __logf is 3 ulp (2^-21.4 absolute near 1) and cos(2 pi r2) comes from the SFU (__cosf on (-pi, pi): absolute error
// 2^-21.4, so c^2 ln r3 is off by at most 7.2e-7 |c| |ln r3| <= max(4e-6 E, 2.2e-6)).  The accept test of the fp32
// kernels is taken in float and re-evaluated in double inside a guard band (kp_accept below).
template <> struct KpRand<float> {
  static __device__ __forceinline__ void run(const Philox4& x, float& E, float& w) {
    const float r1 = uniform23f(x.x), r2 = uniform23f(x.y), r3 = uniform23f(x.z), r4 = uniform23f(x.w);
    const float c = __cosf(6.283185307f * (r2 - 0.5f));          // = -cos(2 pi r2); only c^2 is used
    E = -(__logf(r1) + c * c * __logf(r3));
    w = r4 * r4;
  }
};
template <typename R> __device__ __forceinline__ void hb_direction(const Philox4& x, R& n1, R& n2, R& n3) {
  const R u1 = uniform_real<R>(x.x), u2 = uniform_real<R>(x.y);
  const R ct = R(1) - R(2) * u1;
  const R st = q_sqrt(R(1) - ct * ct);
  R sphi, cphi;
  q_sincospi(R(2) * u2, &sphi, &cphi);
  n1 = st * cphi; n2 = st * sphi; n3 = ct;
}
// fp64: sin, cos(2 pi u2) with the octant reduction done on the Philox word (hb_math.cuh)
template <> __device__ __forceinline__ void hb_direction<double>(const Philox4& x, double& n1, double& n2, double& n3) {
  const double ct = 1.0 - 2.0 * uniform64(x.x);
  const double st = hbm::sqrt_pos(1.0 - ct * ct);
  double sphi, cphi;
  hbm::sincos_2pi_uniform32(x.y, &sphi, &cphi);
  n1 = st * cphi; n2 = st * sphi; n3 = ct;
}
// fp32: the azimuth from the SFU, argument folded into (-pi, pi) where __sinf / __cosf are good to 2^-21.4 absolute
// (the link tolerance is 2e-5): sin(2 pi u) = -sin(2 pi (u - 1/2)), cos likewise
template <> __device__ __forceinline__ void hb_direction<float>(const Philox4& x, float& n1, float& n2, float& n3) {
  const float u1 = uniform23f(x.x), u2 = uniform23f(x.y);
  const float ct = 1.0f - 2.0f * u1;
  const float st = sqrtf(1.0f - ct * ct);
  const float ang = 6.283185307f * (u2 - 0.5f);
  n1 = -st * __cosf(ang); n2 = -st * __sinf(ang); n3 = ct;
}
// trial 0 and direction of subgroup sg of this link
template <typename R>
__device__ __forceinline__ HbDraw<R> hb_first_draw(uint32_t lex, const UpdateArgs& a, int mu, int sg) {
  const uint32_t c2 = philox_c2(mu, a.parity, sg, a.hit, 0);
  HbDraw<R> d;
  KpRand<R>::run(philox4x32_10(lex, a.sweep, c2, 1u, a.rk), d.E, d.w);
  hb_direction<R>(philox4x32_10(lex, a.sweep, c2, 0u, a.rk), d.n1, d.n2, d.n3);
  return d;
}

// Which Philox block a trial comes from: (lex, sweep, c2, draw = 1 + t) under the launch's key
struct KpKey { uint32_t lex, sweep, c2, key0, key1; };
// the whole trial in double from its regenerated Philox block (guard-band path of the fp32 kernels; out of line, rarely taken)
static __device__ __noinline__ bool kp_trial_f64_cold(double alpha, uint32_t lex, uint32_t sweep, uint32_t c2, uint32_t draw, uint32_t key0,
                                                      uint32_t key1, double* g0) {
  const Philox4 b = philox4x32_10(lex, sweep, c2, draw, key0, key1);
  const double r1 = uniform23(b.x), r2 = uniform23(b.y), r3 = uniform23(b.z), r4 = uniform23(b.w);
  const double c = cospi(2.0 * r2);
  const double delta = -(log(r1) + c * c * log(r3)) / alpha;
  *g0 = 1.0 - delta;
  return r4 * r4 <= 1.0 - 0.5 * delta;
}
// accept test of trial `draw` given its random part (E, w)
__device__ __forceinline__ bool kp_accept(double inv_alpha, double E, double w, const KpKey&, uint32_t, double& g0) {
  const double delta = E * inv_alpha;
  g0 = 1.0 - delta;
  return w <= 1.0 - 0.5 * delta;
}
// fp32: |error of delta| < (4e-6 E + 2.5e-6) / alpha, so outside the guard band below the float decision is the fp64 one;
// inside it (probability ~1e-5 per trial) the trial is recomputed in double from its own Philox block.  The band is decided
// here, once, from one rounding of the margin.
__device__ __forceinline__ bool kp_accept(float inv, float E, float w, const KpKey& k, uint32_t draw, float& g0) {
  const float delta = E * inv;
  const float margin = (1.0f - 0.5f * delta) - w;
  g0 = 1.0f - delta;
  if (fabsf(margin) < (6e-6f * E + 4e-6f) * inv + 5e-7f) {
    double g0d;
    const bool acc = kp_trial_f64_cold(1.0 / (double)inv, k.lex, k.sweep, k.c2, draw, k.key0, k.key1, &g0d);
    g0 = (float)g0d;
    return acc;
  }
  return margin >= 0.0f;
}

// Trials 1 .. max_trials-1 of a subgroup whose trial 0 was rejected (3 % of the lanes at beta = 6, but 60 % of the warps
// have such a lane).  Inlined into each of the three subgroup hits: one shared out-of-line copy was measured and lost
// (fp32 HB 79.5 -> 86.5 us, fp64 190 -> 204 us: the call spills the hit's live matrices around it).  Round keys from the
// launch arguments, like trial 0.
template <typename R>
static __device__ __forceinline__ bool kp_retry(R inv_alpha, const KpKey& key, const PhiloxKeys& rk, int max_trials, R& g0, int& code) {
  code = 0x80 | max_trials;
  for (int t = 1; t < max_trials; ++t) {
    R E, w;
    KpRand<R>::run(philox4x32_10(key.lex, key.sweep, key.c2, 1u + (uint32_t)t, rk), E, w);
    if (kp_accept(inv_alpha, E, w, key, 1u + (uint32_t)t, g0)) { code = t + 1; return true; }
  }
  return false;
}

// quaternion a of the subgroup update from the projected v = proj(W) (not normalised), k2 = |v|^2;
// d0 = trial 0 and direction (heatbath only)
template <typename R, int KIND, int NC>
__device__ __forceinline__ bool subgroup_quaternion(const Q4<R>& v, R k2, uint32_t lex, const UpdateArgs& a, int mu, int sg,
                                                    const HbDraw<R>& d0, Q4<R>& out, int& code) {
  if (KIND == 1) {
    // overrelaxation: a = (vt^dagger)^2 = (v0^2 - |vec v|^2, -2 v0 vec v) / k^2
    const R inv = q_rcp(k2);
    const R vv = v.a1 * v.a1 + v.a2 * v.a2 + v.a3 * v.a3;
    const R m2 = R(-2) * v.a0 * inv;
    out = q4<R>((v.a0 * v.a0 - vv) * inv, m2 * v.a1, m2 * v.a2, m2 * v.a3);
    return true;
  } else {
    const R rk = q_rsqrt(k2);
    // 1 / alpha, alpha = 2 beta k / N.  The SU(3) hit hands in v = 2 proj(W) (it leaves out the factor 1/2 of the
    // projection: everything else here is homogeneous of degree 0 in v), so k = |v| / 2 there.
    const R inv_alpha = (R)a.inv_c * rk * (NC == 3 ? R(2) : R(1));
    KpKey key;
    key.lex = lex; key.sweep = a.sweep; key.c2 = philox_c2(mu, a.parity, sg, a.hit, 0); key.key0 = a.key0; key.key1 = a.key1;
    R g0;
    bool acc = kp_accept(inv_alpha, d0.E, d0.w, key, 1u, g0);     // trial 0 from the precomputed random part
    code = 1;
    if (!acc) acc = kp_retry<R>(inv_alpha, key, a.rk, a.max_trials, g0, code);
    // fp32: no early return: the lanes that needed further trials re-join the warp here, so what follows is executed
    // once per warp and not once per divergent path (it was 1.57 times per subgroup at 3 % rejection).  fp64 keeps the
    // early exit (the straight-line form costs it two spilled registers at its 168-register cap).
    if constexpr (sizeof(R) == 8) { if (!acc) return false; }
    const R rr = q_sqrt(fmax(R(0), R(1) - g0 * g0));
    const Q4<R> g = q4<R>(g0, rr * d0.n1, rr * d0.n2, rr * d0.n3);
    const Q4<R> vtc = q4<R>(v.a0 * rk, -v.a1 * rk, -v.a2 * rk, -v.a3 * rk);   // vt^dagger
    out = q4_mul(g, vtc);
    return acc;
  }
}

template <typename R> struct Tiny;
template <> struct Tiny<float> { static __device__ __forceinline__ float k2() { return 1e-20f; } };
template <> struct Tiny<double> { static __device__ __forceinline__ double k2() { return 1e-30; } };

// =====================================================================================
// SU(3)
// =====================================================================================
// twice the SU(2) projection of the 2x2 block (wii wij; wji wjj), and its squared norm
template <typename R>
__device__ __forceinline__ void su3_project2(const Cx<R>& wii, const Cx<R>& wij, const Cx<R>& wji, const Cx<R>& wjj, Q4<R>& v, R& k2) {
  v.a0 = wii.re + wjj.re;
  v.a1 = wij.im + wji.im;
  v.a2 = wij.re - wji.re;
  v.a3 = wii.im - wjj.im;
  k2 = v.a0 * v.a0 + v.a1 * v.a1 + v.a2 * v.a2 + v.a3 * v.a3;
}
__device__ __forceinline__ void su3_project2(const Cx<float>& wii, const Cx<float>& wij, const Cx<float>& wji, const Cx<float>& wjj,
                                             Q4<float>& v, float& k2) {
  const float2 p = __ffma2_rn(f2_of(wjj), make_float2(1.0f, -1.0f), f2_of(wii));     // (a0, a3)
  const float2 q = __ffma2_rn(f2_of(wji), make_float2(-1.0f, 1.0f), f2_of(wij));     // (a2, a1)
  float2 t = __fmul2_rn(p, p);
  t = __ffma2_rn(q, q, t);
  v.a0 = p.x; v.a3 = p.y; v.a2 = q.x; v.a1 = q.y;
  k2 = t.x + t.y;
}

// one Cabibbo-Marinari subgroup hit on rows (I,J) of U given the staple sum A
template <typename R, int KIND, int I, int J>
__device__ __forceinline__ void su3_subgroup_hit(M3<R>& U, const M3<R>& A, uint32_t lex, const UpdateArgs& a, int mu, int sg,
                                                 const HbDraw<R>& d0, int& code) {
  Cx<R> wii = cx<R>(0, 0), wij = cx<R>(0, 0), wji = cx<R>(0, 0), wjj = cx<R>(0, 0);
  cdot3<CD_NN>(wii, U.e[I][0], U.e[I][1], U.e[I][2], A.e[0][I], A.e[1][I], A.e[2][I]);
  cdot3<CD_NN>(wij, U.e[I][0], U.e[I][1], U.e[I][2], A.e[0][J], A.e[1][J], A.e[2][J]);
  cdot3<CD_NN>(wji, U.e[J][0], U.e[J][1], U.e[J][2], A.e[0][I], A.e[1][I], A.e[2][I]);
  cdot3<CD_NN>(wjj, U.e[J][0], U.e[J][1], U.e[J][2], A.e[0][J], A.e[1][J], A.e[2][J]);
  // v = 2 proj(W): the factor 1/2 of the projection is left out (four multiplies); k2 = 4 k^2
  Q4<R> v;
  R k2;
  su3_project2(wii, wij, wji, wjj, v, k2);
  // reading R4 (k -> 0) and R5 (all trials rejected): the subgroup factor is the identity.  Applied as a = 1 rather than
  // by skipping the row update (1 * u + 0 * u' = u exactly), so that the warp does not diverge around it.
  const bool tiny = k2 < R(4) * Tiny<R>::k2();
  if constexpr (sizeof(R) == 8) { if (tiny) { code = 0; return; } }
  Q4<R> q;
  int cd = 0;
  const bool ok = subgroup_quaternion<R, KIND, 3>(v, tiny ? R(1) : k2, lex, a, mu, sg, d0, q, cd) && !tiny;
  code = tiny ? 0 : cd;
  if constexpr (sizeof(R) == 8) { if (!ok) return; }
  if (!ok) q = q4<R>(R(1), R(0), R(0), R(0));
  const Cx<R> aii = cx<R>(q.a0, q.a3), aij = cx<R>(q.a2, q.a1), aji = cx<R>(-q.a2, q.a1), ajj = cx<R>(q.a0, -q.a3);
#pragma unroll
  for (int c = 0; c < 3; ++c) {
    const Cx<R> ui = U.e[I][c], uj = U.e[J][c];
    U.e[I][c] = cdot2_nn(aii, aij, ui, uj);
    U.e[J][c] = cdot2_nn(aji, ajj, ui, uj);
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
__device__ __forceinline__ void m3_add(M3<float>& a, const M3<float>& s) {
#pragma unroll
  for (int r = 0; r < 3; ++r)
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      const float2 v = __fadd2_rn(f2_of(a.e[r][c]), f2_of(s.e[r][c]));
      a.e[r][c].re = v.x; a.e[r][c].im = v.y;
    }
}
template <typename R> __device__ __forceinline__ void m3_add(M3<R>& a, const M3<R>& s) {
#pragma unroll
  for (int r = 0; r < 3; ++r)
#pragma unroll
    for (int c = 0; c < 3; ++c) { a.e[r][c].re += s.e[r][c].re; a.e[r][c].im += s.e[r][c].im; }
}

// The links a thread consumes, in order.  For the i-th direction nu != MU, slot j = 0..5:
//   j=0  U2  = U_mu(x+nu)        j=1  U3  = U_nu(x)        j=2  U1  = U_nu(x+mu)          upper staple U1 (U3 U2)^+
//   j=3  U1' = U_nu(x+mu-nu)     j=4  U2' = U_mu(x-nu)     j=5  U3' = U_nu(x-nu)          lower staple (U2' U1')^+ U3'
// and last the thread's own link U_mu(x).
//
// Template parameters: K = ring slots per thread (3 or 6, so that the slot of link (i, j) is j % K whatever i is; K = 0:
// no ring, every link is loaded from global memory when it is consumed); B threads per CTA; MINB = CTAs per SM the
// register allocation must allow.  ROLL: the loop over nu is not unrolled (heatbath kernels: their straight-line code
// would be 60+ KB against a 32 KB instruction cache level; the three subgroup hits ARE unrolled, see su3_launch.cuh).
// Heatbath: the random-number-only part of trial 0 of every subgroup is computed at the start of the kernel, before
// griddepcontrol.wait, and parked in shared memory.
// 18-real storage only: the links of which a thread uses rows 0,1 alone (J as in the table above; 6 = the own link, whose
// third row is rebuilt).  Every product of SU(3) matrices is in SU(3), so the third rows of X = U3 U2, Y = U2' U1' and of
// the staples are rebuilt as conj(row0 x row1) whatever the storage; what 18-real storage saves is the rebuilding of
// the third rows of the RIGHT factors U2, U1', U3' (J = 0, 3, 5), which are read in full.
template <bool COMP> __host__ __device__ constexpr bool rows01_only_t(int J) { return !COMP && (J == 1 || J == 2 || J == 4 || J == 6); }

// MEAS: fused plaquette measurement (see meas_store above); whole warps stay alive for the warp reduction.
template <typename R, int D, int MU, bool COMP, int KIND, bool FIELD, int B, int K, int MINB, bool ROLL, bool MEAS>
__global__ void __launch_bounds__(B, MINB)
su3_update_kernel(Geom g, typename PlaneTraits<R, (COMP ? 12 : 18)>::Vec* links, UpdateArgs a) {
  typedef PlaneTraits<R, (COMP ? 12 : 18)> T;
  typedef typename T::Vec Vec;
  constexpr int NREAL = COMP ? 12 : 18, NP = T::NP;
  static_assert(!MEAS || MU >= 1, "planes (nu, mu), nu < mu");
  // cumulative staple sums kept for the measurement: after directions nu = 0 .. NSNAP-1 (the last cumulative sum of
  // mu = D-1 is A itself)
  constexpr int NSNAP = !MEAS ? 0 : (MU == D - 1 ? MU - 1 : MU);
  // link n = 6 i + J of the sequence goes to slot n % K; with the rolled direction loop the slot must not depend on i
  static_assert(K == 0 || (K >= 2 && K <= 7 && (!ROLL || 6 % K == 0)), "ring slots: K | 6 when the direction loop is rolled");
  constexpr int KR = K > 0 ? K : 1;
  extern __shared__ __align__(16) unsigned char ring_raw[];
  Vec* ring = reinterpret_cast<Vec*>(ring_raw) + threadIdx.x;      // [slot][plane][B], this thread's column

  const int p = a.parity;
  uint32_t h;
  SiteCoord sc;
  bool active = true;
  if (a.tm.on) {
    sc = decode_site_tiled(g, a.tm, p, logical_block(a), h);       // the tiles cover the lattice exactly
  } else {
    uint32_t hl = logical_block(a) * B + threadIdx.x;              // launch index over the interior (= h unless a slab)
    if constexpr (MEAS) {
      active = hl < g.Vh_int;                                      // a surplus thread shadows the last site: it neither
      if (!active) hl = g.Vh_int - 1;                              // stores nor contributes, but stays for the shuffles
    } else {
      if (hl >= g.Vh_int) return;                                  // no block barrier anywhere below
    }
    sc = decode_launch(g, hl, p, h);
  }
  int fo[D], bo[D];
#pragma unroll
  for (int d = 0; d < D; ++d) nbr_offsets(g, sc, d, fo[d], bo[d]);
  // A (parity, direction) array holds arr = NP * Vh_pad vectors (< 2^32, checked at creation); its base is a 64-bit,
  // warp-uniform pointer and elements are addressed by the 32-bit in-array offset blk_off(h').

  Vec* const own_ptr = (Vec*)a.pbase[MU];
  const Vec* const qmu_ptr = (const Vec*)a.qbase[MU];
  auto at = [&](const Vec* base, int off) -> const Vec* { return base + blk_off<NP>(h + (uint32_t)off); };

  struct Dir { const Vec *pp, *qp; int f, b, nu; };                // per-direction addressing (array bases), run-time nu
  auto make_dir = [&](int i) {
    Dir d;
    d.nu = i + (i >= MU ? 1 : 0);
    d.f = fo[0]; d.b = bo[0];
#pragma unroll
    for (int k = 1; k < D; ++k) if (d.nu == k) { d.f = fo[k]; d.b = bo[k]; }
    d.pp = (const Vec*)a.pbase[d.nu];
    d.qp = (const Vec*)a.qbase[d.nu];
    return d;
  };
  // plane 0 of link j of direction d (j = 6: the own link)
  auto link_ptr = [&](auto jc, const Dir& d) -> const Vec* {
    constexpr int J = decltype(jc)::value;
    if constexpr (J == 0) return at(qmu_ptr, d.f);
    else if constexpr (J == 1) return at(d.pp, 0);
    else if constexpr (J == 2) return at(d.qp, fo[MU]);
    else if constexpr (J == 3) return at(d.pp, fo[MU] + d.b);
    else if constexpr (J == 4) return at(qmu_ptr, d.b);
    else if constexpr (J == 5) return at(d.qp, d.b);
    else return at(own_ptr, 0);
  };
  auto issue = [&](auto jc, const Dir& d, int n) {                  // cp.async link J (n-th of the sequence) into ring slot n % K
    constexpr int J = decltype(jc)::value;
    const Vec* src = link_ptr(jc, d);
    Vec* dst = ring + (n % KR) * NP * B;
    // Links that enter only as the LEFT factor of a product whose third row is rebuilt anyway (U3, U1, U2': J = 1, 2, 4)
    // and the own link (J = 6) contribute rows 0,1 only: with 18-real storage the planes of their third row are not
    // fetched (L2 -> SM traffic 19 -> 15.7 link-sizes per link-hit; every neighbour array is still read in full from
    // DRAM once, by the thread that needs all rows of that link as a right factor).
    constexpr int NPJ = rows01_only_t<COMP>(J) ? (NP * 2) / 3 : NP;
#pragma unroll
    for (int k = 0; k < NPJ; ++k) cp_async_vec<(int)sizeof(Vec)>(dst + k * B, src + k * PLANE_STRIDE);
  };
  auto fetch = [&](auto jc, const Dir& d, M3<R>& u, bool row2, int n) {
    constexpr int J = decltype(jc)::value;
    R r[NREAL];
    if constexpr (K > 0) {
      const Vec* src = ring + (n % KR) * NP * B;
#pragma unroll
      for (int k = 0; k < NP; ++k) vec_unpack(src[k * B], r + k * T::VW);
    } else {
      const Vec* src = link_ptr(jc, d);
      // the own-link array is written by this kernel (each thread its own element): plain load; the rest is read-only
#pragma unroll
      for (int k = 0; k < NP; ++k) vec_unpack(J == 6 ? src[k * PLANE_STRIDE] : __ldg(src + k * PLANE_STRIDE), r + k * T::VW);
    }
    if constexpr (rows01_only_t<COMP>(J)) {
      m3_from_reals<R, 12>(u, r);                                  // planes of rows 0,1 (the first 12 reals) only
      if (row2) m3_complete_row2(u);
    } else {
      m3_from_reals<R, NREAL>(u, r);
      if (COMP && row2) m3_complete_row2(u);
    }
  };

  const uint32_t lex = lex_global(g, sc);
  // Prologue: links 0 .. K-2 of the first direction nu0.  They come from the arrays (q, mu), (p, nu0), (q, nu0); unless the
  // update kernel running just before this one writes one of them, they are fetched before griddepcontrol.wait, i.e.
  // while that kernel drains (in sweep order the previous kernel writes (p, mu-1): only mu = 1 has to wait).  The trigger
  // for the next kernel comes after this kernel's own wait, so at most one earlier update kernel is ever in flight.
  Dir cur = make_dir(0);
  // prev_parity = -2: the kernel before this one wrote every array (init, set_links): nothing may be read early.
  const bool early = a.prev_parity != -2 &&
                     !((a.prev_parity == 1 - p && (a.prev_mu == MU || a.prev_mu == cur.nu)) || (a.prev_parity == p && a.prev_mu == cur.nu));
  auto prologue = [&]() {
    if constexpr (K > 0) static_for<0, KR - 1>([&](auto jc) { issue(jc, cur, decltype(jc)::value); cp_async_commit(); });
  };
  if (early) prologue();
  // heatbath: the random-number-only part of trial 0 and the direction of each subgroup, parked in shared memory behind
  // the ring ([subgroup][5][B] reals, this thread's column).  It does not touch the links, so it runs before pdl_wait()
  // -- in the tail of the previous sub-step's kernel when this CTA became resident early -- and after the early prologue,
  // whose loads are then in flight meanwhile.
  R* draws = reinterpret_cast<R*>(ring_raw + (size_t)K * NP * B * sizeof(Vec)) + threadIdx.x;
  if constexpr (KIND == 0) {
#pragma unroll 1
    for (int sg = 0; sg < 3; ++sg) {
      const HbDraw<R> d = hb_first_draw<R>(lex, a, MU, sg);
      R* o = draws + sg * 5 * B;
      o[0] = d.E; o[B] = d.w; o[2 * B] = d.n1; o[3 * B] = d.n2; o[4 * B] = d.n3;
    }
  }

  pdl_wait();                                                      // the previous sub-step's links are complete and visible
  pdl_trigger();
  if (!early) prologue();

  M3<R> A, P, Q;      // A: staple sum; P: the link kept for the next product (U2 / U1'); Q: X = U3 U2 or Y = U2' U1'
  m3_zero(A);
  Row2Sum<R> row2;    // third row of the staple sum, accumulated in its unreduced form (sun_math.cuh); without a field only
  row2.zero();
  M3<R> snap[NSNAP > 0 ? NSNAP : 1];
  auto direction_step = [&](int i) {
    const bool last = (i == D - 2);
    const int n0 = ROLL ? 0 : 6 * i;                               // sequence number of this direction's first link
    const Dir nxt = make_dir(last ? i : i + 1);
    const int fsign = !FIELD ? 0 : (MU == a.f.mu && cur.nu == a.f.nu) ? 1 : (MU == a.f.nu && cur.nu == a.f.mu) ? -1 : 0;
    static_for<0, 6>([&](auto jc) {
      constexpr int J = decltype(jc)::value;
      if constexpr (K > 0) {
        // keep K-1 links in flight: the link K-1 ahead goes to the slot whose previous content has been consumed
        constexpr int JA = J + KR - 1;
        if constexpr (JA < 6) {
          issue(std::integral_constant<int, JA>{}, cur, n0 + JA);
        } else {
          if (!last) issue(std::integral_constant<int, JA - 6>{}, nxt, n0 + JA);
          else if (JA == 6) issue(std::integral_constant<int, 6>{}, cur, n0 + 6);   // the own link, once, after the last direction
        }
        cp_async_commit();                                         // one group per step, possibly empty
        cp_async_wait<KR - 1>();                                   // link (i, J) has landed
      }
      if constexpr (J == 0) {
        fetch(jc, cur, P, true, n0 + decltype(jc)::value);                                   // U2, all rows
      } else if constexpr (J == 1) {
        M3<R> U3;
        fetch(jc, cur, U3, false, n0 + decltype(jc)::value);
        m3_zero(Q);
        m3_mad_nn<R, 2>(Q, U3, P);                                 // X = U3 U2, rows 0,1; row 2 rebuilt (XY_ROWS)
        m3_complete_row2(Q);
      } else if constexpr (J == 2) {
        M3<R> U1;
        fetch(jc, cur, U1, false, n0 + decltype(jc)::value);
        M3<R> Sm;
        m3_zero(Sm);
        m3_mad_nd<R, 2>(Sm, U1, Q);                                // U1 X^+, rows 0,1; the staple is in SU(3): row 2 rebuilt
        if constexpr (!FIELD) {
          m3_add_rows01(A, Sm);
          row2.add(A, Sm);
        } else {
          m3_complete_row2(Sm);
          if (fsign != 0) su3_scale_cols(Sm, a.f, fsign < 0);            // first direction: . F ; second: . F^+
          m3_add(A, Sm);
        }
      } else if constexpr (J == 3) {
        fetch(jc, cur, P, true, n0 + decltype(jc)::value);                                   // U1', all rows
      } else if constexpr (J == 4) {
        M3<R> U2;
        fetch(jc, cur, U2, false, n0 + decltype(jc)::value);
        m3_zero(Q);
        m3_mad_nn<R, 2>(Q, U2, P);                                 // Y = U2' U1', rows 0,1; row 2 rebuilt
        m3_complete_row2(Q);
      } else {
        M3<R> U3;
        fetch(jc, cur, U3, true, n0 + decltype(jc)::value);
        if (FIELD && fsign != 0) su3_scale_rows(U3, a.f, fsign > 0);   // first direction: F^+ U3' ; second: F U3'
        if (COMP) {
          M3<R> Sm;
          m3_zero(Sm);
          m3_mad_dn<R, 2>(Sm, Q, U3);                              // Y^+ U3'
          if constexpr (!FIELD) {
            m3_add_rows01(A, Sm);
            row2.add(A, Sm);
          } else {
            m3_complete_row2(Sm);
            m3_add(A, Sm);
          }
        } else {
          m3_mad_dn<R, 3>(A, Q, U3);
        }
      }
    });
    cur = nxt;
    if constexpr (NSNAP > 0) {
#pragma unroll
      for (int k = 0; k < NSNAP; ++k) if (i == k) { snap[k] = A; row2.finish(snap[k]); }   // directions come in the order nu = 0 .. mu-1, mu+1 ..
    }
  };
  if constexpr (ROLL) {
#pragma unroll 1
    for (int i = 0; i < D - 1; ++i) direction_step(i);
  } else {
#pragma unroll
    for (int i = 0; i < D - 1; ++i) direction_step(i);
  }

  row2.finish(A);
  // own link: the last one through the ring
  if constexpr (K > 0) cp_async_wait<0>();
  M3<R> U;
  fetch(std::integral_constant<int, 6>{}, cur, U, true, ROLL ? 6 : 6 * (D - 1));

  if constexpr (KIND == 1) {
    int c;
    HbDraw<R> none;
    none.E = none.w = none.n1 = none.n2 = none.n3 = R(0);
    su3_subgroup_hit<R, KIND, 0, 1>(U, A, lex, a, MU, 0, none, c);
    su3_subgroup_hit<R, KIND, 0, 2>(U, A, lex, a, MU, 1, none, c);
    su3_subgroup_hit<R, KIND, 1, 2>(U, A, lex, a, MU, 2, none, c);
  } else {
    // trial 0 and the direction of each subgroup were parked in shared memory at kernel start; the three hits are
    // unrolled (compile-time rows: no frame permutation)
    auto first_draw = [&](int sg) {
      HbDraw<R> d;
      const R* o = draws + sg * 5 * B;
      d.E = o[0]; d.w = o[B]; d.n1 = o[2 * B]; d.n2 = o[3 * B]; d.n3 = o[4 * B];
      return d;
    };
    int c0, c1, c2;
    su3_subgroup_hit<R, KIND, 0, 1>(U, A, lex, a, MU, 0, first_draw(0), c0);
    su3_subgroup_hit<R, KIND, 0, 2>(U, A, lex, a, MU, 1, first_draw(1), c1);
    su3_subgroup_hit<R, KIND, 1, 2>(U, A, lex, a, MU, 2, first_draw(2), c2);
    if (a.trials) {
      a.trials[(size_t)lex * 3 + 0] = (uint8_t)c0; a.trials[(size_t)lex * 3 + 1] = (uint8_t)c1; a.trials[(size_t)lex * 3 + 2] = (uint8_t)c2;
    }
  }
  m3_reunitarise(U);

  if constexpr (MEAS) {
    double t[MU];
    R prev = R(0);
#pragma unroll
    for (int j = 0; j < MU; ++j) {
      const R c = m3_retr(U, j < NSNAP ? snap[j < NSNAP ? j : 0] : A);
      t[j] = active ? (double)c - (double)prev : 0.0;
      prev = c;
    }
    meas_store<MU>(a, t);
    if (!active) return;
  }
  R r[NREAL];
  m3_to_reals<R, NREAL>(U, r);
  store_reals<R, NREAL>(own_ptr, g, 0, h, r);
  halo_push_store<R, NREAL>(a, g, sc, r);
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

template <typename R, int D, int KIND, bool FIELD, bool MEAS>
__global__ void __launch_bounds__(256)
su2_update_kernel(Geom g, typename PlaneTraits<R, 4>::Vec* links, UpdateArgs a) {
  typedef PlaneTraits<R, 4> T;
  uint32_t hl = logical_block(a) * blockDim.x + threadIdx.x, h;  // launch index over the interior (= h unless a slab)
  bool active = true;
  if constexpr (MEAS) {
    active = hl < g.Vh_int;
    if (!active) hl = g.Vh_int - 1;                        // surplus threads stay for the warp reduction (see su3_update_kernel)
  } else {
    if (hl >= g.Vh_int) { pdl_wait(); pdl_trigger(); return; }
  }
  const int p = a.parity, mu = a.mu, q = 1 - p;
  const SiteCoord sc = decode_launch(g, hl, p, h);
  int fmu, bmu;
  nbr_offsets(g, sc, mu, fmu, bmu);
  pdl_wait();
  pdl_trigger();
  const typename T::Vec* __restrict__ ro = links;
  Q4<R> A = q4<R>(0, 0, 0, 0);
  Q4<R> cum[D - 1];                                        // MEAS: cumulative staple sums after each direction
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
    if constexpr (MEAS) cum[i] = A;
  }
  const size_t own = array_base<T::NP>(g, D, p, mu);
  Q4<R> U = su2_load<R, false>(links, g, own, h);
  const uint32_t lex = lex_global(g, sc);
  const Q4<R> v = q4_mul(U, A);                       // proj(W) = W itself in the quaternion algebra
  const R k2 = v.a0 * v.a0 + v.a1 * v.a1 + v.a2 * v.a2 + v.a3 * v.a3;
  int code = 0;
  if (!(k2 < Tiny<R>::k2())) {
    Q4<R> qa;
    HbDraw<R> d0;
    if (KIND == 0) d0 = hb_first_draw<R>(lex, a, mu, 0);
    else d0.E = d0.w = d0.n1 = d0.n2 = d0.n3 = R(0);
    if (subgroup_quaternion<R, KIND, 2>(v, k2, lex, a, mu, 0, d0, qa, code)) U = q4_mul(qa, U);
  }
  const R n = q_rsqrt(U.a0 * U.a0 + U.a1 * U.a1 + U.a2 * U.a2 + U.a3 * U.a3);
  R r[4] = {U.a0 * n, U.a1 * n, U.a2 * n, U.a3 * n};
  if constexpr (MEAS) {
    // Re Tr[U' A_nu] = 2 (U' . A_nu)_0 in the quaternion algebra; directions nu = 0 .. mu-1 come first
    double t[D - 1];
    R prev = R(0);
#pragma unroll
    for (int j = 0; j < D - 1; ++j) {
      const R c = R(2) * (r[0] * cum[j].a0 - r[1] * cum[j].a1 - r[2] * cum[j].a2 - r[3] * cum[j].a3);
      t[j] = (active && j < mu) ? (double)c - (double)prev : 0.0;
      prev = c;
    }
    const uint32_t w = (logical_block(a) * blockDim.x + threadIdx.x) >> 5;
#pragma unroll
    for (int j = 0; j < D - 1; ++j) {
      double x = t[j];
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) x += __shfl_down_sync(0xffffffffu, x, o);
      if ((threadIdx.x & 31) == 0 && j < mu) a.meas[(size_t)a.meas_plane[j] * a.meas_stride + w] = x;
    }
    if (!active) return;
  }
  store_reals<R, 4>(links, g, own, h, r);
  halo_push_store<R, 4>(a, g, sc, r);
  if (KIND == 0 && a.trials) {
    a.trials[(size_t)lex * 3 + 0] = (uint8_t)code; a.trials[(size_t)lex * 3 + 1] = 0; a.trials[(size_t)lex * 3 + 2] = 0;
  }
}

}  // namespace qcd
