// update_tiled.cuh -- the D = 4 SU(3) sub-step with the U_mu neighbourhood of a CTA resident in shared memory.
//
// Why (profiles/r1_c_*): with a private copy of its 19 links per thread (the cp.async ring of update.cuh) a launch pulls
// 19 link-sizes per link-hit through the L2 -> SM crossbar although only 9 are compulsory from DRAM; at 32^4 that is
// 478 MB (fp32 x12) / 1434 MB (fp64 x18) per launch, and the L2 slices deliver ~11-12 TB/s: the fp64 kernel sits on that
// limit (load path alone 116 us) and the fp32 kernel's load path (44-51 us alone) is as long as its arithmetic.
// The most re-used operand is U_mu on the other parity q = 1-p:  U_mu(y) is read by the six threads y -+ nu (nu != mu).
// A CTA covers a box of T0 x T1 x T2 x T3 sites of parity p in (half-index j, x1, x2, x3) coordinates and stages the
// box of U_mu^q plus its one-deep faces in the directions nu != mu ONCE (one __syncthreads per kernel); the staple
// operands U_mu(x+nu), U_mu(x-nu) of all three directions are then read from there.  The other 12 neighbour links and
// the own link keep going through the per-thread cp.async ring (latency-tolerant, no further barrier).
// L2 -> SM traffic per link-hit: 13 + (1 + sum_{nu>=1} 2/T_nu + [mu != 0]/T0)  ~ 15.3 link-sizes instead of 19.
// A step of +-1 in direction 0 moves the half-index j by s or s-1 (s = x0 & 1 of the site), so a row of the box needs
// only ONE of its two j-faces; periodic wrap enters only the global address, slots are addressed box-relative.
//
// The arithmetic (products, Cabibbo-Marinari hits, reunitarisation) is the one of update.cuh and the links are consumed
// in the same order; the two kernels agree to rounding (the compiler's FMA contraction may differ between them).
#pragma once
#include "update.cuh"

namespace qcd {

// Slots of the resident region (one plane): the box itself, then per direction d != mu the faces:
//   d >= 1: low face (box coordinate -1) and high face (T_d), B / T_d slots each;  d = 0: one face, B / T0 slots.
template <int T0_, int T1_, int T2_, int T3_> struct TileDims {
  static constexpr int T0 = T0_, T1 = T1_, T2 = T2_, T3 = T3_, B = T0_ * T1_ * T2_ * T3_;
  __host__ __device__ static constexpr int T(int d) { return d == 0 ? T0 : d == 1 ? T1 : d == 2 ? T2 : T3; }
  __host__ __device__ static constexpr int face_slots(int d) { return d == 0 ? B / T0 : 2 * (B / T(d)); }
  // first slot of the face(s) of direction d in a kernel of direction mu
  __host__ __device__ static constexpr int face_base(int mu, int d) {
    int o = B;
    for (int k = 0; k < d; ++k) if (k != mu) o += face_slots(k);
    return o;
  }
  __host__ __device__ static constexpr int res_slots(int mu) { return face_base(mu, 4); }
};

// K ring slots per thread (K-1 links in flight); the ring carries, per direction nu, the four links
//   r=0  U3  = U_nu(x)      r=1  U1  = U_nu(x+mu)      r=2  U1' = U_nu(x+mu-nu)      r=3  U3' = U_nu(x-nu)
// and last the own link; link n = 4 i + r goes to slot n % K (ROLL, the rolled loop over nu, needs K | 4).
// MEAS: fused plaquette measurement of the planes (nu, MU), nu < MU (update.cuh, meas_store).
template <typename R, int MU, bool COMP, int KIND, bool FIELD, typename TD, int K, int MINB, bool ROLL, bool MEAS>
__global__ void __launch_bounds__(TD::B, MINB)
su3_update_tiled_kernel(Geom g, typename PlaneTraits<R, (COMP ? 12 : 18)>::Vec* links, UpdateArgs a) {
  typedef PlaneTraits<R, (COMP ? 12 : 18)> T;
  typedef typename T::Vec Vec;
  constexpr int D = 4, NREAL = COMP ? 12 : 18, NP = T::NP, NR = COMP ? 2 : 3, B = TD::B, RES = TD::res_slots(MU);
  static_assert(!MEAS || MU >= 1, "planes (nu, mu), nu < mu");
  constexpr int NSNAP = !MEAS ? 0 : (MU == D - 1 ? MU - 1 : MU);   // cumulative staple sums kept for the measurement
  static_assert(K >= 2 && K <= 5 && (!ROLL || 4 % K == 0), "ring slots");
  extern __shared__ __align__(16) unsigned char tile_raw[];
  Vec* const res = reinterpret_cast<Vec*>(tile_raw);                        // [plane][RES]
  Vec* const ring = res + NP * RES + threadIdx.x;                            // [slot][plane][B], this thread's column

  // thread -> box-relative coordinates (c0 fastest), CTA -> box origin
  const int p = a.parity;
  int c[4];
  {
    uint32_t t = threadIdx.x;
    c[0] = (int)(t % TD::T0); t /= TD::T0;
    c[1] = (int)(t % TD::T1); t /= TD::T1;
    c[2] = (int)(t % TD::T2); t /= TD::T2;
    c[3] = (int)t;
  }
  SiteCoord sc;
  uint32_t h;
  {
    uint32_t b = logical_block(a);
    uint32_t q = fd_div(b, a.tm.n0); const uint32_t b0 = b - q * a.tm.n0.d; b = q;
    q = fd_div(b, a.tm.n1); const uint32_t b1 = b - q * a.tm.n1.d; b = q;
    q = fd_div(b, a.tm.n2); const uint32_t b2 = b - q * a.tm.n2.d; const uint32_t b3 = q;
    sc.j = (int)b0 * TD::T0 + c[0];
    sc.x1 = (int)b1 * TD::T1 + c[1];
    sc.x2 = (int)b2 * TD::T2 + c[2];
    sc.x3 = (int)b3 * TD::T3 + c[3];
    sc.s = (p + sc.x1 + sc.x2 + sc.x3) & 1;
    h = (uint32_t)(((sc.x3 * g.L[2] + sc.x2) * g.L[1] + sc.x1) * g.Lh0 + sc.j);
  }
  const int s = sc.s;
  int fo[D], bo[D];
#pragma unroll
  for (int d = 0; d < D; ++d) nbr_offsets(g, sc, d, fo[d], bo[d]);
  Vec* const own_ptr = (Vec*)a.pbase[MU];
  const Vec* const qmu_ptr = (const Vec*)a.qbase[MU];
  // In-array vector offsets.  The boxes are 8 half-indices wide, so Lh0 and with it every stride of a direction >= 1 is a
  // multiple of 8: such a step moves whole blocks, blk_off(h + o) = blk_off(h) + NP o.  Only a step along direction 0
  // (k0 = +1 forward, -1 backward) moves inside the row and takes the full formula -- three evaluations per thread
  // instead of one per link.
  const uint32_t vh = blk_off<NP>(h), vf0 = blk_off<NP>(h + (uint32_t)fo[0]), vb0 = blk_off<NP>(h + (uint32_t)bo[0]);
  auto at = [&](const Vec* base, int k0, int rest) -> const Vec* {
    return base + ((k0 == 0 ? vh : k0 > 0 ? vf0 : vb0) + mul_planes<NP>((uint32_t)rest));
  };
  constexpr int F0 = (MU == 0) ? 1 : 0;                                      // x + mu: direction-0 part ...
  const int frest = (MU == 0) ? 0 : fo[MU];                                  // ... and the rest
  const uint32_t lex = lex_global(g, sc);
  const int lin = (int)threadIdx.x;                                          // slot of box element c
  // index of c inside the face of direction d (the d-th coordinate dropped)
  auto lin3 = [&](int d) -> int {
    return d == 0 ? c[1] + TD::T1 * (c[2] + TD::T2 * c[3])
         : d == 1 ? c[0] + TD::T0 * (c[2] + TD::T2 * c[3])
         : d == 2 ? c[0] + TD::T0 * (c[1] + TD::T1 * c[3])
                  : c[0] + TD::T0 * (c[1] + TD::T1 * c[2]);
  };

  // ---- resident region: U_mu^q on the box and its faces, every element fetched by exactly one thread.  Unless the update
  // kernel running just before this one writes the array (q, mu) -- in sweep order it never does -- the region is fetched
  // before griddepcontrol.wait, while that kernel drains.
  auto stage_resident = [&]() {
    auto stage = [&](int slot, const Vec* src) {
#pragma unroll
      for (int k = 0; k < NP; ++k) cp_async_vec<(int)sizeof(Vec)>(res + k * RES + slot, src + k * PLANE_STRIDE);
    };
    stage(lin, at(qmu_ptr, 0, 0));
#pragma unroll
    for (int d = 0; d < D; ++d) {
      if (d == MU) continue;
      const int fb = TD::face_base(MU, d), l3 = lin3(d);
      if (d == 0) {
        // a row with s = 0 needs j-1 of its first site, a row with s = 1 needs j+1 of its last site
        if (c[0] == 0 && s == 0) stage(fb + l3, at(qmu_ptr, -1, 0));
        if (c[0] == TD::T0 - 1 && s == 1) stage(fb + l3, at(qmu_ptr, 1, 0));
      } else {
        if (c[d] == 0) stage(fb + l3, at(qmu_ptr, 0, bo[d]));
        if (c[d] == TD::T(d) - 1) stage(fb + B / TD::T(d) + l3, at(qmu_ptr, 0, fo[d]));
      }
    }
    cp_async_commit();
  };

  // ---- ring
  struct Dir { const Vec *pp, *qp; int b0, brest, nu; };              // x - nu: direction-0 part (-1 or 0) and the rest
  auto make_dir = [&](int i) {
    Dir d;
    d.nu = i + (i >= MU ? 1 : 0);
    d.b0 = (d.nu == 0) ? -1 : 0;
    d.brest = 0;
#pragma unroll
    for (int k = 1; k < D; ++k) if (d.nu == k) d.brest = bo[k];
    d.pp = (const Vec*)a.pbase[d.nu];
    d.qp = (const Vec*)a.qbase[d.nu];
    return d;
  };
  auto ring_idx = [&](auto rc, const Dir& d) -> const Vec* {
    constexpr int RR = decltype(rc)::value;
    if constexpr (RR == 0) return at(d.pp, 0, 0);
    else if constexpr (RR == 1) return at(d.qp, F0, frest);
    else if constexpr (RR == 2) return at(d.pp, F0 + d.b0, frest + d.brest);
    else if constexpr (RR == 3) return at(d.qp, d.b0, d.brest);
    else return at(own_ptr, 0, 0);
  };
  auto issue = [&](int n, const Vec* src) {                     // link n of the sequence -> slot n % K
    Vec* dst = ring + (n % K) * NP * B;
#pragma unroll
    for (int k = 0; k < NP; ++k) cp_async_vec<(int)sizeof(Vec)>(dst + k * B, src + k * PLANE_STRIDE);
  };
  auto from_ring = [&](int n, M3<R>& u, bool row2) {
    const Vec* src = ring + (n % K) * NP * B;
    R r[NREAL];
#pragma unroll
    for (int k = 0; k < NP; ++k) vec_unpack(src[k * B], r + k * T::VW);
    m3_from_reals<R, NREAL>(u, r);
    if (COMP && row2) m3_complete_row2(u);
  };
  auto from_res = [&](int slot, M3<R>& u, bool row2) {
    R r[NREAL];
#pragma unroll
    for (int k = 0; k < NP; ++k) vec_unpack(res[k * RES + slot], r + k * T::VW);
    m3_from_reals<R, NREAL>(u, r);
    if (COMP && row2) m3_complete_row2(u);
  };

  // The first K-1 ring links come from the arrays (p, nu0), (q, nu0) of the first direction: same rule.
  Dir cur = make_dir(0);
  auto prologue = [&]() { static_for<0, K - 1>([&](auto rc) { issue(decltype(rc)::value, ring_idx(rc, cur)); cp_async_commit(); }); };
  const bool early_res = a.prev_parity != -2 && !(a.prev_parity == 1 - p && a.prev_mu == MU);   // -2: every array was just written
  const bool early_ring = early_res && a.prev_mu != cur.nu;
  if (early_res) stage_resident();
  if (early_ring) prologue();
  pdl_wait();                                                  // the previous sub-step's links are complete and visible
  pdl_trigger();                                               // after the wait: at most one earlier update kernel is in flight
  if (!early_res) stage_resident();
  if (!early_ring) prologue();

  M3<R> A, P, Q;
  m3_zero(A);
  Row2Sum<R> row2;                                             // third row of the staple sum, unreduced (sun_math.cuh)
  row2.zero();
  M3<R> snap[NSNAP > 0 ? NSNAP : 1];
  auto phase = [&](int i) {
    const bool last = (i == D - 2);
    const Dir nxt = make_dir(last ? i : i + 1);
    const int nu = cur.nu;
    // keep K-1 links in flight, then wait for link 4 i + r
    auto ring_step = [&](auto rc) {
      constexpr int RR = decltype(rc)::value, RA = RR + K - 1;
      if constexpr (RA < 4) {
        issue(4 * i + RA, ring_idx(std::integral_constant<int, RA>{}, cur));
      } else {
        if (!last) issue(4 * i + RA, ring_idx(std::integral_constant<int, RA - 4>{}, nxt));
        else if (RA == 4) issue(4 * i + RA, at(own_ptr, 0, 0));          // the own link, once, after the last direction
      }
      cp_async_commit();                                       // one group per step, possibly empty
      cp_async_wait<K - 1>();
    };
    // slots of U_mu(x+nu), U_mu(x-nu) in the resident region
    int cnu = c[0], Tnu = TD::T0, stnu = 1, fb = TD::face_base(MU, 0), l3 = lin3(0), hi_off = 0;
#pragma unroll
    for (int k = 1; k < D; ++k)
      if (nu == k) {
        cnu = c[k]; Tnu = TD::T(k); fb = TD::face_base(MU, k); l3 = lin3(k); hi_off = B / TD::T(k);
        stnu = (k == 1) ? TD::T0 : (k == 2) ? TD::T0 * TD::T1 : TD::T0 * TD::T1 * TD::T2;
      }
    const int up = (nu == 0) ? s : 1, dn = (nu == 0) ? s - 1 : -1;
    const int slot_up = (cnu + up < Tnu) ? lin + up * stnu : fb + hi_off + l3;
    const int slot_dn = (cnu + dn >= 0) ? lin + dn * stnu : fb + l3;
    const int fsign = !FIELD ? 0 : (MU == a.f.mu && nu == a.f.nu) ? 1 : (MU == a.f.nu && nu == a.f.mu) ? -1 : 0;

    ring_step(std::integral_constant<int, 0>{});
    if (i == 0) __syncthreads();                               // the resident region is complete (every thread waited for its part)
    {                                                          // upper staple  U1 (U3 U2)^+
      from_res(slot_up, P, true);                              // U2 = U_mu(x+nu), all rows
      M3<R> U3;
      from_ring(4 * i + 0, U3, false);
      m3_zero(Q);
      m3_mad_nn<R, NR>(Q, U3, P);                              // X = U3 U2
      if (COMP) m3_complete_row2(Q);
      ring_step(std::integral_constant<int, 1>{});
      M3<R> U1;
      from_ring(4 * i + 1, U1, false);
      if (COMP || FIELD) {
        M3<R> Sm;
        m3_zero(Sm);
        m3_mad_nd<R, NR>(Sm, U1, Q);                           // U1 X^+
        if constexpr (COMP && !FIELD) {
          m3_add_rows01(A, Sm);
          row2.add(A, Sm);
        } else {
          if (COMP) m3_complete_row2(Sm);
          if (FIELD && fsign != 0) su3_scale_cols(Sm, a.f, fsign < 0);
          m3_add(A, Sm);
        }
      } else {
        m3_mad_nd<R, 3>(A, U1, Q);
      }
    }
    {                                                          // lower staple  (U2' U1')^+ U3'
      ring_step(std::integral_constant<int, 2>{});
      from_ring(4 * i + 2, P, true);                           // U1' = U_nu(x+mu-nu), all rows
      M3<R> U2;
      from_res(slot_dn, U2, false);                            // U2' = U_mu(x-nu)
      m3_zero(Q);
      m3_mad_nn<R, NR>(Q, U2, P);                              // Y = U2' U1'
      if (COMP) m3_complete_row2(Q);
      ring_step(std::integral_constant<int, 3>{});
      M3<R> U3;
      from_ring(4 * i + 3, U3, true);
      if (FIELD && fsign != 0) su3_scale_rows(U3, a.f, fsign > 0);
      if (COMP) {
        M3<R> Sm;
        m3_zero(Sm);
        m3_mad_dn<R, 2>(Sm, Q, U3);                            // Y^+ U3'
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
    cur = nxt;
    if constexpr (NSNAP > 0) {
#pragma unroll
      for (int k = 0; k < NSNAP; ++k) if (i == k) { snap[k] = A; row2.finish(snap[k]); }
    }
  };
  if constexpr (ROLL) {
#pragma unroll 1
    for (int i = 0; i < D - 1; ++i) phase(i);
  } else {
#pragma unroll
    for (int i = 0; i < D - 1; ++i) phase(i);
  }

  row2.finish(A);
  // own link: the last one through the ring
  cp_async_wait<0>();
  M3<R> U;
  from_ring(4 * (D - 1), U, true);

  if constexpr (KIND == 1) {
    int cd;
    HbDraw<R> none;
    none.E = none.w = none.n1 = none.n2 = none.n3 = R(0);
    su3_subgroup_hit<R, KIND, 0, 1>(U, A, lex, a, MU, 0, none, cd);
    su3_subgroup_hit<R, KIND, 0, 2>(U, A, lex, a, MU, 1, none, cd);
    su3_subgroup_hit<R, KIND, 1, 2>(U, A, lex, a, MU, 2, none, cd);
  } else {
    int c0, c1, c2;
    su3_subgroup_hit<R, KIND, 0, 1>(U, A, lex, a, MU, 0, hb_first_draw<R>(lex, a, MU, 0), c0);
    su3_subgroup_hit<R, KIND, 0, 2>(U, A, lex, a, MU, 1, hb_first_draw<R>(lex, a, MU, 1), c1);
    su3_subgroup_hit<R, KIND, 1, 2>(U, A, lex, a, MU, 2, hb_first_draw<R>(lex, a, MU, 2), c2);
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
      t[j] = (double)c - (double)prev;
      prev = c;
    }
    meas_store<MU>(a, t);
  }
  R r[NREAL];
  m3_to_reals<R, NREAL>(U, r);
  store_reals<R, NREAL>(own_ptr, g, 0, h, r);
  halo_push_store<R, NREAL>(a, g, sc, r);
}

}  // namespace qcd
