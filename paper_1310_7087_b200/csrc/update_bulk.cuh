// update_bulk.cuh -- the D = 4 SU(3) sub-step with ALL operands staged by bulk asynchronous copies (cp.async.bulk, the
// TMA unit's 1-D form; SASS UBLKCP) that a producer warp issues and mbarriers complete: the 128 consumer threads of a CTA
// spend no issue slots on global addresses or copy instructions.
//
// Why: with the blocked link layout [h/8][plane][h%8] a row of 8 sites of one (parity, direction)
// array is ONE contiguous 384-byte (fp32 x12) segment, so a whole operand of a CTA's box of 128 sites (16 rows) is 16
// bulk copies; an operand shifted by one site along direction 0 is displaced by one half-index on the rows of one
// row-parity and takes 2 pieces per plane there.  The per-thread cp.async ring of update.cuh / update_tiled.cuh issues 51
// LDGSTS and ~200 address instructions per thread instead.
//
// A first form (boxes 8 half-indices wide, one 384-byte copy per row and operand, 2 pieces per plane on shifted rows) was
// correct and 2.8 times SLOWER than the tiled kernel (126 us against 46 us at 32^4): UBLKCP is a warp-uniform instruction
// (uniform-register operands), so the ~350 copies of a CTA are issued one after the other by the producer warp.  This
// form cuts the copies to ~40 per CTA:
//   * the box spans the FULL x0 row (T0 = Lh0 = 16 half-indices, i.e. L0 = 32): lattice rows that are consecutive in x1 are
//     consecutive in memory, so T1 rows of an operand are ONE copy of T1 * 768 bytes;
//   * a step along direction 0 moves a site to another element of the SAME row (periodic wrap included), so operands
//     shifted along 0 need no other copy: the consumer reads element (j + shift) mod Lh0, and U_mu needs no x0 face.
// Structure: box Lh0 x T1 x T2 x T3 = 128 sites per CTA;
//   resident region  U_mu^q on the box and its faces in the directions 1..3 other than mu (rows of [2 blocks][plane][8]),
//   ring of K CTA-wide slots, each one operand of all 128 threads (8 rows, 6 KB): per direction nu
//       r=0  U_nu(x)   r=1  U_nu(x+mu)   r=2  U_nu(x+mu-nu)   r=3  U_nu(x-nu)        and last the own link,
//   mbarriers full[K] (expect_tx = 6144 bytes per slot), empty[K] (128 consumer arrivals), one for the resident region.
// Warp 4 is the producer: lane l < T2 T3 owns the run of T1 rows at (x2, x3) = box origin + l.  The arithmetic is the one
// of update_tiled.cuh.
#pragma once
#include "update_tiled.cuh"

namespace qcd {

__device__ __forceinline__ void mbar_init(uint64_t* bar, unsigned count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"((unsigned)__cvta_generic_to_shared(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, unsigned bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"((unsigned)__cvta_generic_to_shared(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"((unsigned)__cvta_generic_to_shared(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, unsigned parity) {
  const unsigned a = (unsigned)__cvta_generic_to_shared(bar);
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "WAIT_%=:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra DONE_%=;\n"
      "bra WAIT_%=;\n"
      "DONE_%=:\n"
      "}\n" ::"r"(a), "r"(parity)
      : "memory");
}
// 1-D bulk copy global -> shared, completion counted in bytes on an mbarrier (16-byte aligned addresses, size % 16 == 0)
__device__ __forceinline__ void bulk_g2s(void* smem_dst, const void* gmem_src, unsigned bytes, uint64_t* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                   (unsigned)__cvta_generic_to_shared(smem_dst)),
               "l"(gmem_src), "r"(bytes), "r"((unsigned)__cvta_generic_to_shared(bar))
               : "memory");
}

template <typename R, int MU, bool COMP, int KIND, bool FIELD, typename TD, int K, int MINB>
__global__ void __launch_bounds__(TD::B + 32, MINB)
su3_update_bulk_kernel(Geom g, typename PlaneTraits<R, (COMP ? 12 : 18)>::Vec* links, UpdateArgs a) {
  typedef PlaneTraits<R, (COMP ? 12 : 18)> T;
  typedef typename T::Vec Vec;
  constexpr int D = 4, NREAL = COMP ? 12 : 18, NP = T::NP, NR = COMP ? 2 : 3, B = TD::B;
  constexpr int LH = TD::T0;                                                   // = Lh0: the box spans the whole x0 row
  static_assert(LH == 16 && sizeof(Vec) == 16, "full rows of 16 half-indices, 16-byte vectors");
  static_assert(KIND == 1, "overrelaxation only (the heatbath keeps the ring kernel)");
  constexpr int ROWS = B / LH, ROWV = NP * LH;                                 // rows per operand, vectors per row (768 bytes)
  constexpr int RUNS = TD::T2 * TD::T3;                                        // runs of T1 consecutive rows
  // rows of the resident region: the box, then per direction d = 1..3 (d != MU) its low and high face
  constexpr int FR1 = ROWS / TD::T1, FR2 = ROWS / TD::T2, FR3 = ROWS / TD::T3;
  constexpr int FB1 = ROWS, FB2 = FB1 + (MU != 1 ? 2 * FR1 : 0), FB3 = FB2 + (MU != 2 ? 2 * FR2 : 0), RROWS = FB3 + (MU != 3 ? 2 * FR3 : 0);
  constexpr int NSEQ = 4 * (D - 1) + 1;
  extern __shared__ __align__(128) unsigned char bulk_raw[];
  Vec* const res = reinterpret_cast<Vec*>(bulk_raw);                          // [RROWS][2][NP][8]
  Vec* const ring = res + RROWS * ROWV;                                       // [K][ROWS][2][NP][8]
  uint64_t* const bars = reinterpret_cast<uint64_t*>(ring + K * ROWS * ROWV); // full[K], empty[K], resident
  uint64_t* const full = bars;
  uint64_t* const empty = bars + K;
  uint64_t* const resbar = bars + 2 * K;

  const int p = a.parity;
  // CTA -> box origin (the box covers x0 completely)
  uint32_t bb = logical_block(a);
  uint32_t qd = fd_div(bb, a.tm.n1); const uint32_t b1 = bb - qd * a.tm.n1.d; bb = qd;
  qd = fd_div(bb, a.tm.n2); const uint32_t b2 = bb - qd * a.tm.n2.d; const uint32_t b3 = qd;
  const int o1 = (int)b1 * TD::T1, o2 = (int)b2 * TD::T2, o3 = (int)b3 * TD::T3;
  const size_t arr = (size_t)NP * g.Vh_pad;

  if (threadIdx.x == 0) {
#pragma unroll
    for (int k = 0; k < K; ++k) { mbar_init(full + k, 1); mbar_init(empty + k, B); }
    mbar_init(resbar, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();

  if (threadIdx.x >= B) {
    // ===================================================================== producer warp
    const int lane = (int)threadIdx.x - B;
    const int r2 = lane % TD::T2, r3 = lane / TD::T2;                        // run `lane`: rows x1 = o1 .. o1 + T1 - 1 at (x2, x3)
    const bool has_run = lane < RUNS;
    const int x2 = o2 + r2, x3 = o3 + r3;
    auto wrap = [](int x, int L) { return x < 0 ? x + L : (x >= L ? x - L : x); };
    // vector index of element j = 0 of row (y1, y2, y3) inside one (parity, direction) array
    auto row_v = [&](int y1, int y2, int y3) -> size_t { return (size_t)((y3 * g.L[2] + y2) * g.L[1] + y1) * ROWV; };
    // nrows consecutive rows x1 = y1 .. y1 + nrows - 1 (mod L1) at (y2, y3): one copy, or two when the run crosses the wrap
    auto copy_rows = [&](Vec* dst, const Vec* base, int y1, int y2, int y3, int nrows, uint64_t* bar) {
      y1 = wrap(y1, g.L[1]); y2 = wrap(y2, g.L[2]); y3 = wrap(y3, g.L[3]);
      const int first = (y1 + nrows <= g.L[1]) ? nrows : g.L[1] - y1;
      bulk_g2s(dst, base + row_v(y1, y2, y3), (unsigned)(first * ROWV * 16), bar);
      if (first < nrows) bulk_g2s(dst + first * ROWV, base + row_v(0, y2, y3), (unsigned)((nrows - first) * ROWV * 16), bar);
    };
    const Vec* const qmu = links + (size_t)((1 - p) * D + MU) * arr;
    auto stage_resident = [&]() {
      if (lane == 0) mbar_expect_tx(resbar, (unsigned)(RROWS * ROWV * 16));
      __syncwarp();
      if (!has_run) return;
      const int run = r2 + TD::T2 * r3;
      copy_rows(res + run * TD::T1 * ROWV, qmu, o1, x2, x3, TD::T1, resbar);
      if (MU != 1) {                                                         // faces x1 = o1 - 1, o1 + T1: one row per run
        copy_rows(res + (FB1 + run) * ROWV, qmu, o1 - 1, x2, x3, 1, resbar);
        copy_rows(res + (FB1 + FR1 + run) * ROWV, qmu, o1 + TD::T1, x2, x3, 1, resbar);
      }
      if (MU != 2) {                                                         // faces x2 = o2 - 1, o2 + T2: T1 rows per x3
        if (r2 == 0) copy_rows(res + (FB2 + TD::T1 * r3) * ROWV, qmu, o1, o2 - 1, x3, TD::T1, resbar);
        if (r2 == TD::T2 - 1) copy_rows(res + (FB2 + FR2 + TD::T1 * r3) * ROWV, qmu, o1, o2 + TD::T2, x3, TD::T1, resbar);
      }
      if (MU != 3) {                                                         // faces x3 = o3 - 1, o3 + T3: T1 rows per x2
        if (r3 == 0) copy_rows(res + (FB3 + TD::T1 * r2) * ROWV, qmu, o1, x2, o3 - 1, TD::T1, resbar);
        if (r3 == TD::T3 - 1) copy_rows(res + (FB3 + FR3 + TD::T1 * r2) * ROWV, qmu, o1, x2, o3 + TD::T3, TD::T1, resbar);
      }
    };
    // operand n of the sequence: array and displacement of its rows (steps along 0 stay inside the row)
    auto stage_ring = [&](int n) {
      const int slot = n % K;
      if (n >= K) mbar_wait(empty + slot, (unsigned)((n / K - 1) & 1));
      if (lane == 0) mbar_expect_tx(full + slot, (unsigned)(ROWS * ROWV * 16));
      __syncwarp();
      if (!has_run) return;
      Vec* dst = ring + (slot * ROWS + (r2 + TD::T2 * r3) * TD::T1) * ROWV;
      if (n == NSEQ - 1) { copy_rows(dst, links + (size_t)(p * D + MU) * arr, o1, x2, x3, TD::T1, full + slot); return; }
      const int i = n >> 2, rr = n & 3, nu = i + (i >= MU ? 1 : 0);
      int d[4] = {0, 0, 0, 0};
      if (rr == 1 || rr == 2) d[MU] += 1;
      if (rr == 2 || rr == 3) d[nu] -= 1;
      const bool qarr = (rr == 1 || rr == 3);
      copy_rows(dst, links + (size_t)((qarr ? 1 - p : p) * D + nu) * arr, o1 + d[1], x2 + d[2], x3 + d[3], TD::T1, full + slot);
    };
    // programmatic dependent launch: before the wait only arrays the previous kernel did not write (update.cuh)
    auto safe = [&](int par_arr, int dir) { return a.prev_parity != -2 && !(a.prev_parity == par_arr && a.prev_mu == dir); };
    bool waited = false;
    auto need_wait = [&](bool ok) { if (!ok && !waited) { pdl_wait(); waited = true; } };
    need_wait(safe(1 - p, MU));
    stage_resident();
#pragma unroll 1
    for (int n = 0; n < NSEQ; ++n) {
      if (!waited) {
        bool ok;
        if (n == NSEQ - 1) ok = safe(p, MU);
        else { const int i = n >> 2, rr = n & 3, nu = i + (i >= MU ? 1 : 0); ok = safe((rr == 1 || rr == 3) ? 1 - p : p, nu); }
        need_wait(ok);
      }
      stage_ring(n);
    }
    if (!waited) pdl_wait();
    return;
  }

  // ======================================================================= consumers: one thread per link
  const int lin = (int)threadIdx.x;
  const int c0 = lin & (LH - 1), row = lin / LH;
  const int c1 = row % TD::T1, c2 = (row / TD::T1) % TD::T2, c3 = row / (TD::T1 * TD::T2);
  SiteCoord sc;
  sc.j = c0; sc.x1 = o1 + c1; sc.x2 = o2 + c2; sc.x3 = o3 + c3;
  sc.s = (p + sc.x1 + sc.x2 + sc.x3) & 1;
  const int s = sc.s;
  const uint32_t h = (uint32_t)(((sc.x3 * g.L[2] + sc.x2) * g.L[1] + sc.x1) * LH + sc.j);
  pdl_wait();                                   // the store of the own link may not pass the previous kernel's reads of that array
  pdl_trigger();

  // element j of row r of a region: rows keep the memory layout [block of 8][plane][8]
  auto load_elem = [&](const Vec* region, int r, int j, M3<R>& u, bool row2) {
    const Vec* src = region + r * ROWV + (j >> 3) * (NP * 8) + (j & 7);
    R rr_[NREAL];
#pragma unroll
    for (int k = 0; k < NP; ++k) vec_unpack(src[k * 8], rr_ + k * T::VW);
    m3_from_reals<R, NREAL>(u, rr_);
    if (COMP && row2) m3_complete_row2(u);
  };
  // operand n of the ring; sh = its displacement along direction 0 in half-indices (inside the row, periodic)
  auto from_ring = [&](int n, int sh, M3<R>& u, bool row2) {
    const int slot = n % K;
    mbar_wait(full + slot, (unsigned)((n / K) & 1));
    load_elem(ring + slot * ROWS * ROWV, row, (c0 + sh) & (LH - 1), u, row2);
    mbar_arrive(empty + slot);
  };
  // U_mu on the other parity at x + nu (up = true) or x - nu from the resident region
  auto from_res = [&](int nu, bool up, M3<R>& u, bool row2) {
    if (nu == 0) {
      load_elem(res, row, (c0 + (up ? s : s - 1)) & (LH - 1), u, row2);
    } else {
      const int cn = nu == 1 ? c1 : nu == 2 ? c2 : c3, Tn = TD::T(nu), rs = nu == 1 ? 1 : nu == 2 ? TD::T1 : TD::T1 * TD::T2;
      const int fb = nu == 1 ? FB1 : nu == 2 ? FB2 : FB3, frn = nu == 1 ? FR1 : nu == 2 ? FR2 : FR3;
      const int fr = nu == 1 ? c2 + TD::T2 * c3 : nu == 2 ? c1 + TD::T1 * c3 : c1 + TD::T1 * c2;
      int rsel;
      if (up) rsel = (cn + 1 < Tn) ? row + rs : fb + frn + fr;
      else rsel = (cn >= 1) ? row - rs : fb + fr;
      load_elem(res, rsel, c0, u, row2);
    }
  };

  M3<R> A, P, Q;
  m3_zero(A);
  mbar_wait(resbar, 0u);
#pragma unroll
  for (int i = 0; i < D - 1; ++i) {
    const int nu = i + (i >= MU ? 1 : 0);
    const int fsign = !FIELD ? 0 : (MU == a.f.mu && nu == a.f.nu) ? 1 : (MU == a.f.nu && nu == a.f.mu) ? -1 : 0;
    // displacements along direction 0 (update_bulk.cuh header): a step +0 from a site with x0 & 1 = s moves the half-index by s,
    // a step -0 by s - 1, and flips s; steps along other directions leave both unchanged
    const int sh1 = (MU == 0) ? s : 0;                                         // x + mu
    const int sh2 = (MU == 0) ? s : (nu == 0 ? s - 1 : 0);                     // x + mu - nu
    const int sh3 = (nu == 0) ? s - 1 : 0;                                     // x - nu
    {                                                          // upper staple  U1 (U3 U2)^+
      from_res(nu, true, P, true);                             // U2 = U_mu(x+nu), all rows
      M3<R> U3;
      from_ring(4 * i + 0, 0, U3, false);
      m3_zero(Q);
      m3_mad_nn<R, NR>(Q, U3, P);                              // X = U3 U2
      if (COMP) m3_complete_row2(Q);
      M3<R> U1;
      from_ring(4 * i + 1, sh1, U1, false);
      if (COMP || FIELD) {
        M3<R> Sm;
        m3_zero(Sm);
        m3_mad_nd<R, NR>(Sm, U1, Q);                           // U1 X^+
        if (COMP) m3_complete_row2(Sm);
        if (FIELD && fsign != 0) su3_scale_cols(Sm, a.f, fsign < 0);
        m3_add(A, Sm);
      } else {
        m3_mad_nd<R, 3>(A, U1, Q);
      }
    }
    {                                                          // lower staple  (U2' U1')^+ U3'
      from_ring(4 * i + 2, sh2, P, true);                      // U1' = U_nu(x+mu-nu), all rows
      M3<R> U2;
      from_res(nu, false, U2, false);                          // U2' = U_mu(x-nu)
      m3_zero(Q);
      m3_mad_nn<R, NR>(Q, U2, P);                              // Y = U2' U1'
      if (COMP) m3_complete_row2(Q);
      M3<R> U3;
      from_ring(4 * i + 3, sh3, U3, true);
      if (FIELD && fsign != 0) su3_scale_rows(U3, a.f, fsign > 0);
      if (COMP) {
        M3<R> Sm;
        m3_zero(Sm);
        m3_mad_dn<R, 2>(Sm, Q, U3);                            // Y^+ U3'
        m3_complete_row2(Sm);
        m3_add(A, Sm);
      } else {
        m3_mad_dn<R, 3>(A, Q, U3);
      }
    }
  }
  M3<R> U;
  from_ring(NSEQ - 1, 0, U, true);
  const uint32_t lex = lex_global(g, sc);
  int cd;
  HbDraw<R> none;
  none.E = none.w = none.n1 = none.n2 = none.n3 = R(0);
  su3_subgroup_hit<R, KIND, 0, 1>(U, A, lex, a, MU, 0, none, cd);
  su3_subgroup_hit<R, KIND, 0, 2>(U, A, lex, a, MU, 1, none, cd);
  su3_subgroup_hit<R, KIND, 1, 2>(U, A, lex, a, MU, 2, none, cd);
  m3_reunitarise(U);
  R r[NREAL];
  m3_to_reals<R, NREAL>(U, r);
  store_reals<R, NREAL>(links, g, (size_t)(p * D + MU) * arr, h, r);
}

}  // namespace qcd
