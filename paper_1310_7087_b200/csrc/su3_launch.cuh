// su3_launch.cuh -- host-side selection of the SU(3) update kernel instantiation and its shared-memory geometry.
// Every shape below was chosen by measurement at 32^4 on B200 (profiles/); they are compile-time
// constants of the product, not run-time switches.
#pragma once
#include <atomic>
#include <cstring>

#include "launch.h"
#include "update_bulk.cuh"

namespace qcd {

// ---- tiled kernel (update_tiled.cuh), D = 4: box of sites per CTA for direction mu (extent 0 in half-indices): 128 sites,
// extent 1 in direction mu, where the box needs no faces (mu = 0: extent 1 in direction 3).
template <int MU> struct TileFor;
template <> struct TileFor<0> { typedef TileDims<8, 4, 4, 1> TD; };
template <> struct TileFor<1> { typedef TileDims<8, 1, 4, 4> TD; };
template <> struct TileFor<2> { typedef TileDims<8, 4, 1, 4> TD; };
template <> struct TileFor<3> { typedef TileDims<8, 4, 4, 1> TD; };
// The resident region pays only for fp32 x12 overrelaxation (DESIGN.md sec 6.6 / 6.7): the fp64 kernels lose more from
// the occupancy the region costs than they gain from the lighter L2 traffic.  K ring slots, MINB CTAs per SM.
template <typename R, bool COMP, int KIND> struct TiledCfg { static constexpr bool ON = false; static constexpr int K = 2, MINB = 1; };
template <> struct TiledCfg<float, true, 1> { static constexpr bool ON = true; static constexpr int K = 5, MINB = 4; };

// ---- bulk-copy kernel (update_bulk.cuh), D = 4, L0 = 32, fp32 x12 overrelaxation without field: producer warp + mbarriers.
// Instantiated, but run only on request (QCD_OPT_BULK_COPY): it is slower than the tiled kernel (DESIGN.md sec 6.10,
// profiles/r2_a_launches_and_ncu.md) and is kept so that the measurement can be repeated.
template <typename R, bool COMP, int KIND, bool FIELD, bool MEAS> struct BulkCfg { static constexpr bool ON = false; static constexpr int K = 5, MINB = 4; };
template <> struct BulkCfg<float, true, 1, false, false> { static constexpr bool ON = true; static constexpr int K = 5, MINB = 4; };
// boxes of the bulk kernel: the full x0 row (16 half-indices: L0 = 32) x 8 rows, thin in mu where that keeps T1 = 4
template <int MU> struct BulkTileFor { typedef TileDims<16, 4, 2, 1> TD; };
template <> struct BulkTileFor<2> { typedef TileDims<16, 4, 1, 2> TD; };

// ---- ring kernel (update.cuh): B threads per CTA, K link slots per thread (K-1 links in flight; K = 0: direct global
// loads), MINB = second __launch_bounds__ argument.  Shared memory per CTA = K * (bytes per link) * B.
template <int B_, int K_, int MINB_> struct RingShape { static constexpr int B = B_, K = K_, MINB = MINB_; };
template <typename R, bool COMP> struct RingCfg;
template <> struct RingCfg<float, true> : RingShape<128, 6, 1> {};
template <> struct RingCfg<float, false> : RingShape<128, 0, 1> {};
template <> struct RingCfg<double, true> : RingShape<64, 6, 1> {};
template <> struct RingCfg<double, false> : RingShape<128, 3, 3> {};
// Ring slots of the UNROLLED overrelaxation kernels (any K >= 2: the slot of a link is its sequence number mod K); the
// heatbath kernels, whose direction loop is rolled, need K | 6 and take the K above.  -1: same as the heatbath kernel.
template <typename R, bool COMP> struct RingKOr { static constexpr int K = -1; };
template <> struct RingKOr<double, false> { static constexpr int K = 4; };
// Loop shape per kind: ROLL = the direction loop of the heatbath kernels is kept rolled (their straight-line code would
// be 60+ KB).  The three subgroup hits are unrolled in both precisions (round 2: a rolled hit on a permuted frame cost
// ~150 register moves per link: fp32 HB 79.5 -> 76.9 us, fp64 HB 190 -> 181 us on the same box).
template <int KIND> struct LoopCfg { static constexpr bool ROLL = (KIND == 0); };

// Tile of B threads of the ring kernel: 8 half-indices along x0 (one 128-byte line of 16-byte vectors), the rest spread
// over x1, x2, x3 in powers of two; every extent must divide the lattice, else the linear mapping is used.
static inline TileMap choose_tile(const Geom& g, int B) {
  TileMap tm;
  memset(&tm, 0, sizeof(tm));
  if (g.D != 4 || (B & (B - 1))) return tm;
  int lb = 0;
  while ((1 << lb) < B) ++lb;
  auto pow2_part = [](int x) { int s = 0; while (!(x & 1)) { x >>= 1; ++s; } return s; };
  // the tiles cover the sites the launch visits: the interior extents Li (= L unless the lattice is a slab)
  const int m[4] = {pow2_part(g.Lh0), pow2_part(g.Li[1]), pow2_part(g.Li[2]), pow2_part(g.Li[3])};
  int s[4] = {m[0] < 3 ? m[0] : 3, 0, 0, 0};
  int left = lb - s[0];
  for (int d = 1; left > 0; d = d % 3 + 1) {
    bool any = false;
    for (int k = 1; k < 4; ++k) any = any || s[k] < m[k];
    if (!any) break;
    if (s[d] < m[d]) { ++s[d]; --left; }
  }
  if (left > 0) s[0] += left;
  for (int d = 0; d < 4; ++d) if (s[d] > m[d]) return tm;
  tm.on = 1; tm.s0 = s[0]; tm.s1 = s[1]; tm.s2 = s[2];
  tm.n0 = make_fastdiv((uint32_t)(g.Lh0 >> s[0])); tm.n1 = make_fastdiv((uint32_t)(g.Li[1] >> s[1])); tm.n2 = make_fastdiv((uint32_t)(g.Li[2] >> s[2]));
  return tm;
}

// array starts for the kernels (UpdateArgs::pbase / qbase)
template <typename Vec> static void fill_bases(UpdateArgs& a, const Geom& g, void* links, int NP) {
  const size_t arr = (size_t)NP * g.Vh_pad;
  for (int nu = 0; nu < 4; ++nu) {
    a.pbase[nu] = nu < g.D ? (const void*)((Vec*)links + (size_t)(a.parity * g.D + nu) * arr) : nullptr;
    a.qbase[nu] = nu < g.D ? (const void*)((Vec*)links + (size_t)((1 - a.parity) * g.D + nu) * arr) : nullptr;
  }
}

// opt in to > 48 KB of dynamic shared memory once per (kernel instantiation, device); `done` is a per-instantiation
// bit mask over device ordinals.  Racing host threads at worst both set the (idempotent) attribute.
template <typename Kern> static cudaError_t ensure_smem(Kern kern, size_t smem, std::atomic<uint64_t>& done) {
  if (smem <= 48 * 1024) return cudaSuccess;
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  const uint64_t bit = 1ull << (dev & 63);
  if (done.load(std::memory_order_acquire) & bit) return cudaSuccess;
  e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e == cudaSuccess) done.fetch_or(bit, std::memory_order_release);
  return e;
}

template <typename R, int MU, bool COMP, int KIND, bool FIELD, bool MEAS>
static cudaError_t su3_go_tiled(const Geom& g, void* links, const UpdateArgs& a, cudaStream_t st) {
  typedef PlaneTraits<R, (COMP ? 12 : 18)> T;
  typedef typename T::Vec Vec;
  typedef typename TileFor<MU>::TD TD;
  constexpr int K = TiledCfg<R, COMP, KIND>::K, MINB = TiledCfg<R, COMP, KIND>::MINB;
  constexpr bool ROLL = LoopCfg<KIND>::ROLL && (4 % K == 0);
  constexpr size_t smem = (size_t)(TD::res_slots(MU) + K * TD::B) * T::NP * sizeof(Vec);
  auto kern = su3_update_tiled_kernel<R, MU, COMP, KIND, FIELD, TD, K, MINB, ROLL, MEAS>;
  static std::atomic<uint64_t> done{0};
  cudaError_t e = ensure_smem(kern, smem, done);
  if (e != cudaSuccess) return e;
  UpdateArgs a2 = a;
  memset(&a2.tm, 0, sizeof(a2.tm));
  a2.tm.on = 1;
  a2.tm.n0 = make_fastdiv((uint32_t)(g.Lh0 / TD::T0)); a2.tm.n1 = make_fastdiv((uint32_t)(g.Li[1] / TD::T1));
  a2.tm.n2 = make_fastdiv((uint32_t)(g.Li[2] / TD::T2));
  fill_bases<Vec>(a2, g, links, T::NP);
  return launch_pdl(kern, dim3(g.Vh_int / TD::B), dim3(TD::B), smem, st, g, (Vec*)links, a2);
}

template <typename R, int MU, bool COMP, int KIND, bool FIELD>
static cudaError_t su3_go_bulk(const Geom& g, void* links, const UpdateArgs& a, cudaStream_t st) {
  typedef PlaneTraits<R, (COMP ? 12 : 18)> T;
  typedef typename T::Vec Vec;
  typedef typename BulkTileFor<MU>::TD TD;
  constexpr int K = BulkCfg<R, COMP, KIND, FIELD, false>::K, MINB = BulkCfg<R, COMP, KIND, FIELD, false>::MINB;
  constexpr int ROWS = TD::B / TD::T0, ROWV = T::NP * TD::T0;
  constexpr int RROWS = ROWS + (MU != 1 ? 2 * (ROWS / TD::T1) : 0) + (MU != 2 ? 2 * (ROWS / TD::T2) : 0) + (MU != 3 ? 2 * (ROWS / TD::T3) : 0);
  constexpr size_t smem = (size_t)(RROWS * ROWV + K * ROWS * ROWV) * sizeof(Vec) + (2 * K + 1) * 8;
  auto kern = su3_update_bulk_kernel<R, MU, COMP, KIND, FIELD, TD, K, MINB>;
  static std::atomic<uint64_t> done{0};
  cudaError_t e = ensure_smem(kern, smem, done);
  if (e != cudaSuccess) return e;
  UpdateArgs a2 = a;
  memset(&a2.tm, 0, sizeof(a2.tm));
  a2.tm.on = 1;
  a2.tm.n0 = make_fastdiv(1u); a2.tm.n1 = make_fastdiv((uint32_t)(g.Li[1] / TD::T1));
  a2.tm.n2 = make_fastdiv((uint32_t)(g.Li[2] / TD::T2));
  return launch_pdl(kern, dim3(g.Vh_int / TD::B), dim3(TD::B + 32), smem, st, g, (Vec*)links, a2);
}

template <typename R, int D, int MU, bool COMP, int KIND, bool FIELD, bool MEAS>
static cudaError_t su3_go(const Geom& g, void* links, const UpdateArgs& a, cudaStream_t st) {
  typedef PlaneTraits<R, (COMP ? 12 : 18)> T;
  typedef typename T::Vec Vec;
  if constexpr (D == 4 && BulkCfg<R, COMP, KIND, FIELD, MEAS>::ON) {
    typedef typename BulkTileFor<MU>::TD TD;
    // the box spans the whole x0 row (L0 = 32); a slab's halo layers are not visited: plain lattices only
    if (a.use_bulk && g.sd < 0 && g.Lh0 == TD::T0 && g.L[1] % TD::T1 == 0 && g.L[2] % TD::T2 == 0 && g.L[3] % TD::T3 == 0)
      return su3_go_bulk<R, MU, COMP, KIND, FIELD>(g, links, a, st);
  }
  if constexpr (D == 4 && TiledCfg<R, COMP, KIND>::ON) {
    typedef typename TileFor<MU>::TD TD;
    if (g.Lh0 % TD::T0 == 0 && g.Li[1] % TD::T1 == 0 && g.Li[2] % TD::T2 == 0 && g.Li[3] % TD::T3 == 0)
      return su3_go_tiled<R, MU, COMP, KIND, FIELD, MEAS>(g, links, a, st);
  }
  constexpr bool ROLL = LoopCfg<KIND>::ROLL;
  constexpr int B = RingCfg<R, COMP>::B, MINB = RingCfg<R, COMP>::MINB;
  constexpr int K = (KIND == 1 && !ROLL && RingKOr<R, COMP>::K >= 0) ? RingKOr<R, COMP>::K : RingCfg<R, COMP>::K;
  constexpr size_t smem = (size_t)K * T::NP * B * sizeof(Vec) + (KIND == 0 ? (size_t)15 * B * sizeof(R) : 0);
  auto kern = su3_update_kernel<R, D, MU, COMP, KIND, FIELD, B, K, MINB, ROLL, MEAS>;
  static std::atomic<uint64_t> done{0};
  cudaError_t e = ensure_smem(kern, smem, done);
  if (e != cudaSuccess) return e;
  const unsigned grid = (g.Vh_int + B - 1) / B;
  UpdateArgs a2 = a;
  a2.tm = choose_tile(g, B);
  fill_bases<Vec>(a2, g, links, T::NP);
  return launch_pdl(kern, dim3(grid), dim3(B), smem, st, g, (Vec*)links, a2);
}
// MEAS = the fused-measurement variants (update.cuh, meas_store): instantiated by their own translation units; they exist
// for mu >= 1 only (the planes (nu, mu), nu < mu)
template <typename R, int D, int MU, bool COMP, bool MEAS>
static cudaError_t su3_sel_kind(const UpdateSel& s, const Geom& g, void* links, const UpdateArgs& a, cudaStream_t st) {
  if constexpr (MEAS && MU == 0) {
    return cudaErrorInvalidValue;
  } else {
    if (s.kind == 0) return s.field ? su3_go<R, D, MU, COMP, 0, true, MEAS>(g, links, a, st) : su3_go<R, D, MU, COMP, 0, false, MEAS>(g, links, a, st);
    return s.field ? su3_go<R, D, MU, COMP, 1, true, MEAS>(g, links, a, st) : su3_go<R, D, MU, COMP, 1, false, MEAS>(g, links, a, st);
  }
}
template <typename R, int D, int MU, bool MEAS>
static cudaError_t su3_sel_comp(const UpdateSel& s, const Geom& g, void* links, const UpdateArgs& a, cudaStream_t st) {
  return s.comp ? su3_sel_kind<R, D, MU, true, MEAS>(s, g, links, a, st) : su3_sel_kind<R, D, MU, false, MEAS>(s, g, links, a, st);
}
template <typename R, int D, bool MEAS>
static cudaError_t su3_sel_mu(const UpdateSel& s, const Geom& g, void* links, const UpdateArgs& a, cudaStream_t st) {
  switch (a.mu) {
    case 0: return su3_sel_comp<R, D, 0, MEAS>(s, g, links, a, st);
    case 1: return su3_sel_comp<R, D, 1, MEAS>(s, g, links, a, st);
    case 2: if constexpr (D > 2) return su3_sel_comp<R, D, 2, MEAS>(s, g, links, a, st); break;
    case 3: if constexpr (D > 3) return su3_sel_comp<R, D, 3, MEAS>(s, g, links, a, st); break;
  }
  return cudaErrorInvalidValue;
}

}  // namespace qcd
