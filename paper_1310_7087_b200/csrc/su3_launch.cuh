// su3_launch.cuh -- host-side selection of the SU(3) update kernel instantiation and its ring geometry.
#pragma once
#include <cstdio>
#include <cstdlib>
#include <cstring>

#include "launch.h"
#include "update_tiled.cuh"

namespace qcd {

// Tiled kernel (update_tiled.cuh), D = 4 only: box of sites per CTA for direction mu (extent 0 in half-indices; default: 128
// sites, extent 1 in direction mu where the box has no faces; one hex digit per extent), ring slots per thread, CTAs per SM the register allocation
// must allow.  QCD_TILED=0 in the environment, or a lattice the box does not divide, selects the ring kernel of update.cuh.
#ifndef QCD_TILE_MU0
#define QCD_TILE_MU0 0x8441
#endif
#ifndef QCD_TILE_MU1
#define QCD_TILE_MU1 0x8144
#endif
#ifndef QCD_TILE_MU2
#define QCD_TILE_MU2 0x8414
#endif
#ifndef QCD_TILE_MU3
#define QCD_TILE_MU3 0x8441
#endif
#ifndef QCD_TILE_F32X12_K
#define QCD_TILE_F32X12_K 5
#endif
#ifndef QCD_TILE_F32X12_MINB
#define QCD_TILE_F32X12_MINB 4
#endif
template <int X> struct TileHex { typedef TileDims<((X >> 12) & 15), ((X >> 8) & 15), ((X >> 4) & 15), (X & 15)> TD; };
template <int MU> struct TileFor;
template <> struct TileFor<0> { typedef TileHex<QCD_TILE_MU0>::TD TD; };
template <> struct TileFor<1> { typedef TileHex<QCD_TILE_MU1>::TD TD; };
template <> struct TileFor<2> { typedef TileHex<QCD_TILE_MU2>::TD TD; };
template <> struct TileFor<3> { typedef TileHex<QCD_TILE_MU3>::TD TD; };
// Measured at 32^4 (profiles/r1_c_tiling.md): the resident region pays only for fp32 x12 overrelaxation (sustained 52.0
// vs 53.2 us); the fp64 kernels lose more from the occupancy the region costs (2 instead of 3 CTAs per SM) than they gain
// from the lighter L2 traffic, and the heatbath kernels are bound by their random numbers.  Those keep the ring kernel.
template <typename R, bool COMP, int KIND> struct TiledCfg { static constexpr bool ON = false; static constexpr int K = 2, MINB = 1; };
template <> struct TiledCfg<float, true, 1> { static constexpr bool ON = true; static constexpr int K = QCD_TILE_F32X12_K, MINB = QCD_TILE_F32X12_MINB; };

// Ring geometry per storage format: B threads per CTA, K link slots per thread (K-1 links in flight).
// Shared memory per CTA = K * (bytes per link) * B; chosen so that several CTAs fit in the 227 KB of an SM.
// K = 0 selects direct global loads; MINB is the second __launch_bounds__ argument (register cap).
#ifndef QCD_F32X12_B
#define QCD_F32X12_B 128
#endif
#ifndef QCD_F32X12_K
#define QCD_F32X12_K 6
#endif
#ifndef QCD_F32X12_MINB
#define QCD_F32X12_MINB 1
#endif
#ifndef QCD_F32X18_B
#define QCD_F32X18_B 128
#endif
#ifndef QCD_F32X18_K
#define QCD_F32X18_K 0
#endif
#ifndef QCD_F32X18_MINB
#define QCD_F32X18_MINB 1
#endif
#ifndef QCD_F64X12_B
#define QCD_F64X12_B 64
#endif
#ifndef QCD_F64X12_K
#define QCD_F64X12_K 6
#endif
#ifndef QCD_F64X12_MINB
#define QCD_F64X12_MINB 1
#endif
#ifndef QCD_F64X18_B
#define QCD_F64X18_B 128
#endif
#ifndef QCD_F64X18_K
#define QCD_F64X18_K 3
#endif
#ifndef QCD_F64X18_MINB
#define QCD_F64X18_MINB 3
#endif
// Loop shape per precision and kind (measured at 32^4, see profiles/): ROLL = keep the direction / subgroup loops rolled,
// PRE = heatbath random part of trial 0 precomputed into shared memory.
#ifndef QCD_F32_ROLL_HB
#define QCD_F32_ROLL_HB true
#endif
#ifndef QCD_F32_ROLL_OR
#define QCD_F32_ROLL_OR false
#endif
#ifndef QCD_F32_PRE
#define QCD_F32_PRE true
#endif
#ifndef QCD_F64_ROLL_OR
#define QCD_F64_ROLL_OR false
#endif
#ifndef QCD_F64_ROLL_HB
#define QCD_F64_ROLL_HB true
#endif
#ifndef QCD_F64_PRE
#define QCD_F64_PRE false
#endif
template <typename R, int KIND> struct LoopCfg;
template <int KIND> struct LoopCfg<float, KIND> { static constexpr bool ROLL = (KIND == 0) ? QCD_F32_ROLL_HB : QCD_F32_ROLL_OR, PRE = QCD_F32_PRE; };
template <int KIND> struct LoopCfg<double, KIND> { static constexpr bool ROLL = (KIND == 0) ? QCD_F64_ROLL_HB : QCD_F64_ROLL_OR, PRE = QCD_F64_PRE; };
// Ring slots of the UNROLLED overrelaxation kernels (any K >= 2: the slot of a link is its sequence number mod K); the
// heatbath kernels, whose direction loop is rolled, need K | 6 and take the K above.
#ifndef QCD_F64X18_K_OR
#define QCD_F64X18_K_OR 4
#endif
template <typename R, bool COMP> struct RingKOr { static constexpr int K = -1; };          // -1: same as the heatbath kernel
template <> struct RingKOr<double, false> { static constexpr int K = QCD_F64X18_K_OR; };
template <int B_, int K_, int MINB_> struct RingShape { static constexpr int B = B_, K = K_, MINB = MINB_; };
template <typename R, bool COMP> struct RingCfg;
template <> struct RingCfg<float, true> : RingShape<QCD_F32X12_B, QCD_F32X12_K, QCD_F32X12_MINB> {};
template <> struct RingCfg<float, false> : RingShape<QCD_F32X18_B, QCD_F32X18_K, QCD_F32X18_MINB> {};
template <> struct RingCfg<double, true> : RingShape<QCD_F64X12_B, QCD_F64X12_K, QCD_F64X12_MINB> {};
template <> struct RingCfg<double, false> : RingShape<QCD_F64X18_B, QCD_F64X18_K, QCD_F64X18_MINB> {};

// Tile of B threads: e0 half-indices along x0, then powers of two along x1, x2, (x3); every extent must divide the lattice.
// QCD_TILE="s0,s1,s2" (log2 extents) overrides the default choice; QCD_TILE=off selects the linear mapping.
static inline TileMap choose_tile(const Geom& g, int B) {
  TileMap tm;
  memset(&tm, 0, sizeof(tm));
  if (g.D != 4 || (B & (B - 1))) return tm;
  int lb = 0;
  while ((1 << lb) < B) ++lb;
  auto pow2_part = [](int x) { int s = 0; while (!(x & 1)) { x >>= 1; ++s; } return s; };
  const int m[4] = {pow2_part(g.Lh0), pow2_part(g.L[1]), pow2_part(g.L[2]), pow2_part(g.L[3])};
  int s[4] = {0, 0, 0, 0};
  const char* env = getenv("QCD_TILE");
  if (env && !strcmp(env, "off")) return tm;
  if (env && sscanf(env, "%d,%d,%d", &s[0], &s[1], &s[2]) == 3) {
    s[3] = lb - s[0] - s[1] - s[2];
  } else {
    // default: 8 half-indices along x0 (one 128-byte line of 16-byte vectors), the rest spread over x1, x2, x3
    s[0] = m[0] < 3 ? m[0] : 3;
    int left = lb - s[0];
    for (int d = 1; left > 0; d = d % 3 + 1) {
      bool any = false;
      for (int k = 1; k < 4; ++k) any = any || s[k] < m[k];
      if (!any) break;
      if (s[d] < m[d]) { ++s[d]; --left; }
    }
    if (left > 0) { s[0] += left; }
  }
  for (int d = 0; d < 4; ++d) if (s[d] < 0 || s[d] > m[d]) return tm;      // does not tile this lattice: linear mapping
  if (s[0] + s[1] + s[2] + s[3] != lb) return tm;
  tm.on = 1; tm.s0 = s[0]; tm.s1 = s[1]; tm.s2 = s[2];
  tm.n0 = make_fastdiv((uint32_t)(g.Lh0 >> s[0])); tm.n1 = make_fastdiv((uint32_t)(g.L[1] >> s[1])); tm.n2 = make_fastdiv((uint32_t)(g.L[2] >> s[2]));
  return tm;
}

static inline bool tiled_enabled() {
  static int on = -1;
  if (on < 0) { const char* e = getenv("QCD_TILED"); on = (e && e[0] == '0') ? 0 : 1; }
  return on != 0;
}

template <typename R, int MU, bool COMP, int KIND, bool FIELD>
static cudaError_t su3_go_tiled(const Geom& g, void* links, const UpdateArgs& a, cudaStream_t st) {
  typedef PlaneTraits<R, (COMP ? 12 : 18)> T;
  typedef typename T::Vec Vec;
  typedef typename TileFor<MU>::TD TD;
  constexpr int K = TiledCfg<R, COMP, KIND>::K, MINB = TiledCfg<R, COMP, KIND>::MINB;
  constexpr bool ROLL = LoopCfg<R, KIND>::ROLL && (4 % K == 0);
  constexpr size_t smem = (size_t)(TD::res_slots(MU) + K * TD::B) * T::NP * sizeof(Vec);
  auto kern = su3_update_tiled_kernel<R, MU, COMP, KIND, FIELD, TD, K, MINB, ROLL>;
  static int attr_dev = -1;
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if (smem > 48 * 1024 && attr_dev != dev) {
    e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    attr_dev = dev;
  }
  UpdateArgs a2 = a;
  memset(&a2.tm, 0, sizeof(a2.tm));
  a2.tm.on = 1;
  a2.tm.n0 = make_fastdiv((uint32_t)(g.Lh0 / TD::T0)); a2.tm.n1 = make_fastdiv((uint32_t)(g.L[1] / TD::T1));
  a2.tm.n2 = make_fastdiv((uint32_t)(g.L[2] / TD::T2));
  return launch_pdl(kern, dim3(g.Vh / TD::B), dim3(TD::B), smem, st, g, (Vec*)links, a2);
}

template <typename R, int D, int MU, bool COMP, int KIND, bool FIELD>
static cudaError_t su3_go(const Geom& g, void* links, const UpdateArgs& a, cudaStream_t st) {
  typedef PlaneTraits<R, (COMP ? 12 : 18)> T;
  typedef typename T::Vec Vec;
  if constexpr (D == 4 && TiledCfg<R, COMP, KIND>::ON) {
    typedef typename TileFor<MU>::TD TD;
    if (tiled_enabled() && g.Lh0 % TD::T0 == 0 && g.L[1] % TD::T1 == 0 && g.L[2] % TD::T2 == 0 && g.L[3] % TD::T3 == 0)
      return su3_go_tiled<R, MU, COMP, KIND, FIELD>(g, links, a, st);
  }
  constexpr bool ROLL = LoopCfg<R, KIND>::ROLL, PRE = LoopCfg<R, KIND>::PRE;
  constexpr int B = RingCfg<R, COMP>::B, MINB = RingCfg<R, COMP>::MINB;
  constexpr int K = (KIND == 1 && !ROLL && RingKOr<R, COMP>::K >= 0) ? RingKOr<R, COMP>::K : RingCfg<R, COMP>::K;
  constexpr size_t smem = (size_t)K * T::NP * B * sizeof(Vec) + ((KIND == 0 && PRE) ? (size_t)15 * B * sizeof(R) : 0);
  auto kern = su3_update_kernel<R, D, MU, COMP, KIND, FIELD, B, K, MINB, ROLL, PRE>;
  static int attr_dev = -1;                  // opt in to > 48 KB of dynamic shared memory once per device
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if (smem > 48 * 1024 && attr_dev != dev) {
    e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    attr_dev = dev;
  }
  const unsigned grid = (g.Vh + B - 1) / B;
  UpdateArgs a2 = a;
  a2.tm = choose_tile(g, B);
  return launch_pdl(kern, dim3(grid), dim3(B), smem, st, g, (Vec*)links, a2);
}
template <typename R, int D, int MU, bool COMP>
static cudaError_t su3_sel_kind(const UpdateSel& s, const Geom& g, void* links, const UpdateArgs& a, cudaStream_t st) {
#ifdef QCD_TUNE_MINIMAL   // tuning builds: only what bench.py launches (D = 4, no field, x12 in float, x18 in double)
  if (D != 4 || s.field || COMP != std::is_same<R, float>::value) return cudaErrorInvalidValue;
  if constexpr (D == 4 && COMP == std::is_same<R, float>::value)
    return s.kind == 0 ? su3_go<R, D, MU, COMP, 0, false>(g, links, a, st) : su3_go<R, D, MU, COMP, 1, false>(g, links, a, st);
  return cudaErrorInvalidValue;
#else
  if (s.kind == 0) return s.field ? su3_go<R, D, MU, COMP, 0, true>(g, links, a, st) : su3_go<R, D, MU, COMP, 0, false>(g, links, a, st);
  return s.field ? su3_go<R, D, MU, COMP, 1, true>(g, links, a, st) : su3_go<R, D, MU, COMP, 1, false>(g, links, a, st);
#endif
}
template <typename R, int D, int MU>
static cudaError_t su3_sel_comp(const UpdateSel& s, const Geom& g, void* links, const UpdateArgs& a, cudaStream_t st) {
  return s.comp ? su3_sel_kind<R, D, MU, true>(s, g, links, a, st) : su3_sel_kind<R, D, MU, false>(s, g, links, a, st);
}
template <typename R, int D>
static cudaError_t su3_sel_mu(const UpdateSel& s, const Geom& g, void* links, const UpdateArgs& a, cudaStream_t st) {
  switch (a.mu) {
    case 0: return su3_sel_comp<R, D, 0>(s, g, links, a, st);
    case 1: return su3_sel_comp<R, D, 1>(s, g, links, a, st);
    case 2: if constexpr (D > 2) return su3_sel_comp<R, D, 2>(s, g, links, a, st); break;
    case 3: if constexpr (D > 3) return su3_sel_comp<R, D, 3>(s, g, links, a, st); break;
  }
  return cudaErrorInvalidValue;
}

}  // namespace qcd
