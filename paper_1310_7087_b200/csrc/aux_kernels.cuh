// aux_kernels.cuh -- everything on the path that is not the link update:
//   init (cold / hot; "hot" start), layout transforms for qcd_get/set_links (8(a)-1),
//   plaquette and Polyakov-loop reductions with fp64 accumulation (8(a)-8, 8(a)-9; "working sweep").
#pragma once
#include <type_traits>

#include "common.cuh"
#include "philox.cuh"
#include "sun_math.cuh"

namespace qcd {

// ------------------------------------------------------------------ generic link access (any group / storage)
// LinkIO<NC, R, COMP>: load to / store from a full N x N complex matrix in registers, Cx<R> m[NC][NC]
template <int NC, typename R, bool COMP> struct LinkIO;

template <typename R, bool COMP> struct LinkIO<3, R, COMP> {
  static constexpr int NREAL = COMP ? 12 : 18;
  typedef PlaneTraits<R, NREAL> T;
  typedef typename T::Vec Vec;
  template <bool NCLOAD>
  static __device__ __forceinline__ void load(Cx<R> (&m)[3][3], const Vec* __restrict__ links, const Geom& g, size_t base, uint32_t h) {
    R r[NREAL];
    load_reals<R, NREAL, NCLOAD>(links, g, base, h, r);
    M3<R> u;
    m3_from_reals<R, NREAL>(u, r);
    if (COMP) m3_complete_row2(u);
#pragma unroll
    for (int i = 0; i < 3; ++i)
#pragma unroll
      for (int j = 0; j < 3; ++j) m[i][j] = u.e[i][j];
  }
  static __device__ __forceinline__ void store(const Cx<R> (&m)[3][3], Vec* links, const Geom& g, size_t base, uint32_t h) {
    R r[NREAL];
#pragma unroll
    for (int e = 0; e < NREAL / 2; ++e) { r[2 * e] = m[e / 3][e % 3].re; r[2 * e + 1] = m[e / 3][e % 3].im; }
    store_reals<R, NREAL>(links, g, base, h, r);
  }
};

template <typename R, bool COMP> struct LinkIO<2, R, COMP> {
  static constexpr int NREAL = 4;
  typedef PlaneTraits<R, 4> T;
  typedef typename T::Vec Vec;
  template <bool NCLOAD>
  static __device__ __forceinline__ void load(Cx<R> (&m)[2][2], const Vec* __restrict__ links, const Geom& g, size_t base, uint32_t h) {
    R r[4];
    load_reals<R, 4, NCLOAD>(links, g, base, h, r);
    m[0][0] = cx<R>(r[0], r[3]); m[0][1] = cx<R>(r[2], r[1]);
    m[1][0] = cx<R>(-r[2], r[1]); m[1][1] = cx<R>(r[0], -r[3]);
  }
  static __device__ __forceinline__ void store(const Cx<R> (&m)[2][2], Vec* links, const Geom& g, size_t base, uint32_t h) {
    R r[4] = {m[0][0].re, m[0][1].im, m[0][1].re, m[0][0].im};
    store_reals<R, 4>(links, g, base, h, r);
  }
};

template <int NC, typename R> __device__ __forceinline__ void mm_nn(Cx<R> (&c)[NC][NC], const Cx<R> (&a)[NC][NC], const Cx<R> (&b)[NC][NC]) {
#pragma unroll
  for (int i = 0; i < NC; ++i)
#pragma unroll
    for (int j = 0; j < NC; ++j) {
      Cx<R> s = cx<R>(0, 0);
#pragma unroll
      for (int k = 0; k < NC; ++k) cmad(s, a[i][k], b[k][j]);
      c[i][j] = s;
    }
}

// ------------------------------------------------------------------ init
// hot start (reading R9): Gaussians by Box-Muller on consecutive 32-bit-mode uniforms of Philox domain 1, always
// in double; SU(2): 4 Gaussians -> unit quaternion; SU(3): 12 Gaussians -> rows 0,1 -> Gram-Schmidt.
__device__ __forceinline__ void box_muller4(const Philox4& w, double* z) {
  const double ua = uniform64(w.x), ub = uniform64(w.y), uc = uniform64(w.z), ud = uniform64(w.w);
  double s, c;
  double rad = sqrt(-2.0 * log(ua));
  sincospi(2.0 * ub, &s, &c);
  z[0] = rad * c; z[1] = rad * s;
  rad = sqrt(-2.0 * log(uc));
  sincospi(2.0 * ud, &s, &c);
  z[2] = rad * c; z[3] = rad * s;
}

template <int NC, int D, typename R, bool COMP>
__global__ void __launch_bounds__(128) init_kernel(Geom g, typename LinkIO<NC, R, COMP>::Vec* links, int hot, uint32_t key0, uint32_t key1) {
  typedef LinkIO<NC, R, COMP> IO;
  const uint32_t hl = blockIdx.x * blockDim.x + threadIdx.x;
  const int p = blockIdx.y;
  if (hl >= g.Vh_int) return;                              // a slab initialises its own sites; the halo layers are exchanged
  uint32_t h;
  const SiteCoord sc = decode_launch(g, hl, p, h);
  const uint32_t lex = lex_global(g, sc);
#pragma unroll
  for (int mu = 0; mu < D; ++mu) {
    Cx<R> m[NC][NC];
    if (!hot) {
#pragma unroll
      for (int i = 0; i < NC; ++i)
#pragma unroll
        for (int j = 0; j < NC; ++j) m[i][j] = cx<R>(i == j ? R(1) : R(0), R(0));
    } else {
      const uint32_t c2 = philox_c2(mu, p, 0, 0, 1);
      if (NC == 2) {
        double z[4];
        box_muller4(philox4x32_10(lex, 0u, c2, 0u, key0, key1), z);
        const double n = 1.0 / sqrt(z[0] * z[0] + z[1] * z[1] + z[2] * z[2] + z[3] * z[3]);
        const double a0 = z[0] * n, a1 = z[1] * n, a2 = z[2] * n, a3 = z[3] * n;
        m[0][0] = cx<R>((R)a0, (R)a3); m[0][1] = cx<R>((R)a2, (R)a1);
        m[1][0] = cx<R>((R)-a2, (R)a1); m[1][1] = cx<R>((R)a0, (R)-a3);
      } else {
        double z[12];
#pragma unroll
        for (int d = 0; d < 3; ++d) box_muller4(philox4x32_10(lex, 0u, c2, (uint32_t)d, key0, key1), z + 4 * d);
        M3<double> u;
#pragma unroll
        for (int c = 0; c < 3; ++c) { u.e[0][c] = cx<double>(z[2 * c], z[2 * c + 1]); u.e[1][c] = cx<double>(z[6 + 2 * c], z[6 + 2 * c + 1]); }
        // Gram-Schmidt with true divisions (matches the oracle's order of operations to the last bits)
        double n0 = 0.0;
#pragma unroll
        for (int c = 0; c < 3; ++c) n0 += u.e[0][c].re * u.e[0][c].re + u.e[0][c].im * u.e[0][c].im;
        n0 = sqrt(n0);
#pragma unroll
        for (int c = 0; c < 3; ++c) { u.e[0][c].re /= n0; u.e[0][c].im /= n0; }
        Cx<double> dd = cx<double>(0.0, 0.0);
#pragma unroll
        for (int c = 0; c < 3; ++c) cmad_conja(dd, u.e[0][c], u.e[1][c]);
#pragma unroll
        for (int c = 0; c < 3; ++c) {
          u.e[1][c].re -= dd.re * u.e[0][c].re - dd.im * u.e[0][c].im;
          u.e[1][c].im -= dd.re * u.e[0][c].im + dd.im * u.e[0][c].re;
        }
        double n1 = 0.0;
#pragma unroll
        for (int c = 0; c < 3; ++c) n1 += u.e[1][c].re * u.e[1][c].re + u.e[1][c].im * u.e[1][c].im;
        n1 = sqrt(n1);
#pragma unroll
        for (int c = 0; c < 3; ++c) { u.e[1][c].re /= n1; u.e[1][c].im /= n1; }
        m3_complete_row2(u);
#pragma unroll
        for (int i = 0; i < NC; ++i)
#pragma unroll
          for (int j = 0; j < NC; ++j) m[i][j] = cx<R>((R)u.e[i % 3][j % 3].re, (R)u.e[i % 3][j % 3].im);
      }
    }
    IO::store(m, links, g, array_base<IO::T::NP>(g, D, p, mu), h);
  }
}

// ------------------------------------------------------------------ canonical <-> internal layout
// canonical: [lex][mu][row][col][re,im] of R, full N x N.  One thread per site, all directions.
// sites per CTA of layout_kernel: one CTA's block of the canonical array (BL * D * N*N complex numbers) fits 48 KB
template <typename R> struct LayoutShape { static constexpr int BL = sizeof(R) == 4 ? 128 : 64; };

// NRC = rows of a link in the canonical array: NC, or 2 for the compressed exchange format of 12-real SU(3) lattices
// (QCD_OPT_EXCHANGE_ROWS01: rows 0,1 only, [lex][mu][2][3][re,im]).
template <int NC, int D, typename R, bool COMP, bool TO_INTERNAL, int NRC>
__global__ void __launch_bounds__(LayoutShape<R>::BL) layout_kernel(Geom g, typename LinkIO<NC, R, COMP>::Vec* links, R* canon,
                                                                    uint32_t lex_begin, uint32_t lex_end) {
  // sites [lex_begin, lex_end); `canon` is the canonical address of site lex_begin (a chunk of a host transfer, or the
  // whole array when lex_begin = 0, lex_end = V)
  // One thread per site in LEX order (both parities in one CTA).  A CTA owns BL consecutive sites, i.e. one contiguous
  // block of BL * D * N*N complex numbers of the canonical array, and moves it through shared memory: the global side is
  // a flat, fully coalesced copy (consecutive threads, consecutive complex numbers), the per-site side (a thread's D
  // links, 36 complex numbers apart from its neighbour's) stays in shared memory (row pitch NCX + 1 against bank
  // conflicts).  The internal side is one 16-byte vector per thread and plane, 16 consecutive half-indices per parity
  // and half-warp.
  typedef LinkIO<NC, R, COMP> IO;
  typedef typename std::conditional<sizeof(R) == 4, float2, double2>::type C2;   // one complex number of the canonical array
  static_assert(NRC == NC || (NRC == 2 && NC == 3 && COMP), "rows 0,1 only for 12-real SU(3) links");
  constexpr int BL = LayoutShape<R>::BL, NCX = D * NRC * NC, PITCH = NCX + 1;
  __shared__ C2 buf[BL * PITCH];
  const uint32_t lex0 = lex_begin + blockIdx.x * BL, t = threadIdx.x;
  const uint32_t nsite = (lex_end - lex0 < (uint32_t)BL) ? lex_end - lex0 : (uint32_t)BL;
  const uint32_t nel = nsite * NCX;
  C2* gc = reinterpret_cast<C2*>(canon) + (size_t)(lex0 - lex_begin) * NCX;
  if (TO_INTERNAL) {
    for (uint32_t i = t; i < nel; i += BL) buf[(i / NCX) * PITCH + (i % NCX)] = gc[i];
    __syncthreads();
  }
  if (t < nsite) {
    // lex runs over the lattice's own sites in lex order of their extents Li (a slab: its interior block)
    const uint32_t lex = lex0 + t, hl = lex >> 1;
    const uint32_t row = fd_div(hl, g.iLh0);
    const uint32_t r2 = fd_div(row, g.iL1);
    const uint32_t x1 = row - r2 * (uint32_t)g.Li[1];
    const uint32_t r3 = fd_div(r2, g.iL2);
    const uint32_t x2 = r2 - r3 * (uint32_t)g.Li[2], x3 = r3;
    const uint32_t h = ((x3 * (uint32_t)g.L[2] + x2) * (uint32_t)g.L[1] + x1) * (uint32_t)g.Lh0 + (hl - row * (uint32_t)g.Lh0);
    const int p = (int)(((lex & 1u) + x1 + x2 + x3) & 1u);         // x0 & 1 = lex & 1 (L0 even)
#pragma unroll
    for (int mu = 0; mu < D; ++mu) {
      C2* c = buf + t * PITCH + mu * NRC * NC;
      Cx<R> m[NC][NC];
      const size_t base = array_base<IO::T::NP>(g, D, p, mu);
      if (TO_INTERNAL) {
#pragma unroll
        for (int i = 0; i < NC; ++i)
#pragma unroll
          for (int j = 0; j < NC; ++j) {
            if (i < NRC) { const C2 v = c[i * NC + j]; m[i][j] = cx<R>(v.x, v.y); }
            else m[i][j] = cx<R>(R(0), R(0));                      // row 2 is not stored by 12-real links
          }
        IO::store(m, links, g, base, h);
      } else {
        IO::template load<false>(m, links, g, base, h);
#pragma unroll
        for (int i = 0; i < NRC; ++i)
#pragma unroll
          for (int j = 0; j < NC; ++j) { C2 v; v.x = m[i][j].re; v.y = m[i][j].im; c[i * NC + j] = v; }
      }
    }
  }
  if (!TO_INTERNAL) {
    __syncthreads();
    for (uint32_t i = t; i < nel; i += BL) gc[i] = buf[(i / NCX) * PITCH + (i % NCX)];
  }
}

// ------------------------------------------------------------------ halo layers of a slab
// Copy one layer (coordinate `layer` of the split direction sd) of the (parity, mu) link array: the boundary exchange of a
// lattice divided into parts ("exchanging values of boundary sites").  One thread per half-index of the layer,
// all NP planes.  MODE 0: lattice layer -> contiguous buffer [plane][site of the layer] (pack, for a message to another
// process); 1: buffer -> lattice layer (unpack); 2: layer of one part -> layer of another part directly (same process; the
// destination may be peer memory of another GPU reached over NVLink).  The half-index of a site does not depend on its
// parity, and part extents are even, so source and destination enumerate the same sites.
template <typename Vec, int NP, int MODE>
__global__ void __launch_bounds__(128) halo_kernel(Geom gs, const Vec* __restrict__ src, int src_layer, Geom gd, Vec* __restrict__ dst, int dst_layer,
                                                   int parity, int mu, int D, uint32_t count) {
  const uint32_t idx = blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= count) return;
  const Geom& g = (MODE == 1) ? gd : gs;                  // the geometry that enumerates the layer (both agree off the split direction)
  const int sd = g.sd;
  uint32_t rest = idx / (uint32_t)g.Lh0;
  const uint32_t j = idx - rest * (uint32_t)g.Lh0;
  uint32_t x[4] = {0, 0, 0, 0};
#pragma unroll
  for (int d = 1; d < 4; ++d) {
    if (d == sd) continue;
    const uint32_t q = rest / (uint32_t)g.L[d];
    x[d] = rest - q * (uint32_t)g.L[d];
    rest = q;
  }
  auto half_index = [&](const Geom& gg, int layer) -> uint32_t {
    uint32_t y[4] = {0, x[1], x[2], x[3]};
    y[sd] = (uint32_t)layer;
    return ((y[3] * (uint32_t)gg.L[2] + y[2]) * (uint32_t)gg.L[1] + y[1]) * (uint32_t)gg.Lh0 + j;
  };
  const Vec* ps = (MODE == 1) ? src + idx : src + array_base<NP>(gs, D, parity, mu) + blk_off<NP>(half_index(gs, src_layer));
  Vec* pd = (MODE == 0) ? dst + idx : dst + array_base<NP>(gd, D, parity, mu) + blk_off<NP>(half_index(gd, dst_layer));
  const size_t ss = (MODE == 1) ? (size_t)count : (size_t)PLANE_STRIDE, ds = (MODE == 0) ? (size_t)count : (size_t)PLANE_STRIDE;
#pragma unroll
  for (int k = 0; k < NP; ++k) pd[k * ds] = ps[k * ss];
}

// Both boundary layers of one part in ONE launch (the single-process driver qcd_split_*): blockIdx.y = 0 copies the part's
// first own layer into the previous part's "next" copy, blockIdx.y = 1 its last own layer into the next part's "previous"
// copy.  Same addressing as halo_kernel<., ., 2>.
template <typename Vec> struct HaloTarget { Geom g; Vec* mem; int src_layer, dst_layer; };
template <typename Vec, int NP>
__global__ void __launch_bounds__(128) halo_pair_kernel(Geom gs, const Vec* __restrict__ src, HaloTarget<Vec> t0, HaloTarget<Vec> t1, int parity, int mu,
                                                        int D, uint32_t count) {
  // launched with programmatic stream serialization behind the part's update kernel: resident while that kernel drains,
  // reads its output only after the wait; the trigger comes after the wait (as in the update kernels: at most one earlier
  // kernel of the chain is in flight)
  pdl_wait();
  pdl_trigger();
  const uint32_t idx = blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= count) return;
  const HaloTarget<Vec>& t = blockIdx.y ? t1 : t0;
  const int sd = gs.sd;
  uint32_t rest = idx / (uint32_t)gs.Lh0;
  const uint32_t j = idx - rest * (uint32_t)gs.Lh0;
  uint32_t x[4] = {0, 0, 0, 0};
#pragma unroll
  for (int d = 1; d < 4; ++d) {
    if (d == sd) continue;
    const uint32_t q = rest / (uint32_t)gs.L[d];
    x[d] = rest - q * (uint32_t)gs.L[d];
    rest = q;
  }
  auto half_index = [&](const Geom& gg, int layer) -> uint32_t {
    uint32_t y[4] = {0, x[1], x[2], x[3]};
    y[sd] = (uint32_t)layer;
    return ((y[3] * (uint32_t)gg.L[2] + y[2]) * (uint32_t)gg.L[1] + y[1]) * (uint32_t)gg.Lh0 + j;
  };
  const Vec* ps = src + array_base<NP>(gs, D, parity, mu) + blk_off<NP>(half_index(gs, t.src_layer));
  Vec* pd = t.mem + array_base<NP>(t.g, D, parity, mu) + blk_off<NP>(half_index(t.g, t.dst_layer));
#pragma unroll
  for (int k = 0; k < NP; ++k) pd[k * PLANE_STRIDE] = ps[k * PLANE_STRIDE];
}

// ------------------------------------------------------------------ reductions
// block-wide sums of NV doubles per thread: warp shuffle, then shared memory, fixed order => deterministic
template <int NV, int BLOCK>
__device__ __forceinline__ void block_reduce_store(double (&v)[NV], double* out /* [NV][gridDim.x*gridDim.y] */, uint32_t nblocks, uint32_t bid) {
  __shared__ double sm[NV][BLOCK / 32];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
  for (int k = 0; k < NV; ++k) {
    double x = v[k];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) x += __shfl_down_sync(0xffffffffu, x, o);
    if (lane == 0) sm[k][warp] = x;
  }
  __syncthreads();
  if (threadIdx.x < NV) {
    double s = 0.0;
#pragma unroll
    for (int w = 0; w < BLOCK / 32; ++w) s += sm[threadIdx.x][w];
    out[(size_t)threadIdx.x * nblocks + bid] = s;
  }
}

// second stage: one block per quantity, fixed-order tree over the per-block partials
__global__ void __launch_bounds__(256) final_reduce_kernel(const double* partials, uint32_t nblocks, double* out, double scale) {
  __shared__ double sm[256];
  const double* p = partials + (size_t)blockIdx.x * nblocks;
  double s = 0.0;
  for (uint32_t i = threadIdx.x; i < nblocks; i += 256) s += p[i];
  sm[threadIdx.x] = s;
  __syncthreads();
  for (int o = 128; o > 0; o >>= 1) {
    if ((int)threadIdx.x < o) sm[threadIdx.x] += sm[threadIdx.x + o];
    __syncthreads();
  }
  if (threadIdx.x == 0) out[blockIdx.x] = sm[0] * scale;
}

struct MeasureField {
  int enabled, mu, nu;
  double c[3], s[3];
  // plaquette kernel, D = 4 with L0/2 a multiple of 8: a CTA covers a box of 8 half-indices x 2 x 2 x 2 sites on BOTH
  // parities (128 threads) instead of 128 consecutive half-indices of one parity, so that the link U_nu(y) a site loads as
  // its own and the three sites y - mu load as a neighbour meet in the same L1 (the kernel uses no shared memory, so the
  // L1 is ~200 KB).  n0, n1, n2 = boxes per direction 0, 1, 2.
  int boxed;
  FastDiv n0, n1, n2;
};

// plaquette: one thread per site; the D own links stay in registers, each plane loads its two neighbours
template <int NC, int D, typename R, bool COMP>
__global__ void __launch_bounds__(128) plaquette_kernel(Geom g, const typename LinkIO<NC, R, COMP>::Vec* __restrict__ links, MeasureField f,
                                                        double* partials) {
  typedef LinkIO<NC, R, COMP> IO;
  constexpr int NPL = D * (D - 1) / 2;
  uint32_t h;
  int p;
  SiteCoord sc;
  bool active;
  if (D == 4 && f.boxed) {
    const uint32_t t = threadIdx.x;
    uint32_t b = blockIdx.x;
    uint32_t qq = fd_div(b, f.n0); const uint32_t b0 = b - qq * f.n0.d; b = qq;
    qq = fd_div(b, f.n1); const uint32_t b1 = b - qq * f.n1.d; b = qq;
    qq = fd_div(b, f.n2); const uint32_t b2 = b - qq * f.n2.d; const uint32_t b3 = qq;
    p = (int)(t >> 6);
    sc.j = (int)(b0 * 8u + (t & 7u));
    sc.x1 = (int)(b1 * 2u + ((t >> 3) & 1u));
    sc.x2 = (int)(b2 * 2u + ((t >> 4) & 1u));
    sc.x3 = (int)(b3 * 2u + ((t >> 5) & 1u));
    sc.s = (p + sc.x1 + sc.x2 + sc.x3) & 1;
    h = (uint32_t)(((sc.x3 * g.L[2] + sc.x2) * g.L[1] + sc.x1) * g.Lh0 + sc.j);
    active = true;
  } else {
    const uint32_t hl = blockIdx.x * blockDim.x + threadIdx.x;
    p = blockIdx.y;
    active = hl < g.Vh_int;
    h = 0;
    if (active) sc = decode_launch(g, hl, p, h);
  }
  const int q = 1 - p;
  double acc[NPL];
#pragma unroll
  for (int k = 0; k < NPL; ++k) acc[k] = 0.0;
  // One plane at a time, loop NOT unrolled: the four links of a plane are loaded when the plane is reached, so a thread
  // holds one plane's worth of registers (fp64 x18 needed 254 registers with the own links kept across planes: 2 CTAs per
  // SM, and the kernel is bound by load latency).  The own links are re-read per plane; they hit in L1 (boxed mapping).
  if (active) {
    int fwd[D];
#pragma unroll
    for (int d = 0; d < D; ++d) { int bb; nbr_offsets(g, sc, d, fwd[d], bb); }
#pragma unroll 1
    for (int pl = 0; pl < NPL; ++pl) {
      // plane index -> (mu, nu), mu < nu, in the order (0,1),(0,2),..,(D-2,D-1)
      int mu = 0, nu = 1;
      {
        int k = pl;
#pragma unroll
        for (int m = 0; m < D - 1; ++m) { const int cnt = D - 1 - m; if (k >= cnt && mu == m) { k -= cnt; mu = m + 1; } }
        nu = mu + 1 + k;
      }
      int fmu = fwd[0], fnu = fwd[0];
#pragma unroll
      for (int d = 1; d < D; ++d) { if (mu == d) fmu = fwd[d]; if (nu == d) fnu = fwd[d]; }
      const bool dressed = f.enabled && f.mu == mu && f.nu == nu;
      R tr;
      if constexpr (NC == 3 && COMP) {
        // 12-real links: rows 0,1 of M = U_mu(x) U_nu(x+mu) and N = U_nu(x) U_mu(x+nu) only.  With
        // G_ab = sum_j M_aj conj(N_bj) (a, b in {0,1}) the diagonal of M N^+ is (G_00, G_11, conj(G_00 G_11 - G_01 G_10)):
        // third rows of SU(3) matrices are conj(row0 x row1), and (a x b).conj(c x d) = (a.conj c)(b.conj d) - (a.conj d)(b.conj c).
        // The own links need no third row at all; the neighbours do (they are summed over in the products).
        typedef PlaneTraits<R, 12> T12;
        M3<R> u, w, M, N;
        R r[12];
        load_reals<R, 12, true>(links, g, array_base<T12::NP>(g, D, q, nu), h + fmu, r);          // U_nu(x+mu)
        m3_from_reals<R, 12>(w, r);
        m3_complete_row2(w);
        load_reals<R, 12, true>(links, g, array_base<T12::NP>(g, D, p, mu), h, r);                // U_mu(x)
        m3_from_reals<R, 12>(u, r);
        m3_zero(M);
        m3_mad_nn<R, 2>(M, u, w);
        load_reals<R, 12, true>(links, g, array_base<T12::NP>(g, D, q, mu), h + fnu, r);          // U_mu(x+nu)
        m3_from_reals<R, 12>(w, r);
        m3_complete_row2(w);
        load_reals<R, 12, true>(links, g, array_base<T12::NP>(g, D, p, nu), h, r);                // U_nu(x)
        m3_from_reals<R, 12>(u, r);
        m3_zero(N);
        m3_mad_nn<R, 2>(N, u, w);
        Cx<R> G00 = cx<R>(0, 0), G01 = cx<R>(0, 0), G10 = cx<R>(0, 0), G11 = cx<R>(0, 0);
        cdot3<CD_ND>(G00, M.e[0][0], M.e[0][1], M.e[0][2], N.e[0][0], N.e[0][1], N.e[0][2]);
        cdot3<CD_ND>(G01, M.e[0][0], M.e[0][1], M.e[0][2], N.e[1][0], N.e[1][1], N.e[1][2]);
        cdot3<CD_ND>(G10, M.e[1][0], M.e[1][1], M.e[1][2], N.e[0][0], N.e[0][1], N.e[0][2]);
        cdot3<CD_ND>(G11, M.e[1][0], M.e[1][1], M.e[1][2], N.e[1][0], N.e[1][1], N.e[1][2]);
        const Cx<R> dd = cmul(G00, G11), od = cmul(G01, G10);
        const Cx<R> D2 = cx<R>(dd.re - od.re, -(dd.im - od.im));
        tr = dressed ? (G00.re * (R)f.c[0] - G00.im * (R)f.s[0]) + (G11.re * (R)f.c[1] - G11.im * (R)f.s[1]) +
                           (D2.re * (R)f.c[2] - D2.im * (R)f.s[2])
                     : G00.re + G11.re + D2.re;
      } else {
        Cx<R> u[NC][NC], w[NC][NC], ab[NC][NC], dc[NC][NC];
        IO::template load<true>(u, links, g, array_base<IO::T::NP>(g, D, p, mu), h);             // U_mu(x)
        IO::template load<true>(w, links, g, array_base<IO::T::NP>(g, D, q, nu), h + fmu);       // U_nu(x+mu)
        mm_nn<NC, R>(ab, u, w);
        IO::template load<true>(u, links, g, array_base<IO::T::NP>(g, D, p, nu), h);             // U_nu(x)
        IO::template load<true>(w, links, g, array_base<IO::T::NP>(g, D, q, mu), h + fnu);       // U_mu(x+nu)
        mm_nn<NC, R>(dc, u, w);
        // Re Tr [F] ab dc^+ = sum_i Re( ph_i * sum_j ab_ij conj(dc_ij) )
        tr = R(0);
#pragma unroll
        for (int i = 0; i < NC; ++i) {
          Cx<R> d = cx<R>(0, 0);
#pragma unroll
          for (int j = 0; j < NC; ++j) cmad_conj(d, ab[i][j], dc[i][j]);
          tr += dressed ? (d.re * (R)f.c[i] - d.im * (R)f.s[i]) : d.re;
        }
      }
#pragma unroll
      for (int k = 0; k < NPL; ++k) acc[k] += (k == pl) ? (double)tr : 0.0;
    }
  }
  block_reduce_store<NPL, 128>(acc, partials, gridDim.x * gridDim.y, blockIdx.y * gridDim.x + blockIdx.x);
}

// Polyakov loop: ordered product over t of U_{D-1}.  SEG lanes per spatial site: lane g multiplies the links of the time
// segment [g Lt/SEG, (g+1) Lt/SEG) -- the kernel is bound by the latency of its dependent loads, and the segments' loads are
// independent -- then the SEG partial products are combined in order by shuffles (P0 P1)(P2 P3).  SEG = 1: one thread per
// spatial site walks all of Lt.  SEG must divide Lt and 32.
template <int NC, typename R> __device__ __forceinline__ void mat_shfl_down(Cx<R> (&dst)[NC][NC], const Cx<R> (&src)[NC][NC], int delta) {
#pragma unroll
  for (int i = 0; i < NC; ++i)
#pragma unroll
    for (int j = 0; j < NC; ++j) {
      dst[i][j].re = __shfl_down_sync(0xffffffffu, src[i][j].re, delta);
      dst[i][j].im = __shfl_down_sync(0xffffffffu, src[i][j].im, delta);
    }
}
template <int NC, int D, typename R, bool COMP, int SEG>
__global__ void __launch_bounds__(128) polyakov_kernel(Geom g, const typename LinkIO<NC, R, COMP>::Vec* __restrict__ links, double* partials) {
  typedef LinkIO<NC, R, COMP> IO;
  const uint32_t Lt = (uint32_t)g.L[D - 1];
  const uint32_t Vs = g.V / Lt;                            // spatial sites of the local lattice (time stride)
  const uint32_t Vs_int = 2u * g.Vh_int / Lt;              // ... of which the lattice's own (a slab is split along a spatial direction)
  const uint32_t tid = blockIdx.x * blockDim.x + threadIdx.x;
  const uint32_t seg = tid % SEG;
  const uint32_t s_raw = tid / SEG;
  const bool live = s_raw < Vs_int;
  const uint32_t s = live ? s_raw : Vs_int - 1;            // surplus lanes shadow the last site (whole warps do the shuffles)
  double acc[2] = {0.0, 0.0};
  {
    // spatial coordinates of the t = 0 site with interior lex index s; its parity is (x0 + x1 + x2) & 1 with x0 & 1 = s & 1
    // (L0 even); x1, x2 decode to 0 when they are not spatial directions (D < 4), because s < Vs_int.
    const uint32_t hl = s >> 1;
    const uint32_t row = fd_div(hl, g.iLh0);
    const uint32_t r2 = fd_div(row, g.iL1);
    const int x1 = (int)(row - r2 * (uint32_t)g.Li[1]);
    const int x2 = (D == 4) ? (int)r2 : 0;
    const uint32_t hs = (uint32_t)((x2 * g.L[1] + x1) * g.Lh0) + (hl - row * (uint32_t)g.Lh0);
    const int par0 = ((int)(s & 1u) + x1 + x2) & 1;
    Cx<R> P[NC][NC];
#pragma unroll
    for (int i = 0; i < NC; ++i)
#pragma unroll
      for (int j = 0; j < NC; ++j) P[i][j] = cx<R>(i == j ? R(1) : R(0), R(0));
    const uint32_t nt = Lt / SEG, t0 = seg * nt;
    for (uint32_t t = t0; t < t0 + nt; ++t) {
      const int p = (par0 + (int)t) & 1;
      const uint32_t h = hs + t * (Vs >> 1);
      Cx<R> u[NC][NC], n[NC][NC];
      IO::template load<true>(u, links, g, array_base<IO::T::NP>(g, D, p, D - 1), h);
      mm_nn<NC, R>(n, P, u);
#pragma unroll
      for (int i = 0; i < NC; ++i)
#pragma unroll
        for (int j = 0; j < NC; ++j) P[i][j] = n[i][j];
    }
    // combine the segments in time order: lanes seg, seg + delta hold consecutive runs of segments
#pragma unroll
    for (int delta = 1; delta < SEG; delta <<= 1) {
      Cx<R> o[NC][NC], n[NC][NC];
      mat_shfl_down<NC, R>(o, P, delta);
      mm_nn<NC, R>(n, P, o);
#pragma unroll
      for (int i = 0; i < NC; ++i)
#pragma unroll
        for (int j = 0; j < NC; ++j) P[i][j] = n[i][j];
    }
    if (live && seg == 0) {
#pragma unroll
      for (int i = 0; i < NC; ++i) { acc[0] += (double)P[i][i].re; acc[1] += (double)P[i][i].im; }
    }
  }
  block_reduce_store<2, 128>(acc, partials, gridDim.x, blockIdx.x);
}

}  // namespace qcd
