// common.cuh -- geometry, link layout and small device helpers shared by all kernels of libqcd_b200.
//
// Link layout in HBM ("fastest index - number of lattice site ... next
// index - direction ... group matrices are represented as structures of 4-vectors"):
//   vec-plane SoA   links[parity p][direction mu][h / 8][plane k][h % 8]     (blocks of 8 half-indices, see blk_off)
// where a site x of parity p = (sum x_d) & 1 has h = lex(x) >> 1, lex = x0 + L0*(x1 + L1*(x2 + L2*x3)), and the
// NREAL stored reals of one link (row-major, re then im) are cut into NP = NREAL/VW planes of VW-wide vectors:
//   SU(3) fp32 x12 : 3 x float4      SU(3) fp32 x18 : 9 x float2
//   SU(3) fp64 x18 : 9 x double2     SU(3) fp64 x12 : 6 x double2
//   SU(2) fp32 q4  : 1 x float4      SU(2) fp64 q4  : 2 x double2        (quaternion a0,a1,a2,a3)
// Every plane holds Vh_pad = roundup(V/2, 32) vectors, so every plane starts 128-byte aligned.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "hb_math.cuh"

namespace qcd {

// ------------------------------------------------------------------ division by run-time constants
struct FastDiv {
  uint32_t d, m, s;
};
inline FastDiv make_fastdiv(uint32_t d) {
  FastDiv f; f.d = d; f.s = 0;
  while ((1u << f.s) < d) ++f.s;
  f.m = (uint32_t)((((uint64_t)1 << 32) * (((uint64_t)1 << f.s) - d)) / d + 1);
  return f;
}
__device__ __forceinline__ uint32_t fd_div(uint32_t n, const FastDiv& f) { return (__umulhi(n, f.m) + n) >> f.s; }  // n < 2^31

// ------------------------------------------------------------------ geometry (kernel parameter, constant bank)
struct Geom {
  int D;
  int L[4];          // extents, 1 beyond D
  int Lh0;           // L[0] / 2
  int stride[4];     // half-index stride of a +1 step in direction d >= 1: Lh0, Lh0*L1, Lh0*L1*L2 ; stride[0] unused
  uint32_t Vh;       // V / 2
  uint32_t Vh_pad;   // plane length in vectors
  uint32_t V;
  FastDiv dLh0, dL1, dL2;
  // ---- slab of a larger lattice ("dividing lattice into parts ... exchanging values of
  // boundary sites").  The local lattice is a part split off along direction sd (sd = -1: not a slab).  Its layers
  // [0, n_int) of direction sd are the part's own sites (global coordinate off + layer); layer n_int holds a copy of the next
  // part's first layer and layer n_int + 1 a copy of the previous part's last layer, so the local periodic wrap of the
  // extent L[sd] = n_int + 2 lands on the right neighbours.  Kernels visit the interior only: the launch index runs over
  // the extents Li[d] (= L[d], except Li[sd] = n_int).  Part extents and offsets are even, so local and global parity
  // coincide.  The Philox counter takes the GLOBAL lex index: lex_g = x0 + x1 lexS[1] + x2 lexS[2] + x3 lexS[3] + lex0.
  int sd;
  int Li[4];
  uint32_t Vh_int;   // interior sites of one parity
  uint32_t lexS[4], lex0;
  FastDiv iLh0, iL1, iL2;     // launch-index decoding (interior extents); equal to dLh0, dL1, dL2 when sd < 0
};

struct SiteCoord {
  int j, x1, x2, x3, s;  // x0 = 2*j + s
};

__device__ __forceinline__ SiteCoord decode_site(const Geom& g, uint32_t h, int parity) {
  SiteCoord c;
  uint32_t row = fd_div(h, g.dLh0);
  c.j = (int)(h - row * (uint32_t)g.Lh0);
  uint32_t r2 = fd_div(row, g.dL1);
  c.x1 = (int)(row - r2 * (uint32_t)g.L[1]);
  uint32_t r3 = fd_div(r2, g.dL2);
  c.x2 = (int)(r2 - r3 * (uint32_t)g.L[2]);
  c.x3 = (int)r3;
  c.s = (parity + c.x1 + c.x2 + c.x3) & 1;
  return c;
}

// launch index hl in [0, Vh_int) of one parity -> site coordinates and local half-index h (h = hl unless the lattice is a slab)
__device__ __forceinline__ SiteCoord decode_launch(const Geom& g, uint32_t hl, int parity, uint32_t& h) {
  if (g.sd < 0) { h = hl; return decode_site(g, hl, parity); }
  SiteCoord c;
  uint32_t row = fd_div(hl, g.iLh0);
  c.j = (int)(hl - row * (uint32_t)g.Lh0);
  uint32_t r2 = fd_div(row, g.iL1);
  c.x1 = (int)(row - r2 * (uint32_t)g.Li[1]);
  uint32_t r3 = fd_div(r2, g.iL2);
  c.x2 = (int)(r2 - r3 * (uint32_t)g.Li[2]);
  c.x3 = (int)r3;
  c.s = (parity + c.x1 + c.x2 + c.x3) & 1;
  h = (uint32_t)(((c.x3 * g.L[2] + c.x2) * g.L[1] + c.x1) * g.Lh0 + c.j);
  return c;
}
// global lex index of a site (the Philox counter word c0, reading R7): the local one unless the lattice is a slab
__device__ __forceinline__ uint32_t lex_global(const Geom& g, const SiteCoord& c) {
  return (uint32_t)(2 * c.j + c.s) + (uint32_t)c.x1 * g.lexS[1] + (uint32_t)c.x2 * g.lexS[2] + (uint32_t)c.x3 * g.lexS[3] + g.lex0;
}

// ------------------------------------------------------------------ CTA tile mapping
// A CTA's threads can cover a 4-D box of sites (power-of-two extents e_d = 1 << s_d, e_0 counted in half-indices) instead of
// B consecutive half-indices, so that the links one thread reads as a neighbour are the links another thread of the CTA
// reads too (they then hit in L1 / are fetched once) -- DESIGN.md "Tile mapping".
struct TileMap {
  int on;              // 0: linear mapping h = blockIdx.x * B + threadIdx.x
  int s0, s1, s2;      // log2 of the tile extents in directions 0 (half-indices), 1, 2; direction 3 takes the rest of B
  FastDiv n0, n1, n2;  // tiles per direction 0, 1, 2
};
// b = the CTA's logical block index (UpdateArgs::rev reverses the launch order, see update.cuh)
__device__ __forceinline__ SiteCoord decode_site_tiled(const Geom& g, const TileMap& tm, int parity, uint32_t b, uint32_t& h) {
  uint32_t t = threadIdx.x;
  const uint32_t jl = t & ((1u << tm.s0) - 1u); t >>= tm.s0;
  const uint32_t y1 = t & ((1u << tm.s1) - 1u); t >>= tm.s1;
  const uint32_t y2 = t & ((1u << tm.s2) - 1u); t >>= tm.s2;
  uint32_t q = fd_div(b, tm.n0); const uint32_t b0 = b - q * tm.n0.d; b = q;
  q = fd_div(b, tm.n1); const uint32_t b1 = b - q * tm.n1.d; b = q;
  q = fd_div(b, tm.n2); const uint32_t b2 = b - q * tm.n2.d; const uint32_t b3 = q;
  SiteCoord c;
  c.j = (int)((b0 << tm.s0) + jl);
  c.x1 = (int)((b1 << tm.s1) + y1);
  c.x2 = (int)((b2 << tm.s2) + y2);
  const int s3 = 31 - __clz((int)blockDim.x) - tm.s0 - tm.s1 - tm.s2;
  c.x3 = (int)((b3 << s3) + t);
  c.s = (parity + c.x1 + c.x2 + c.x3) & 1;
  h = (uint32_t)(((c.x3 * g.L[2] + c.x2) * g.L[1] + c.x1) * g.Lh0 + c.j);
  return c;
}

// half-index offsets to the +d / -d neighbour (which has the other parity).  d is warp-uniform.
__device__ __forceinline__ void nbr_offsets(const Geom& g, const SiteCoord& c, int d, int& fwd, int& bwd) {
  if (d == 0) {
    fwd = c.s ? ((c.j == g.Lh0 - 1) ? -(g.Lh0 - 1) : 1) : 0;
    bwd = c.s ? 0 : ((c.j == 0) ? (g.Lh0 - 1) : -1);
  } else {
    const int xd = (d == 1) ? c.x1 : (d == 2) ? c.x2 : c.x3;
    const int Ld = g.L[d], st = g.stride[d];
    fwd = (xd == Ld - 1) ? -(Ld - 1) * st : st;
    bwd = (xd == 0) ? (Ld - 1) * st : -st;
  }
}

// ------------------------------------------------------------------ vector planes
template <typename R, int NREAL> struct PlaneTraits;
template <> struct PlaneTraits<float, 12> { typedef float4 Vec; static constexpr int VW = 4, NP = 3; };
template <> struct PlaneTraits<float, 18> { typedef float2 Vec; static constexpr int VW = 2, NP = 9; };
template <> struct PlaneTraits<float, 4> { typedef float4 Vec; static constexpr int VW = 4, NP = 1; };
template <> struct PlaneTraits<double, 12> { typedef double2 Vec; static constexpr int VW = 2, NP = 6; };
template <> struct PlaneTraits<double, 18> { typedef double2 Vec; static constexpr int VW = 2, NP = 9; };
template <> struct PlaneTraits<double, 4> { typedef double2 Vec; static constexpr int VW = 2, NP = 2; };

__device__ __forceinline__ void vec_unpack(const float4& v, float* r) { r[0] = v.x; r[1] = v.y; r[2] = v.z; r[3] = v.w; }
__device__ __forceinline__ void vec_unpack(const float2& v, float* r) { r[0] = v.x; r[1] = v.y; }
__device__ __forceinline__ void vec_unpack(const double2& v, double* r) { r[0] = v.x; r[1] = v.y; }
__device__ __forceinline__ void vec_pack(float4& v, const float* r) { v = make_float4(r[0], r[1], r[2], r[3]); }
__device__ __forceinline__ void vec_pack(float2& v, const float* r) { v = make_float2(r[0], r[1]); }
__device__ __forceinline__ void vec_pack(double2& v, const double* r) { v = make_double2(r[0], r[1]); }

// element offset (in vectors) of plane 0 of the (parity, mu) link array
template <int NP>
__device__ __forceinline__ size_t array_base(const Geom& g, int D, int parity, int mu) {
  return (size_t)((parity * D + mu) * NP) * (size_t)g.Vh_pad;
}

// Inside one (parity, mu) array the vector of (half-index h, plane k) sits at  (h / 8) * (8 NP) + k * 8 + (h % 8):
// blocks of 8 half-indices (128 bytes of 16-byte vectors) with their NP planes back to back, so the planes of a link are
// PLANE_STRIDE vectors apart (an immediate offset) and all of a link lies within NP * 128 bytes (page locality on large
// lattices).  A warp's load of one plane of 8 consecutive half-indices is still one full 128-byte line.
constexpr int PLANE_STRIDE = 8;
// Written with shifts and adds (the ALU pipe): as a multiply it becomes an IMAD on the FMA pipe, which is the pipe the
// fp32 kernels are bound by.
// x * NP (mod 2^32) by shifts and adds
template <int NP> __device__ __forceinline__ uint32_t mul_planes(uint32_t x) {
  if constexpr (NP == 1) return x;
  else if constexpr (NP == 2) return x << 1;
  else if constexpr (NP == 3) return (x << 1) + x;
  else if constexpr (NP == 6) return ((x << 1) + x) << 1;
  else if constexpr (NP == 9) return (x << 3) + x;
  else return x * (uint32_t)NP;
}
template <int NP> __device__ __forceinline__ uint32_t blk_off(uint32_t h) {
  const uint32_t q = h >> 3, r = h & 7u;
  if constexpr (NP == 1) return (q << 3) + r;
  else if constexpr (NP == 2) return (q << 4) + r;
  else if constexpr (NP == 3) return (((q << 1) + q) << 3) + r;
  else if constexpr (NP == 6) return (((q << 1) + q) << 4) + r;
  else if constexpr (NP == 9) return (((q << 3) + q) << 3) + r;
  else return q * (8u * NP) + r;
}

// load the NREAL reals of link h of the array starting at `base` (vectors); NC = through the read-only path
template <typename R, int NREAL, bool NC>
__device__ __forceinline__ void load_reals(const typename PlaneTraits<R, NREAL>::Vec* __restrict__ links, const Geom& g,
                                           size_t base, uint32_t h, R* out) {
  typedef PlaneTraits<R, NREAL> T;
  const typename T::Vec* p = links + base + blk_off<T::NP>(h);
#pragma unroll
  for (int k = 0; k < T::NP; ++k) {
    typename T::Vec v = NC ? __ldg(p + k * PLANE_STRIDE) : p[k * PLANE_STRIDE];
    vec_unpack(v, out + k * T::VW);
  }
}
template <typename R, int NREAL>
__device__ __forceinline__ void store_reals(typename PlaneTraits<R, NREAL>::Vec* links, const Geom& g, size_t base, uint32_t h,
                                            const R* in) {
  typedef PlaneTraits<R, NREAL> T;
  typename T::Vec* p = links + base + blk_off<T::NP>(h);
#pragma unroll
  for (int k = 0; k < T::NP; ++k) {
    typename T::Vec v;
    vec_pack(v, in + k * T::VW);
    p[k * PLANE_STRIDE] = v;
  }
}

// ------------------------------------------------------------------ programmatic dependent launch
// The sub-steps of a sweep are a chain of dependent kernels on one stream.  Each update kernel is launched with the
// programmatic-stream-serialization attribute: its CTAs may become resident while the previous kernel drains, run the part
// that does not touch the links (site decoding, neighbour offsets, the heatbath's random numbers) and then block in
// pdl_wait() until the previous grid has completed and its stores are visible.  pdl_trigger() at the top of a kernel lets
// the next one do the same.  Without the attribute both are no-ops.
__device__ __forceinline__ void pdl_trigger() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
template <typename... KArgs, typename... Args>
inline cudaError_t launch_pdl(void (*kern)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st, Args... args) {
  cudaLaunchConfig_t cfg;
  cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = st;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  return cudaLaunchKernelEx(&cfg, kern, KArgs(args)...);
}

// ------------------------------------------------------------------ math dispatch
// The arguments of these calls are positive normal numbers (squared norms guarded by reading R4, radicands 1 - x^2 of
// numbers strictly inside (-1, 1)), so the special-case paths of the library routines are dead weight.
//   float:  the SFU approximations (MUFU.RSQ / MUFU.SQRT / MUFU.RCP, 1-2 ulp; the link tolerance is 2e-5) in place of the
//           IEEE sqrtf and division, whose slow paths put a branch and a call into the hit;
//   double: seed + Newton forms without branches (hb_math.cuh, ~1e-16 relative; tolerance 1e-12).
__device__ __forceinline__ float q_rsqrt(float x) { float r; asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
__device__ __forceinline__ float q_sqrt(float x) { float r; asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
__device__ __forceinline__ float q_rcp(float x) { float r; asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
__device__ __forceinline__ double q_rsqrt(double x) { return hbm::rsqrt(x); }
__device__ __forceinline__ double q_sqrt(double x) { return hbm::sqrt_pos(x); }
__device__ __forceinline__ double q_rcp(double x) { return hbm::rcp(x); }
__device__ __forceinline__ void q_sincospi(float x, float* s, float* c) { sincospif(x, s, c); }
__device__ __forceinline__ void q_sincospi(double x, double* s, double* c) { sincospi(x, s, c); }
__device__ __forceinline__ float q_fma(float a, float b, float c) { return fmaf(a, b, c); }
__device__ __forceinline__ double q_fma(double a, double b, double c) { return fma(a, b, c); }

}  // namespace qcd
