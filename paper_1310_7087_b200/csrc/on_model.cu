// on_model.cu -- the second workload of the paper: the O(N) scalar model on lattice SITES, updated by multi-hit ("improved")
// Metropolis on the checkerboard.  PAPER.md:106 "In case of O(N) models the fields are set with
// N-vectors, which are associated with lattice sites"; :108 "Improved Metropolis algorithm [7] is used for O(N) update";
// :134 "For O(4) model NHIT=100 tries were used to update each lattice site".  Ref [7] is not available; the readings
// R16-R19 of DESIGN.md sec 3 fix the action, the meaning of NHIT, the Philox keying and the starts:
//   S = sum_x [ -2 kappa sum_mu phi(x).phi(x+mu) + phi.phi + lambda (phi.phi - 1)^2 ]                       (R16)
//   a visit of a site = NHIT tries phi' = phi + delta (2u - 1) per component, accepted iff u' < exp(-dS), all NHIT made (R17)
//   one Philox4x32-10 block per try -> five 23-bit numbers (four components, one acceptance), N <= 4          (R18)
// Layout: a site's N reals padded to 4, one 16-byte vector (fp32) or two (fp64) per site in the blocked vector-plane
// arrays of common.cuh, [parity][h / 8][plane][h % 8]: a warp's load of 8 neighbouring sites is one 128-byte line.
// One thread per site; the 2D neighbour vectors are read once and summed, the NHIT tries run in registers.  The kernel is
// bound by the instruction stream of Philox and the exponential (NHIT = 100: ~10^4 instructions per site against 9 vectors
// of memory traffic), not by HBM.
#include <cmath>
#include <cstdio>
#include <cstring>
#include <string>

#include "../../include/qcd.h"
#include "common.cuh"
#include "philox.cuh"

namespace qcd { int set_error(int code, const std::string& msg); }
using namespace qcd;

#define ON_TRY(expr)                                                                                             \
  do {                                                                                                           \
    cudaError_t e_ = (expr);                                                                                     \
    if (e_ != cudaSuccess) return set_error(QCD_ERR_CUDA, std::string(#expr) + ": " + cudaGetErrorString(e_));   \
  } while (0)

struct qcd_on {
  int D, dims[4], N, precision;
  Geom g;
  size_t bytes;
  void* mem;
  bool owns_mem, has_field;
  cudaStream_t stream;
  uint64_t seed;
  uint32_t sweep;
  unsigned long long* d_counts;   // [accepted tries] since the last init (device counter)
  unsigned long long tried;       // tries made since the last init (known on the host: V/2 * nhit per half sweep)
  double* d_partials;
  size_t partials_cap;
  double* d_results;              // 8 doubles
  double* h_results;              // pinned
  void* d_canon;
};

namespace {

struct OnArgs {
  double kappa, lambda, delta;
  int parity, nhit;
  uint32_t sweep, key0, key1;
  unsigned long long* counts;
};

template <typename R> struct OnIO {
  typedef PlaneTraits<R, 4> T;
  typedef typename T::Vec Vec;
  static __device__ __forceinline__ void load(const Vec* __restrict__ f, const Geom& g, int parity, uint32_t h, R* out) {
    load_reals<R, 4, true>(f, g, (size_t)parity * T::NP * g.Vh_pad, h, out);
  }
  static __device__ __forceinline__ void store(Vec* f, const Geom& g, int parity, uint32_t h, const R* in) {
    store_reals<R, 4>(f, g, (size_t)parity * T::NP * g.Vh_pad, h, in);
  }
};

// the five 23-bit numbers of one Philox block (R18)
__device__ __forceinline__ void on_numbers(const Philox4& w, uint32_t (&k)[5]) {
  k[0] = w.x & 0x7FFFFFu; k[1] = w.y & 0x7FFFFFu; k[2] = w.z & 0x7FFFFFu; k[3] = w.w & 0x7FFFFFu;
  k[4] = (w.x >> 23) | ((w.y >> 23) << 9) | (((w.z >> 23) & 31u) << 18);
}
__device__ __forceinline__ uint32_t on_c2(int parity, int hit, int domain) {
  return ((uint32_t)parity << 4) | ((uint32_t)hit << 8) | ((uint32_t)domain << 24);
}
// u = (k + 1/2) 2^-23, exact in both precisions; float: without an integer conversion (philox.cuh, uniform23f)
__device__ __forceinline__ float on_uniform(uint32_t k, float) { return __uint_as_float(0x3F800000u | k) - 0.99999994f; }
// double: k < 2^23 placed in the low mantissa bits of 2^52 is the double 2^52 + k, and 2^52 - 1/2 is a double too, so one
// exact subtraction gives k + 1/2 without an integer conversion (five I2F.F64 per try otherwise)
__device__ __forceinline__ double on_uniform(uint32_t k, double) {
  return (__hiloint2double(0x43300000, (int)k) - 4503599627370495.5) * 1.1920928955078125e-07;
}

template <int N> __device__ __forceinline__ double on_local_action(const double* p, const double* h, double kappa, double lambda) {
  double ph = 0.0, pp = 0.0;
#pragma unroll
  for (int a = 0; a < N; ++a) { ph += p[a] * h[a]; pp += p[a] * p[a]; }
  return -2.0 * kappa * ph + pp + lambda * (pp - 1.0) * (pp - 1.0);
}
// guard-band path of the fp32 kernel: the decision of one try in double from the float-valued operands (out of line, rare)
// The operands travel BY VALUE: handed over as pointers, phi and h had to live in local memory, and the hot loop stored
// phi there on every accepted try (1.7 STL per try, profiles/r3_on_model.md).
template <int N> struct OnVecF { float v[N]; };
template <int N> struct OnVecD { double v[N]; };
template <int N> static __device__ __noinline__ bool on_accept_f64_cold(OnVecF<N> p, OnVecF<N> q, OnVecD<N> h, double kappa, double lambda, double u) {
  double pd[N], qd[N];
#pragma unroll
  for (int a = 0; a < N; ++a) { pd[a] = (double)p.v[a]; qd[a] = (double)q.v[a]; }
  const double dS = on_local_action<N>(qd, h.v, kappa, lambda) - on_local_action<N>(pd, h.v, kappa, lambda);
  return u < exp(-dS);
}

template <typename R, int D, int N>
__global__ void __launch_bounds__(128) on_update_kernel(Geom g, typename OnIO<R>::Vec* field, OnArgs a) {
  typedef OnIO<R> IO;
  const uint32_t h = blockIdx.x * blockDim.x + threadIdx.x;
  unsigned acc = 0;
  if (h < g.Vh) {
    const int p = a.parity, q = 1 - p;
    const SiteCoord sc = decode_site(g, h, p);
    const uint32_t lex = 2u * h + (uint32_t)sc.s;
    // sum of the 2D neighbours (the other parity), in double: exact for float operands
    double hs[N];
#pragma unroll
    for (int c = 0; c < N; ++c) hs[c] = 0.0;
#pragma unroll
    for (int d = 0; d < D; ++d) {
      int fo, bo;
      nbr_offsets(g, sc, d, fo, bo);
      R v[4];
      IO::load(field, g, q, h + (uint32_t)fo, v);
#pragma unroll
      for (int c = 0; c < N; ++c) hs[c] += (double)v[c];
      IO::load(field, g, q, h + (uint32_t)bo, v);
#pragma unroll
      for (int c = 0; c < N; ++c) hs[c] += (double)v[c];
    }
    R own[4];
    {
      // the own array is written by this kernel (each thread its own element): plain load
      const typename IO::Vec* src = field + (size_t)p * IO::T::NP * g.Vh_pad + blk_off<IO::T::NP>(h);
#pragma unroll
      for (int k = 0; k < IO::T::NP; ++k) vec_unpack(src[k * PLANE_STRIDE], own + k * IO::T::VW);
    }
    R ph[N], hr[N];
    R pp = R(0);
#pragma unroll
    for (int c = 0; c < N; ++c) { ph[c] = own[c]; hr[c] = (R)hs[c]; pp = q_fma(ph[c], ph[c], pp); }
    const R k2 = (R)(-2.0 * a.kappa), lam = (R)a.lambda, delta = (R)a.delta;
    const uint32_t c2 = on_c2(p, 0, 2);
#pragma unroll 2
    for (int t = 0; t < a.nhit; ++t) {
      uint32_t k[5];
      on_numbers(philox4x32_10(lex, a.sweep, c2 | ((uint32_t)t << 8), 0u, a.key0, a.key1), k);
      R qv[N];
      R qq = R(0), dh = R(0);
#pragma unroll
      for (int c = 0; c < N; ++c) {
        const R s = q_fma(R(2), on_uniform(k[c], R(0)), R(-1));       // exact
        qv[c] = q_fma(delta, s, ph[c]);
        qq = q_fma(qv[c], qv[c], qq);
        dh = q_fma(qv[c] - ph[c], hr[c], dh);
      }
      // dS = -2 kappa (phi' - phi).h + (phi'^2 - phi^2) + lambda (phi'^2 - phi^2)(phi'^2 + phi^2 - 2)
      const R d2 = qq - pp;
      const R t1 = k2 * dh, t3 = lam * d2 * (qq + pp - R(2));
      const R dS = t1 + d2 + t3;
      const R u = on_uniform(k[4], R(0));
      bool ok;
      if constexpr (sizeof(R) == 4) {
        const float e = __expf(-dS);
        ok = u < e;
        // the float error of dS is below 8e-7 (|t1| + |d2| + |t3|) + 1e-6 (roundings of the sums, of h and of the products),
        // __expf adds 2e-6 relative: inside that band around the acceptance boundary the try is decided in double, like
        // the oracle does, from the same float-valued operands
        if (fabsf(u - e) < (8e-7f * (fabsf(t1) + fabsf(d2) + fabsf(t3)) + 4e-6f) * e) {
          OnVecF<N> pv, qw;
          OnVecD<N> hv;
#pragma unroll
          for (int c = 0; c < N; ++c) { pv.v[c] = ph[c]; qw.v[c] = qv[c]; hv.v[c] = hs[c]; }
          ok = on_accept_f64_cold<N>(pv, qw, hv, a.kappa, a.lambda, (double)u);
        }
      } else {
        ok = u < exp(-dS);
      }
      if (ok) {
#pragma unroll
        for (int c = 0; c < N; ++c) ph[c] = qv[c];
        pp = qq;
        ++acc;
      }
    }
#pragma unroll
    for (int c = 0; c < 4; ++c) own[c] = c < N ? ph[c] : R(0);
    IO::store(field, g, p, h, own);
  }
  // accepted tries: warp sum, one integer atomic per warp (integer addition: order-independent, deterministic)
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) acc += __shfl_down_sync(0xffffffffu, acc, o);
  if ((threadIdx.x & 31) == 0 && acc) atomicAdd(a.counts, (unsigned long long)acc);
}

template <typename R, int N>
__global__ void __launch_bounds__(128) on_init_kernel(Geom g, typename OnIO<R>::Vec* field, int hot, uint32_t key0, uint32_t key1) {
  const uint32_t h = blockIdx.x * blockDim.x + threadIdx.x;
  const int p = blockIdx.y;
  if (h >= g.Vh) return;
  const SiteCoord sc = decode_site(g, h, p);
  const uint32_t lex = 2u * h + (uint32_t)sc.s;
  uint32_t k[5];
  on_numbers(philox4x32_10(lex, 0u, on_c2(p, 0, 3), 0u, key0, key1), k);
  R v[4];
#pragma unroll
  for (int c = 0; c < 4; ++c) v[c] = c >= N ? R(0) : hot ? (R)(2.0 * on_uniform(k[c], 0.0) - 1.0) : (c == 0 ? R(1) : R(0));
  OnIO<R>::store(field, g, p, h, v);
}

// canonical [lex][N] <-> internal
template <typename R, int N, bool TO_INTERNAL>
__global__ void __launch_bounds__(128) on_layout_kernel(Geom g, typename OnIO<R>::Vec* field, R* canon) {
  const uint32_t lex = blockIdx.x * blockDim.x + threadIdx.x;
  if (lex >= g.V) return;
  const uint32_t h = lex >> 1;
  const uint32_t row = fd_div(h, g.dLh0), r2 = fd_div(row, g.dL1), r3 = fd_div(r2, g.dL2);
  const uint32_t x1 = row - r2 * (uint32_t)g.L[1], x2 = r2 - r3 * (uint32_t)g.L[2];
  const int p = (int)(((lex & 1u) + x1 + x2 + r3) & 1u);
  R v[4] = {R(0), R(0), R(0), R(0)};
  if (TO_INTERNAL) {
#pragma unroll
    for (int c = 0; c < N; ++c) v[c] = canon[(size_t)lex * N + c];
    OnIO<R>::store(field, g, p, h, v);
  } else {
    const typename OnIO<R>::Vec* src = field + (size_t)p * OnIO<R>::T::NP * g.Vh_pad + blk_off<OnIO<R>::T::NP>(h);
#pragma unroll
    for (int k = 0; k < OnIO<R>::T::NP; ++k) vec_unpack(src[k * PLANE_STRIDE], v + k * OnIO<R>::T::VW);
#pragma unroll
    for (int c = 0; c < N; ++c) canon[(size_t)lex * N + c] = v[c];
  }
}

// observables: per-block partial sums of phi.phi, sum_mu phi(x).phi(x+mu), phi_a  (fp64 accumulation, fixed order)
template <typename R, int D, int N>
__global__ void __launch_bounds__(128) on_measure_kernel(Geom g, const typename OnIO<R>::Vec* __restrict__ field, double* partials) {
  typedef OnIO<R> IO;
  const uint32_t h = blockIdx.x * blockDim.x + threadIdx.x;
  const int p = blockIdx.y;
  double v[6] = {0, 0, 0, 0, 0, 0};
  if (h < g.Vh) {
    const SiteCoord sc = decode_site(g, h, p);
    R own[4];
    IO::load(field, g, p, h, own);
#pragma unroll
    for (int c = 0; c < N; ++c) { v[0] += (double)own[c] * (double)own[c]; v[2 + c] = (double)own[c]; }
#pragma unroll
    for (int d = 0; d < D; ++d) {
      int fo, bo;
      nbr_offsets(g, sc, d, fo, bo);
      R w[4];
      IO::load(field, g, 1 - p, h + (uint32_t)fo, w);
#pragma unroll
      for (int c = 0; c < N; ++c) v[1] += (double)own[c] * (double)w[c];
    }
  }
  __shared__ double sm[6][4];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
  for (int k = 0; k < 6; ++k) {
    double x = v[k];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) x += __shfl_down_sync(0xffffffffu, x, o);
    if (lane == 0) sm[k][warp] = x;
  }
  __syncthreads();
  if (threadIdx.x < 6) {
    const uint32_t nb = gridDim.x * gridDim.y, bid = blockIdx.y * gridDim.x + blockIdx.x;
    partials[(size_t)threadIdx.x * nb + bid] = sm[threadIdx.x][0] + sm[threadIdx.x][1] + sm[threadIdx.x][2] + sm[threadIdx.x][3];
  }
}
__global__ void __launch_bounds__(256) on_reduce_kernel(const double* partials, uint32_t nblocks, double* out) {
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
  if (threadIdx.x == 0) out[blockIdx.x] = sm[0];
}

Geom on_geom(int D, const int* dims) {
  Geom g;
  memset(&g, 0, sizeof(g));
  g.D = D;
  uint64_t V = 1;
  for (int d = 0; d < 4; ++d) { g.L[d] = d < D ? dims[d] : 1; g.Li[d] = g.L[d]; V *= g.L[d]; }
  g.Lh0 = g.L[0] / 2;
  g.stride[1] = g.Lh0; g.stride[2] = g.Lh0 * g.L[1]; g.stride[3] = g.Lh0 * g.L[1] * g.L[2];
  g.V = (uint32_t)V; g.Vh = (uint32_t)(V / 2); g.Vh_pad = (g.Vh + 31u) & ~31u; g.Vh_int = g.Vh;
  g.dLh0 = make_fastdiv((uint32_t)g.Lh0); g.dL1 = make_fastdiv((uint32_t)g.L[1]); g.dL2 = make_fastdiv((uint32_t)g.L[2]);
  g.iLh0 = g.dLh0; g.iL1 = g.dL1; g.iL2 = g.dL2;
  g.sd = -1;
  return g;
}

bool on_valid(int D, const int* dims, int N, int precision) {
  if (D < 2 || D > 4 || !dims || N < 1 || N > 4 || (precision != QCD_FP32 && precision != QCD_FP64)) return false;
  double v = 1.0;
  for (int d = 0; d < D; ++d) { if (dims[d] < 2 || (dims[d] & 1)) return false; v *= dims[d]; }
  return v <= 2147483648.0;
}

// f.template operator()<R, D, N>()
template <typename F> int on_dispatch(const qcd_on* L, F&& f) {
#define ON_CASE(D_, N_)                                                                                                              \
  if (L->D == D_ && L->N == N_) return L->precision == QCD_FP32 ? f.template operator()<float, D_, N_>() : f.template operator()<double, D_, N_>();
  ON_CASE(2, 1) ON_CASE(2, 2) ON_CASE(2, 3) ON_CASE(2, 4) ON_CASE(3, 1) ON_CASE(3, 2) ON_CASE(3, 3) ON_CASE(3, 4)
  ON_CASE(4, 1) ON_CASE(4, 2) ON_CASE(4, 3) ON_CASE(4, 4)
#undef ON_CASE
  return set_error(QCD_ERR_UNSUPPORTED, "unsupported (D, N)");
}

struct OnUpdateOp {
  qcd_on* L; OnArgs a;
  template <typename R, int D, int N> int operator()() {
    on_update_kernel<R, D, N><<<(L->g.Vh + 127) / 128, 128, 0, L->stream>>>(L->g, (typename OnIO<R>::Vec*)L->mem, a);
    ON_TRY(cudaGetLastError());
    return QCD_OK;
  }
};
struct OnInitOp {
  qcd_on* L; int hot;
  template <typename R, int D, int N> int operator()() {
    on_init_kernel<R, N><<<dim3((L->g.Vh + 127) / 128, 2), 128, 0, L->stream>>>(L->g, (typename OnIO<R>::Vec*)L->mem, hot, (uint32_t)(L->seed & 0xFFFFFFFFull),
                                                                              (uint32_t)(L->seed >> 32));
    ON_TRY(cudaGetLastError());
    return QCD_OK;
  }
};
struct OnLayoutOp {
  qcd_on* L; void* canon; bool to_internal;
  template <typename R, int D, int N> int operator()() {
    const dim3 grid((L->g.V + 127) / 128);
    if (to_internal) on_layout_kernel<R, N, true><<<grid, 128, 0, L->stream>>>(L->g, (typename OnIO<R>::Vec*)L->mem, (R*)canon);
    else on_layout_kernel<R, N, false><<<grid, 128, 0, L->stream>>>(L->g, (typename OnIO<R>::Vec*)L->mem, (R*)canon);
    ON_TRY(cudaGetLastError());
    return QCD_OK;
  }
};
struct OnMeasureOp {
  qcd_on* L;
  template <typename R, int D, int N> int operator()() {
    const uint32_t nb = ((L->g.Vh + 127) / 128) * 2;
    if ((size_t)6 * nb > L->partials_cap) {
      if (L->d_partials) ON_TRY(cudaFree(L->d_partials));
      L->d_partials = nullptr; L->partials_cap = 0;
      ON_TRY(cudaMalloc(&L->d_partials, (size_t)6 * nb * sizeof(double)));
      L->partials_cap = (size_t)6 * nb;
    }
    on_measure_kernel<R, D, N><<<dim3(nb / 2, 2), 128, 0, L->stream>>>(L->g, (const typename OnIO<R>::Vec*)L->mem, L->d_partials);
    on_reduce_kernel<<<6, 256, 0, L->stream>>>(L->d_partials, nb, L->d_results);
    ON_TRY(cudaGetLastError());
    return QCD_OK;
  }
};

size_t on_canonical_bytes(const qcd_on* L) { return (size_t)L->g.V * L->N * (L->precision == QCD_FP32 ? 4 : 8); }

int on_half_sweep(qcd_on* L, int parity, double kappa, double lambda, double delta, int nhit) {
  OnUpdateOp op;
  op.L = L;
  memset(&op.a, 0, sizeof(op.a));
  op.a.kappa = kappa; op.a.lambda = lambda; op.a.delta = L->precision == QCD_FP32 ? (double)(float)delta : delta;
  op.a.parity = parity; op.a.nhit = nhit; op.a.sweep = L->sweep;
  op.a.key0 = (uint32_t)(L->seed & 0xFFFFFFFFull); op.a.key1 = (uint32_t)(L->seed >> 32);
  op.a.counts = L->d_counts;
  int rc = on_dispatch(L, op);
  if (rc != QCD_OK) return rc;
  L->tried += (unsigned long long)L->g.Vh * (unsigned long long)nhit;
  return QCD_OK;
}

bool on_params_ok(double kappa, double lambda, double delta, int nhit) {
  return std::isfinite(kappa) && std::isfinite(lambda) && lambda >= 0.0 && std::isfinite(delta) && delta > 0.0 && nhit >= 0 && nhit <= 65535;
}

}  // namespace

extern "C" {

size_t qcd_on_bytes(int D, const int* dims, int N, int precision) {
  if (!on_valid(D, dims, N, precision)) return 0;
  const Geom g = on_geom(D, dims);
  return (size_t)2 * (precision == QCD_FP32 ? 1 : 2) * g.Vh_pad * 16;
}

int qcd_on_create(int D, const int* dims, int N, int precision, void* device_mem, size_t bytes, void* cuda_stream, qcd_on_t** out) {
  if (!out) return set_error(QCD_ERR_INVALID_ARG, "out is NULL");
  *out = nullptr;
  if (!on_valid(D, dims, N, precision)) return set_error(QCD_ERR_INVALID_ARG, "invalid D / dims (even, >= 2) / N (1..4) / precision");
  const size_t need = qcd_on_bytes(D, dims, N, precision);
  if (device_mem && (bytes < need || ((uintptr_t)device_mem & 255u))) return set_error(QCD_ERR_INVALID_ARG, "device_mem too small or not 256-byte aligned");
  qcd_on* L = new qcd_on();
  memset(L, 0, sizeof(*L));
  L->D = D; L->N = N; L->precision = precision;
  for (int d = 0; d < 4; ++d) L->dims[d] = d < D ? dims[d] : 1;
  L->g = on_geom(D, dims);
  L->bytes = need; L->mem = device_mem; L->stream = (cudaStream_t)cuda_stream;
  cudaError_t e = cudaSuccess;
  if (!device_mem) {
    e = cudaMalloc(&L->mem, need);
    if (e != cudaSuccess) { delete L; return set_error(QCD_ERR_ALLOC, std::string("cudaMalloc field: ") + cudaGetErrorString(e)); }
    L->owns_mem = true;
  }
  if (e == cudaSuccess) e = cudaMalloc(&L->d_counts, 2 * sizeof(unsigned long long));
  if (e == cudaSuccess) e = cudaMemsetAsync(L->d_counts, 0, 2 * sizeof(unsigned long long), L->stream);
  if (e == cudaSuccess) e = cudaMalloc(&L->d_results, 8 * sizeof(double));
  if (e == cudaSuccess) e = cudaMallocHost(&L->h_results, 16 * sizeof(double));
  if (e == cudaSuccess) e = cudaMemsetAsync(L->mem, 0, need, L->stream);
  if (e != cudaSuccess) { std::string m = cudaGetErrorString(e); qcd_on_destroy(L); return set_error(QCD_ERR_CUDA, "on_create: " + m); }
  *out = L;
  return QCD_OK;
}

int qcd_on_destroy(qcd_on_t* L) {
  if (!L) return QCD_OK;
  cudaStreamSynchronize(L->stream);
  if (L->owns_mem && L->mem) cudaFree(L->mem);
  if (L->d_counts) cudaFree(L->d_counts);
  if (L->d_partials) cudaFree(L->d_partials);
  if (L->d_results) cudaFree(L->d_results);
  if (L->h_results) cudaFreeHost(L->h_results);
  if (L->d_canon) cudaFree(L->d_canon);
  delete L;
  return QCD_OK;
}

int qcd_on_init(qcd_on_t* L, int start, uint64_t seed) {
  if (!L) return set_error(QCD_ERR_INVALID_ARG, "lattice is NULL");
  if (start != QCD_COLD && start != QCD_HOT) return set_error(QCD_ERR_INVALID_ARG, "start must be QCD_COLD or QCD_HOT");
  L->seed = seed; L->sweep = 0; L->tried = 0;
  ON_TRY(cudaMemsetAsync(L->d_counts, 0, 2 * sizeof(unsigned long long), L->stream));
  OnInitOp op{L, start == QCD_HOT ? 1 : 0};
  int rc = on_dispatch(L, op);
  if (rc == QCD_OK) L->has_field = true;
  return rc;
}

int qcd_on_half_sweep(qcd_on_t* L, int parity, double kappa, double lambda, double delta, int nhit) {
  if (!L) return set_error(QCD_ERR_INVALID_ARG, "lattice is NULL");
  if (!L->has_field) return set_error(QCD_ERR_STATE, "no field yet (qcd_on_init / qcd_on_set_field)");
  if ((parity != 0 && parity != 1) || !on_params_ok(kappa, lambda, delta, nhit)) return set_error(QCD_ERR_INVALID_ARG, "bad parity / kappa / lambda (>= 0) / delta (> 0) / nhit (0..65535)");
  return on_half_sweep(L, parity, kappa, lambda, delta, nhit);
}

int qcd_on_sweep(qcd_on_t* L, double kappa, double lambda, double delta, int nhit) {
  if (!L) return set_error(QCD_ERR_INVALID_ARG, "lattice is NULL");
  if (!L->has_field) return set_error(QCD_ERR_STATE, "no field yet (qcd_on_init / qcd_on_set_field)");
  if (!on_params_ok(kappa, lambda, delta, nhit)) return set_error(QCD_ERR_INVALID_ARG, "bad kappa / lambda (>= 0) / delta (> 0) / nhit (0..65535)");
  for (int p = 0; p < 2; ++p) { int rc = on_half_sweep(L, p, kappa, lambda, delta, nhit); if (rc != QCD_OK) return rc; }
  L->sweep += 1;
  return QCD_OK;
}

int qcd_on_measure(qcd_on_t* L, double* phi2, double* link, double* mag) {
  if (!L) return set_error(QCD_ERR_INVALID_ARG, "lattice is NULL");
  if (!L->has_field) return set_error(QCD_ERR_STATE, "no field yet");
  OnMeasureOp op{L};
  int rc = on_dispatch(L, op);
  if (rc != QCD_OK) return rc;
  ON_TRY(cudaMemcpyAsync(L->h_results, L->d_results, 6 * sizeof(double), cudaMemcpyDeviceToHost, L->stream));
  ON_TRY(cudaStreamSynchronize(L->stream));
  const double V = (double)L->g.V;
  if (phi2) *phi2 = L->h_results[0] / V;
  if (link) *link = L->h_results[1] / (V * L->D);
  if (mag) for (int a = 0; a < L->N; ++a) mag[a] = L->h_results[2 + a] / V;
  return QCD_OK;
}

int qcd_on_get_counts(qcd_on_t* L, uint64_t* accepted, uint64_t* tried) {
  if (!L || !accepted || !tried) return set_error(QCD_ERR_INVALID_ARG, "NULL argument");
  unsigned long long c = 0;
  ON_TRY(cudaMemcpyAsync(&c, L->d_counts, sizeof(c), cudaMemcpyDeviceToHost, L->stream));
  ON_TRY(cudaStreamSynchronize(L->stream));
  *accepted = (uint64_t)c; *tried = (uint64_t)L->tried;
  return QCD_OK;
}

static int on_field_io(qcd_on_t* L, void* ptr, size_t bytes, int is_device, bool set) {
  if (!L || !ptr) return set_error(QCD_ERR_INVALID_ARG, "NULL argument");
  if (!set && !L->has_field) return set_error(QCD_ERR_STATE, "no field yet");
  if (bytes != on_canonical_bytes(L)) return set_error(QCD_ERR_INVALID_ARG, "bytes must equal V*N*sizeof(real)");
  void* canon = ptr;
  if (!is_device) {
    if (!L->d_canon && cudaMalloc(&L->d_canon, bytes) != cudaSuccess) { L->d_canon = nullptr; cudaGetLastError(); return set_error(QCD_ERR_ALLOC, "staging buffer"); }
    canon = L->d_canon;
    if (set) ON_TRY(cudaMemcpyAsync(canon, ptr, bytes, cudaMemcpyHostToDevice, L->stream));
  }
  OnLayoutOp op{L, canon, set};
  int rc = on_dispatch(L, op);
  if (rc != QCD_OK) return rc;
  if (!is_device) {
    if (!set) ON_TRY(cudaMemcpyAsync(ptr, canon, bytes, cudaMemcpyDeviceToHost, L->stream));
    ON_TRY(cudaStreamSynchronize(L->stream));
  }
  if (set) L->has_field = true;
  return QCD_OK;
}
int qcd_on_get_field(qcd_on_t* L, void* dst, size_t bytes, int dst_is_device) { return on_field_io(L, dst, bytes, dst_is_device, false); }
int qcd_on_set_field(qcd_on_t* L, const void* src, size_t bytes, int src_is_device) { return on_field_io(L, const_cast<void*>(src), bytes, src_is_device, true); }

int qcd_on_set_seed(qcd_on_t* L, uint64_t seed) { if (!L) return set_error(QCD_ERR_INVALID_ARG, "NULL argument"); L->seed = seed; return QCD_OK; }
int qcd_on_set_sweep_counter(qcd_on_t* L, uint32_t v) { if (!L) return set_error(QCD_ERR_INVALID_ARG, "NULL argument"); L->sweep = v; return QCD_OK; }
int qcd_on_get_sweep_counter(qcd_on_t* L, uint32_t* out) { if (!L || !out) return set_error(QCD_ERR_INVALID_ARG, "NULL argument"); *out = L->sweep; return QCD_OK; }

}  // extern "C"
