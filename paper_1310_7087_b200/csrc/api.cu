// api.cu -- the C ABI of include/qcd.h: argument checking, lattice state, launch sequencing (sweep order R1/R2, chained by
// programmatic dependent launch), event profiling, and the non-update kernels (init, layout, measurement, probes).
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <string>
#include <vector>

#include <curand_philox4x32_x.h>

#include "../../include/qcd.h"
#include "aux_kernels.cuh"
#include "launch.h"

using namespace qcd;

namespace {

thread_local std::string g_err;
int fail(int code, const std::string& msg) { g_err = msg; return code; }
}  // namespace
// the other translation units of the library (on_model.cu) report errors through the same thread-local message
namespace qcd { int set_error(int code, const std::string& msg) { return fail(code, msg); } }
namespace {
#define CUDA_TRY(expr)                                                                                   \
  do {                                                                                                   \
    cudaError_t e_ = (expr);                                                                             \
    if (e_ != cudaSuccess) return fail(QCD_ERR_CUDA, std::string(#expr) + ": " + cudaGetErrorString(e_)); \
  } while (0)

struct EventPair { cudaEvent_t a, b; int kind; int n; };   // n = update-kernel launches between a and b

}  // namespace

struct qcd_lattice {
  int D, dims[4], Nc, precision;   // dims: the local extents (a slab: n_int + 2 along the split direction)
  // slab of a larger lattice (Geom::sd >= 0): global extents, and the global coordinate of the first own layer
  int gdims[4], slab_off;
  unsigned flags;
  bool comp;
  Geom g;
  size_t bytes;
  void* mem;
  bool owns_mem;
  cudaStream_t stream;
  uint64_t seed;
  uint32_t sweep;
  bool has_links;
  int max_trials;
  bool debug_trials, profile, bulk_copy, alternate_order, exchange_rows01;
  uint8_t* d_trials;
  // per-block / per-warp partial sums of the reductions, one allocation of three regions (sizes fixed by the geometry):
  // [fused plaquette: NPL x np_warp][plaquette kernel: NPL x nb_plaq][Polyakov: 2 x nb_poly]
  double* d_partials;
  size_t partials_cap;   // doubles
  double* d_results;     // 48 doubles: last measurement + accumulator (see qcd_lattice_create)
  double* h_results;     // pinned, 48 doubles
  std::vector<EventPair> ev_used, ev_free;
  double prof_ms[2];
  uint64_t prof_n[2];
  uint64_t launches;
  uint32_t order_toggle;   // flips with every update launch (UpdateArgs::rev)
  qcd_lattice *push_prev, *push_next;   // divided lattice, single-process driver: the update kernels write the boundary layers there too
  // What the kernel launched last on the stream wrote: (parity, mu) of an update kernel; -1: no links (measurement,
  // get_links); -2: all links (init, set_links, the create-time memset).  The next update kernel may fetch, before its
  // griddepcontrol.wait, only arrays that kernel does not write (update.cuh)
  int last_parity, last_mu;
  // side stream + events: the latency-bound Polyakov kernel runs beside the plaquette kernel (qcd_measure)
  cudaStream_t side;
  cudaEvent_t ev_fork, ev_join;
  // bounded staging buffer for qcd_get/set_links with HOST pointers (canonical layout, STAGE_BYTES, allocated on first use)
  void* d_canon;
};

namespace {

int plane_params(int Nc, int precision, bool comp, int* nreal, int* vec_bytes, int* np) {
  int nr = (Nc == 2) ? 4 : (comp ? 12 : 18);
  int vw = (precision == QCD_FP32) ? ((nr % 4 == 0) ? 4 : 2) : 2;
  *nreal = nr;
  *vec_bytes = vw * (precision == QCD_FP32 ? 4 : 8);
  *np = nr / vw;
  return 0;
}

bool valid_shape(int D, const int* dims, int Nc, int precision, unsigned flags, int* why) {
  *why = QCD_ERR_INVALID_ARG;
  if (D < 2 || D > 4 || !dims) return false;
  if (Nc != 2 && Nc != 3) return false;
  if (precision != QCD_FP32 && precision != QCD_FP64) return false;
  if (flags & ~QCD_FLAG_COMPRESS12) return false;
  double v = 1.0;
  for (int d = 0; d < D; ++d) {
    if (dims[d] < 2 || (dims[d] & 1)) return false;
    v *= dims[d];
  }
  if (v > 2147483648.0) return false;          // V/2 and lex must fit 32-bit (Philox c0 = lex)
  if ((flags & QCD_FLAG_COMPRESS12) && Nc == 2) { *why = QCD_ERR_UNSUPPORTED; return false; }
  // the kernels address one (parity, direction) array of NP planes x Vh_pad vectors with 32 bits (array bases are 64-bit)
  int nreal, vb, np;
  plane_params(Nc, precision, (flags & QCD_FLAG_COMPRESS12) != 0, &nreal, &vb, &np);
  if ((double)np * (v / 2.0 + 32.0) >= 4294967296.0) { *why = QCD_ERR_UNSUPPORTED; return false; }
  return true;
}

// dims: local extents.  Not a slab: sd = -1.  Slab: dims[sd] = n_int + 2, gdims = global extents, off = global coordinate of
// the slab's first own layer (common.cuh, Geom).
Geom make_geom(int D, const int* dims, int sd = -1, const int* gdims = nullptr, int off = 0) {
  Geom g;
  memset(&g, 0, sizeof(g));
  g.D = D;
  uint64_t V = 1, Vi = 1;
  for (int d = 0; d < 4; ++d) {
    g.L[d] = (d < D) ? dims[d] : 1;
    g.Li[d] = (d == sd) ? g.L[d] - 2 : g.L[d];
    V *= g.L[d]; Vi *= g.Li[d];
  }
  g.Lh0 = g.L[0] / 2;
  g.stride[0] = 0; g.stride[1] = g.Lh0; g.stride[2] = g.Lh0 * g.L[1]; g.stride[3] = g.Lh0 * g.L[1] * g.L[2];
  g.V = (uint32_t)V; g.Vh = (uint32_t)(V / 2);
  g.Vh_pad = (g.Vh + 31u) & ~31u;
  g.dLh0 = make_fastdiv((uint32_t)g.Lh0); g.dL1 = make_fastdiv((uint32_t)g.L[1]); g.dL2 = make_fastdiv((uint32_t)g.L[2]);
  g.sd = sd;
  g.Vh_int = (uint32_t)(Vi / 2);
  g.iLh0 = g.dLh0; g.iL1 = make_fastdiv((uint32_t)g.Li[1]); g.iL2 = make_fastdiv((uint32_t)g.Li[2]);
  uint32_t st = 1;
  for (int d = 0; d < 4; ++d) {
    g.lexS[d] = st;
    st *= (uint32_t)((sd >= 0 && d < D) ? gdims[d] : g.L[d]);
  }
  g.lex0 = sd >= 0 ? (uint32_t)off * g.lexS[sd] : 0u;
  return g;
}
inline uint32_t own_sites(const qcd_lattice* L) { return 2u * L->g.Vh_int; }   // V, or the interior of a slab

int check_field(const qcd_lattice* L, const qcd_field_t* f, bool* on) {
  *on = false;
  if (!f || !f->enabled) return QCD_OK;
  if (f->mu < 0 || f->nu >= L->D || f->mu >= f->nu) return fail(QCD_ERR_INVALID_ARG, "field plane must satisfy 0 <= mu < nu < D");
  double s = 0.0;
  for (int c = 0; c < L->Nc; ++c) { if (!std::isfinite(f->theta[c])) return fail(QCD_ERR_INVALID_ARG, "field theta not finite"); s += f->theta[c]; }
  if (std::fabs(s) > 1e-12) return fail(QCD_ERR_INVALID_ARG, "field phases must sum to zero (F in SU(N))");
  *on = true;
  return QCD_OK;
}

FieldArgs make_field_args(const qcd_field_t* f, bool on, int Nc) {
  FieldArgs a;
  memset(&a, 0, sizeof(a));
  a.mu = -1; a.nu = -1;
  for (int c = 0; c < 3; ++c) { a.c[c] = 1.0; a.s[c] = 0.0; }
  if (on) {
    a.mu = f->mu; a.nu = f->nu;
    for (int c = 0; c < Nc; ++c) { a.c[c] = std::cos(f->theta[c]); a.s[c] = std::sin(f->theta[c]); }
  }
  return a;
}

cudaError_t launch_update(qcd_lattice* L, int kind, bool field, const UpdateArgs& a0) {
  UpdateSel s; s.Nc = L->Nc; s.D = L->D; s.precision = L->precision; s.comp = L->comp; s.kind = kind; s.field = field;
  s.meas = a0.meas != nullptr;
  UpdateArgs a = a0;
  a.prev_parity = L->last_parity; a.prev_mu = L->last_mu;
  a.rev = L->alternate_order ? (int)(L->order_toggle & 1u) : 0;
  if (L->push_prev && L->push_next) {
    int nreal, vb, np;
    plane_params(L->Nc, L->precision, L->comp, &nreal, &vb, &np);
    qcd_lattice* T[2] = {L->push_prev, L->push_next};
    const int sd = L->g.sd, n_int = L->g.Li[sd];
    a.hp.on = 1; a.hp.last = n_int - 1;
    for (int t = 0; t < 2; ++t) {
      // my first own layer is the previous part's copy "next part's first layer" (its layer n_int'), my last own layer the
      // next part's copy "previous part's last layer" (its layer n_int' + 1)
      a.hp.layer[t] = T[t]->g.Li[sd] + t;
      a.hp.L1[t] = T[t]->g.L[1]; a.hp.L2[t] = T[t]->g.L[2];
      a.hp.base[t] = (char*)T[t]->mem + (size_t)(a.parity * L->D + a.mu) * np * T[t]->g.Vh_pad * (size_t)vb;
    }
  }
  const cudaError_t e = (L->Nc == 2)                ? launch_update_su2(s, L->g, L->mem, a, L->stream)
                        : L->precision == QCD_FP32 ? launch_update_su3_f32(s, L->g, L->mem, a, L->stream)
                                                   : launch_update_su3_f64(s, L->g, L->mem, a, L->stream);
  if (e == cudaSuccess) { L->launches += 1; L->order_toggle ^= 1u; L->last_parity = a.parity; L->last_mu = a.mu; }
  return e;
}

int prof_begin(qcd_lattice* L, int kind, EventPair* ep) {
  if (L->ev_free.empty()) {
    CUDA_TRY(cudaEventCreate(&ep->a)); CUDA_TRY(cudaEventCreate(&ep->b));
  } else { *ep = L->ev_free.back(); L->ev_free.pop_back(); }
  ep->kind = kind; ep->n = 0;
  CUDA_TRY(cudaEventRecord(ep->a, L->stream));
  return QCD_OK;
}
int prof_end(qcd_lattice* L, EventPair* ep, int n) {
  ep->n = n;
  CUDA_TRY(cudaEventRecord(ep->b, L->stream));
  L->ev_used.push_back(*ep);
  return QCD_OK;
}

// bracket: time this single launch with its own event pair (qcd_debug_substep); qcd_sweep brackets whole passes instead
// sizes of the three regions of d_partials
struct MeasLayout {
  uint32_t npl, np_warp, nb_plaq, nb_poly, poly_seg;
  bool boxed;
  size_t off_plaq, off_poly, need;
};
MeasLayout meas_layout(const qcd_lattice* L) {
  MeasLayout m;
  const Geom& g = L->g;
  m.npl = (uint32_t)(L->D * (L->D - 1) / 2);
  // fused measurement: one partial per warp of an update launch; every launch shape has <= Vh_pad/32 + 8 warps (CTAs of
  // <= 256 threads); entries beyond a launch's warps are never written and stay zero from the allocation
  m.np_warp = g.Vh_pad / 32u + 8u;
  m.boxed = (L->D == 4 && g.Lh0 % 8 == 0 && g.Li[1] % 2 == 0 && g.Li[2] % 2 == 0 && g.Li[3] % 2 == 0);
  m.nb_plaq = m.boxed ? 2u * g.Vh_int / 128u : ((g.Vh_int + 127u) / 128u) * 2u;
  // Polyakov kernel: SEG lanes per spatial site, SEG = the largest of 4, 2, 1 that divides Lt
  m.poly_seg = (g.L[L->D - 1] % 4 == 0) ? 4u : (g.L[L->D - 1] % 2 == 0) ? 2u : 1u;
  m.nb_poly = (2u * g.Vh_int / (uint32_t)g.L[L->D - 1] * m.poly_seg + 127u) / 128u;
  m.off_plaq = (size_t)m.npl * m.np_warp;
  m.off_poly = m.off_plaq + (size_t)m.npl * m.nb_plaq;
  m.need = m.off_poly + 2 * (size_t)m.nb_poly;
  return m;
}
int ensure_partials(qcd_lattice* L) {
  const MeasLayout m = meas_layout(L);
  if (L->d_partials && L->partials_cap >= m.need) return QCD_OK;
  if (L->d_partials) CUDA_TRY(cudaFree(L->d_partials));
  L->d_partials = nullptr; L->partials_cap = 0;
  CUDA_TRY(cudaMalloc(&L->d_partials, m.need * sizeof(double)));
  CUDA_TRY(cudaMemsetAsync(L->d_partials, 0, m.need * sizeof(double), L->stream));
  L->partials_cap = m.need;
  return QCD_OK;
}
int plane_index(int D, int nu, int mu) { return nu * D - nu * (nu + 1) / 2 + (mu - nu - 1); }   // nu < mu; order (0,1),(0,2),..

// meas: the fused-measurement form of the sub-step (partials of the planes (nu, mu), nu < mu, into d_partials)
int substep(qcd_lattice* L, double beta, int kind, int hit, int parity, int mu, const qcd_field_t* f, bool field_on, uint8_t* trials,
            bool bracket, bool meas = false) {
  UpdateArgs a;
  memset(&a, 0, sizeof(a));
  if (meas) {
    a.meas = L->d_partials; a.meas_stride = meas_layout(L).np_warp;
    for (int nu = 0; nu < mu && nu < 3; ++nu) a.meas_plane[nu] = plane_index(L->D, nu, mu);
  }
  a.beta = beta; a.inv_c = (double)L->Nc / (2.0 * beta); a.parity = parity; a.mu = mu; a.hit = hit; a.max_trials = L->max_trials;
  a.sweep = L->sweep; a.key0 = (uint32_t)(L->seed & 0xFFFFFFFFull); a.key1 = (uint32_t)(L->seed >> 32);
  a.rk = philox_round_keys(a.key0, a.key1);
  a.trials = trials;
  a.use_bulk = L->bulk_copy ? 1 : 0;
  a.f = make_field_args(f, field_on, L->Nc);
  EventPair ep;
  const bool prof = L->profile && bracket;
  if (prof) { int rc = prof_begin(L, kind, &ep); if (rc != QCD_OK) return rc; }
  const cudaError_t e = launch_update(L, kind, field_on, a);
  if (e != cudaSuccess) {
    if (prof) L->ev_free.push_back(ep);                            // the open pair goes back to the pool
    return fail(QCD_ERR_CUDA, std::string("update kernel launch: ") + cudaGetErrorString(e));
  }
  if (prof) return prof_end(L, &ep, 1);
  return QCD_OK;
}

int drain_profile(qcd_lattice* L) {
  if (L->ev_used.empty()) return QCD_OK;
  CUDA_TRY(cudaStreamSynchronize(L->stream));
  for (auto& ep : L->ev_used) {
    float ms = 0.f;
    CUDA_TRY(cudaEventElapsedTime(&ms, ep.a, ep.b));
    L->prof_ms[ep.kind] += ms; L->prof_n[ep.kind] += (uint64_t)ep.n;
    L->ev_free.push_back(ep);
  }
  L->ev_used.clear();
  return QCD_OK;
}

// ---- template dispatch for the auxiliary kernels
template <typename F> int dispatch(const qcd_lattice* L, F&& f) {
  // f.template operator()<NC, D, R, COMP>()
#define QCD_CASE(NC_, D_)                                                                        \
  if (L->Nc == NC_ && L->D == D_) {                                                               \
    if (L->precision == QCD_FP32) return L->comp ? f.template operator()<NC_, D_, float, (NC_ == 3)>() : f.template operator()<NC_, D_, float, false>(); \
    return L->comp ? f.template operator()<NC_, D_, double, (NC_ == 3)>() : f.template operator()<NC_, D_, double, false>();                            \
  }
  QCD_CASE(2, 2) QCD_CASE(2, 3) QCD_CASE(2, 4) QCD_CASE(3, 2) QCD_CASE(3, 3) QCD_CASE(3, 4)
#undef QCD_CASE
  return fail(QCD_ERR_UNSUPPORTED, "unsupported (Nc, D)");
}

struct InitOp {
  qcd_lattice* L; int hot;
  template <int NC, int D, typename R, bool COMP> int operator()() {
    typedef typename LinkIO<NC, R, COMP>::Vec Vec;
    dim3 grid((L->g.Vh_int + 127) / 128, 2);
    init_kernel<NC, D, R, COMP><<<grid, 128, 0, L->stream>>>(L->g, (Vec*)L->mem, hot, (uint32_t)(L->seed & 0xFFFFFFFFull), (uint32_t)(L->seed >> 32));
    CUDA_TRY(cudaGetLastError());
    L->launches += 1;
    L->last_parity = L->last_mu = -2;                              // every array was written
    return QCD_OK;
  }
};

struct LayoutOp {
  // sites [lex_begin, lex_end) <-> the canonical block starting at `canon` (= the canonical address of site lex_begin)
  qcd_lattice* L; void* canon; bool to_internal; uint32_t lex_begin, lex_end;
  template <int NC, int D, typename R, bool COMP> int operator()() {
    typedef typename LinkIO<NC, R, COMP>::Vec Vec;
    constexpr int BL = LayoutShape<R>::BL;
    dim3 grid((lex_end - lex_begin + BL - 1) / BL, 1);
    if constexpr (NC == 3 && COMP) {
      if (L->exchange_rows01) {
        if (to_internal) layout_kernel<NC, D, R, COMP, true, 2><<<grid, BL, 0, L->stream>>>(L->g, (Vec*)L->mem, (R*)canon, lex_begin, lex_end);
        else layout_kernel<NC, D, R, COMP, false, 2><<<grid, BL, 0, L->stream>>>(L->g, (Vec*)L->mem, (R*)canon, lex_begin, lex_end);
        CUDA_TRY(cudaGetLastError());
        L->launches += 1;
        L->last_parity = L->last_mu = to_internal ? -2 : -1;
        return QCD_OK;
      }
    }
    if (to_internal) layout_kernel<NC, D, R, COMP, true, NC><<<grid, BL, 0, L->stream>>>(L->g, (Vec*)L->mem, (R*)canon, lex_begin, lex_end);
    else layout_kernel<NC, D, R, COMP, false, NC><<<grid, BL, 0, L->stream>>>(L->g, (Vec*)L->mem, (R*)canon, lex_begin, lex_end);
    CUDA_TRY(cudaGetLastError());
    L->launches += 1;
    if (to_internal) L->last_parity = L->last_mu = -2;             // link arrays were written
    else L->last_parity = L->last_mu = -1;                         // a full (non-PDL) kernel boundary: earlier writes are visible
    return QCD_OK;
  }
};

struct MeasureOp {
  // fused: the plaquette partials are already in the fused region of d_partials (written by the MEAS update kernels of the
  // sweep just enqueued); only their second-stage reduction is launched here
  qcd_lattice* L; MeasureField mf; bool want_plaq, want_poly, fused, sums;
  template <int NC, int D, typename R, bool COMP> int operator()() {
    typedef typename LinkIO<NC, R, COMP>::Vec Vec;
    constexpr int NPL = D * (D - 1) / 2;
    int rc = ensure_partials(L);
    if (rc != QCD_OK) return rc;
    const MeasLayout m = meas_layout(L);
    // boxed thread mapping of the plaquette kernel (aux_kernels.cuh, MeasureField): one grid row of V / 128 CTAs
    mf.boxed = m.boxed ? 1 : 0;
    if (mf.boxed) {
      mf.n0 = make_fastdiv((uint32_t)(L->g.Lh0 / 8)); mf.n1 = make_fastdiv((uint32_t)(L->g.Li[1] / 2)); mf.n2 = make_fastdiv((uint32_t)(L->g.Li[2] / 2));
    }
    const uint32_t Vs = own_sites(L) / (uint32_t)L->g.L[D - 1];
    double* pf = L->d_partials;
    double* pp = L->d_partials + m.off_plaq;
    double* pq = L->d_partials + m.off_poly;
    const dim3 plaq_grid = mf.boxed ? dim3(own_sites(L) / 128, 1) : dim3((L->g.Vh_int + 127) / 128, 2);
    // a slab reports SUMS over its own sites (scale 1 / N): the parts' sums are added and divided by the global volume
    const double plaq_scale = sums ? 1.0 / NC : 1.0 / ((double)L->g.V * NC), poly_scale = sums ? 1.0 / NC : 1.0 / ((double)Vs * NC);
    const bool fork = want_plaq && want_poly;
    if (fork) {
      // the Polyakov kernel (one thread per spatial site, bound by the latency of its L_t dependent loads) goes first on a
      // side stream and runs beside the plaquette work; join before the results are read
      if (!L->side) {
        CUDA_TRY(cudaStreamCreateWithFlags(&L->side, cudaStreamNonBlocking));
        CUDA_TRY(cudaEventCreateWithFlags(&L->ev_fork, cudaEventDisableTiming));
        CUDA_TRY(cudaEventCreateWithFlags(&L->ev_join, cudaEventDisableTiming));
      }
      CUDA_TRY(cudaEventRecord(L->ev_fork, L->stream));
      CUDA_TRY(cudaStreamWaitEvent(L->side, L->ev_fork, 0));
    }
    if (want_poly) {
      cudaStream_t ps = fork ? L->side : L->stream;
      if (m.poly_seg == 4) polyakov_kernel<NC, D, R, COMP, 4><<<m.nb_poly, 128, 0, ps>>>(L->g, (const Vec*)L->mem, pq);
      else if (m.poly_seg == 2) polyakov_kernel<NC, D, R, COMP, 2><<<m.nb_poly, 128, 0, ps>>>(L->g, (const Vec*)L->mem, pq);
      else polyakov_kernel<NC, D, R, COMP, 1><<<m.nb_poly, 128, 0, ps>>>(L->g, (const Vec*)L->mem, pq);
      final_reduce_kernel<<<2, 256, 0, ps>>>(pq, m.nb_poly, L->d_results + 8, poly_scale);
      L->launches += 2;
      if (fork) CUDA_TRY(cudaEventRecord(L->ev_join, L->side));
    }
    if (want_plaq) {
      if (fused) {
        final_reduce_kernel<<<NPL, 256, 0, L->stream>>>(pf, m.np_warp, L->d_results, plaq_scale);
        L->launches += 1;
      } else {
        plaquette_kernel<NC, D, R, COMP><<<plaq_grid, 128, 0, L->stream>>>(L->g, (const Vec*)L->mem, mf, pp);
        final_reduce_kernel<<<NPL, 256, 0, L->stream>>>(pp, m.nb_plaq, L->d_results, plaq_scale);
        L->launches += 2;
      }
    }
    if (fork) CUDA_TRY(cudaStreamWaitEvent(L->stream, L->ev_join, 0));
    L->last_parity = L->last_mu = -1;
    CUDA_TRY(cudaGetLastError());
    return QCD_OK;
  }
};

size_t canonical_bytes(const qcd_lattice* L) {
  return (size_t)own_sites(L) * L->D * (L->exchange_rows01 ? 2 : L->Nc) * L->Nc * 2 * (L->precision == QCD_FP32 ? 4 : 8);
}

// ---- probes
template <typename R> __global__ void __launch_bounds__(256) fma_probe_kernel(R* out, int iters, R seed) {
  // 8 independent register-resident FMA chains per thread
  R a0 = seed + threadIdx.x, a1 = a0 + 1, a2 = a0 + 2, a3 = a0 + 3, a4 = a0 + 4, a5 = a0 + 5, a6 = a0 + 6, a7 = a0 + 7;
  const R m = (R)0.999, c = (R)0.001;
  for (int i = 0; i < iters; ++i) {
#pragma unroll
    for (int k = 0; k < 8; ++k) {
      a0 = q_fma(a0, m, c); a1 = q_fma(a1, m, c); a2 = q_fma(a2, m, c); a3 = q_fma(a3, m, c);
      a4 = q_fma(a4, m, c); a5 = q_fma(a5, m, c); a6 = q_fma(a6, m, c); a7 = q_fma(a7, m, c);
    }
  }
  out[blockIdx.x * blockDim.x + threadIdx.x] = a0 + a1 + a2 + a3 + a4 + a5 + a6 + a7;
}

__global__ void __launch_bounds__(256) copy_probe_kernel(const float4* __restrict__ src, float4* __restrict__ dst, size_t n) {
  const size_t stride = (size_t)gridDim.x * blockDim.x;
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) dst[i] = __ldg(src + i);
}

__global__ void hb_math_debug_kernel(const uint32_t* w, size_t n, double* out) {
  const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const double u = uniform64(w[i]);
  double sn, cs;
  hbm::sincos_2pi_uniform32(w[i], &sn, &cs);
  double* o = out + 7 * i;
  o[0] = hbm::log_uniform32(w[i]); o[1] = hbm::cos2_2pi_uniform32(w[i]); o[2] = sn; o[3] = cs;
  o[4] = hbm::sqrt_pos(u); o[5] = hbm::rsqrt(u); o[6] = hbm::rcp(u);
}

__global__ void philox_debug_kernel(const uint32_t* ctr, const uint32_t* key, size_t n, uint32_t* out, int impl) {
  const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  if (impl == 0) {
    Philox4 o = philox4x32_10(ctr[4 * i], ctr[4 * i + 1], ctr[4 * i + 2], ctr[4 * i + 3], key[2 * i], key[2 * i + 1]);
    out[4 * i] = o.x; out[4 * i + 1] = o.y; out[4 * i + 2] = o.z; out[4 * i + 3] = o.w;
  } else {
    uint4 c = make_uint4(ctr[4 * i], ctr[4 * i + 1], ctr[4 * i + 2], ctr[4 * i + 3]);
    uint2 k = make_uint2(key[2 * i], key[2 * i + 1]);
    uint4 o = curand_Philox4x32_10(c, k);
    out[4 * i] = o.x; out[4 * i + 1] = o.y; out[4 * i + 2] = o.z; out[4 * i + 3] = o.w;
  }
}

}  // namespace

// =====================================================================================
extern "C" {

const char* qcd_last_error(void) { return g_err.c_str(); }
const char* qcd_version(void) { return "qcd_b200 0.1 (sm_100a)"; }

size_t qcd_lattice_bytes(int D, const int* dims, int Nc, int precision, unsigned flags) {
  int why;
  if (!valid_shape(D, dims, Nc, precision, flags, &why)) return 0;
  Geom g = make_geom(D, dims);
  int nreal, vb, np;
  plane_params(Nc, precision, (flags & QCD_FLAG_COMPRESS12) != 0, &nreal, &vb, &np);
  return (size_t)2 * D * np * (size_t)g.Vh_pad * vb;
}

// common part of qcd_lattice_create / qcd_slab_create: dims = LOCAL extents (validated by the caller)
static int create_lattice(int D, const int* dims, int Nc, int precision, unsigned flags, int sd, const int* gdims, int off, void* device_mem,
                          size_t bytes, void* cuda_stream, qcd_lattice_t** out) {
  const size_t need = qcd_lattice_bytes(D, dims, Nc, precision, flags);
  if (device_mem) {
    if (bytes < need) return fail(QCD_ERR_INVALID_ARG, "device_mem smaller than the workspace size");
    if (((uintptr_t)device_mem) & 255u) return fail(QCD_ERR_INVALID_ARG, "device_mem must be 256-byte aligned");
  }
  qcd_lattice* L = new qcd_lattice();
  L->D = D; L->Nc = Nc; L->precision = precision; L->flags = flags; L->comp = (flags & QCD_FLAG_COMPRESS12) != 0;
  for (int d = 0; d < 4; ++d) { L->dims[d] = d < D ? dims[d] : 1; L->gdims[d] = d < D ? (gdims ? gdims[d] : dims[d]) : 1; }
  L->slab_off = off;
  L->g = make_geom(D, dims, sd, gdims, off);
  L->bytes = need; L->mem = device_mem; L->owns_mem = false;
  L->stream = (cudaStream_t)cuda_stream;
  L->seed = 0; L->sweep = 0; L->has_links = false; L->max_trials = 10;
  L->debug_trials = false; L->profile = false; L->bulk_copy = false; L->alternate_order = true; L->exchange_rows01 = false;
  L->d_trials = nullptr; L->d_partials = nullptr; L->partials_cap = 0; L->d_results = nullptr; L->h_results = nullptr;
  L->prof_ms[0] = L->prof_ms[1] = 0.0; L->prof_n[0] = L->prof_n[1] = 0; L->launches = 0; L->order_toggle = 0; L->push_prev = L->push_next = nullptr; L->last_parity = L->last_mu = -2; L->d_canon = nullptr;
  L->side = nullptr; L->ev_fork = nullptr; L->ev_join = nullptr;
  cudaError_t e = cudaSuccess;
  if (!device_mem) {
    e = cudaMalloc(&L->mem, need);
    if (e != cudaSuccess) { delete L; return fail(QCD_ERR_ALLOC, std::string("cudaMalloc links: ") + cudaGetErrorString(e)); }
    L->owns_mem = true;
  }
  // d_results: [0,16) the last measurement (planes at 0.., Polyakov at 8,9); [16,48) the accumulator of
  // qcd_measure_accumulate: count, then NQ sums, then NQ sums of squares (NQ <= 9)
  if (e == cudaSuccess) e = cudaMalloc(&L->d_results, 48 * sizeof(double));
  if (e == cudaSuccess) e = cudaMemsetAsync(L->d_results, 0, 48 * sizeof(double), L->stream);
  if (e == cudaSuccess) e = cudaMallocHost(&L->h_results, 48 * sizeof(double));
  // padding lanes of every plane are never read, but keep the workspace defined
  if (e == cudaSuccess) e = cudaMemsetAsync(L->mem, 0, need, L->stream);
  if (e != cudaSuccess) { std::string m = cudaGetErrorString(e); qcd_lattice_destroy(L); return fail(QCD_ERR_CUDA, "create: " + m); }
  *out = L;
  return QCD_OK;
}

int qcd_lattice_create(int D, const int* dims, int Nc, int precision, unsigned flags, void* device_mem, size_t bytes, void* cuda_stream,
                       qcd_lattice_t** out) {
  if (!out) return fail(QCD_ERR_INVALID_ARG, "out is NULL");
  *out = nullptr;
  int why;
  if (!valid_shape(D, dims, Nc, precision, flags, &why))
    return fail(why, why == QCD_ERR_UNSUPPORTED ? "COMPRESS12 needs Nc = 3" : "invalid D / dims (even, >= 2) / Nc / precision / flags");
  return create_lattice(D, dims, Nc, precision, flags, -1, nullptr, 0, device_mem, bytes, cuda_stream, out);
}

// ---- slab of a larger lattice
static int slab_local_dims(int D, const int* gdims, int Nc, int precision, unsigned flags, int offset, int extent, int* ldims) {
  int why;
  if (!valid_shape(D, gdims, Nc, precision, flags, &why)) return fail(why, "invalid global D / dims / Nc / precision / flags");
  if (D < 3) return fail(QCD_ERR_UNSUPPORTED, "a lattice is split along its slowest spatial direction D-2: D >= 3");
  const int sd = D - 2;
  if (extent < 2 || (extent & 1) || offset < 0 || (offset & 1) || offset + extent > gdims[sd])
    return fail(QCD_ERR_INVALID_ARG, "slab offset and extent must be even, extent >= 2, offset + extent <= dims[D-2]");
  for (int d = 0; d < D; ++d) ldims[d] = gdims[d];
  ldims[sd] = extent + 2;
  if (!valid_shape(D, ldims, Nc, precision, flags, &why)) return fail(why, "slab too large for the kernels' indexing");
  return QCD_OK;
}

size_t qcd_slab_bytes(int D, const int* dims, int Nc, int precision, unsigned flags, int offset, int extent) {
  int ld[4];
  if (slab_local_dims(D, dims, Nc, precision, flags, offset, extent, ld) != QCD_OK) return 0;
  return qcd_lattice_bytes(D, ld, Nc, precision, flags);
}

int qcd_slab_create(int D, const int* dims, int Nc, int precision, unsigned flags, int offset, int extent, void* device_mem, size_t bytes,
                    void* cuda_stream, qcd_lattice_t** out) {
  if (!out) return fail(QCD_ERR_INVALID_ARG, "out is NULL");
  *out = nullptr;
  int ld[4];
  int rc = slab_local_dims(D, dims, Nc, precision, flags, offset, extent, ld);
  if (rc != QCD_OK) return rc;
  return create_lattice(D, ld, Nc, precision, flags, D - 2, dims, offset, device_mem, bytes, cuda_stream, out);
}

int qcd_lattice_destroy(qcd_lattice_t* L) {
  if (!L) return QCD_OK;
  cudaStreamSynchronize(L->stream);
  for (auto& ep : L->ev_used) { cudaEventDestroy(ep.a); cudaEventDestroy(ep.b); }
  for (auto& ep : L->ev_free) { cudaEventDestroy(ep.a); cudaEventDestroy(ep.b); }
  if (L->owns_mem && L->mem) cudaFree(L->mem);
  if (L->d_trials) cudaFree(L->d_trials);
  if (L->d_partials) cudaFree(L->d_partials);
  if (L->d_results) cudaFree(L->d_results);
  if (L->h_results) cudaFreeHost(L->h_results);
  if (L->ev_fork) cudaEventDestroy(L->ev_fork);
  if (L->ev_join) cudaEventDestroy(L->ev_join);
  if (L->side) cudaStreamDestroy(L->side);
  if (L->d_canon) cudaFree(L->d_canon);
  delete L;
  return QCD_OK;
}

int qcd_init(qcd_lattice_t* L, int start, uint64_t seed) {
  if (!L) return fail(QCD_ERR_INVALID_ARG, "lattice is NULL");
  if (start != QCD_COLD && start != QCD_HOT) return fail(QCD_ERR_INVALID_ARG, "start must be QCD_COLD or QCD_HOT");
  L->seed = seed; L->sweep = 0;
  InitOp op{L, start == QCD_HOT ? 1 : 0};
  int rc = dispatch(L, op);
  if (rc == QCD_OK) L->has_links = true;
  return rc;
}

// fused: the last pass's (parity 1, mu >= 1) sub-steps run in the fused-measurement form (update.cuh, meas_store)
static int sweep_core(qcd_lattice_t* L, double beta, int n_hb, int n_or, const qcd_field_t* field, bool fused) {
  if (!L) return fail(QCD_ERR_INVALID_ARG, "lattice is NULL");
  if (!L->has_links) return fail(QCD_ERR_STATE, "qcd_sweep before qcd_init / qcd_set_links");
  if (L->g.sd >= 0) return fail(QCD_ERR_UNSUPPORTED, "a slab is swept sub-step by sub-step with halo exchanges in between (qcd_split_sweep)");
  if (!std::isfinite(beta) || beta < 0.0) return fail(QCD_ERR_INVALID_ARG, "beta must be finite and >= 0");
  if (n_hb < 0 || n_or < 0 || n_hb > 65535 || n_or > 65535) return fail(QCD_ERR_INVALID_ARG, "n_hb, n_or must be in 0..65535");
  bool fon;
  int rc = check_field(L, field, &fon);
  if (rc != QCD_OK) return rc;
  if (fused) { rc = ensure_partials(L); if (rc != QCD_OK) return rc; }
  // profiling brackets the run of heatbath launches and the run of overrelaxation launches with one event pair each
  // (3 events per sweep), so the timed stream is not perturbed between kernels
  EventPair ep;
  bool ep_open = false;
  const int n_pass = n_hb + n_or;
  for (int pass = 0; pass < n_pass; ++pass) {
    const int kind = pass < n_hb ? QCD_KIND_HB : QCD_KIND_OR, hit = pass < n_hb ? pass : 0;
    if (L->profile && (pass == 0 || pass == n_hb)) { rc = prof_begin(L, kind, &ep); if (rc != QCD_OK) return rc; ep_open = true; }
    for (int p = 0; p < 2; ++p)
      for (int mu = 0; mu < L->D; ++mu) {
        const bool meas = fused && pass == n_pass - 1 && p == 1 && mu >= 1;
        rc = substep(L, beta, kind, hit, p, mu, field, fon, nullptr, false, meas);
        if (rc != QCD_OK) { if (ep_open) L->ev_free.push_back(ep); return rc; }
      }
    if (L->profile && (pass == n_hb - 1 || pass == n_pass - 1)) {
      rc = prof_end(L, &ep, 2 * L->D * (kind == QCD_KIND_HB ? n_hb : n_or));
      ep_open = false;
      if (rc != QCD_OK) return rc;
    }
  }
  L->sweep += 1;
  return QCD_OK;
}

int qcd_sweep(qcd_lattice_t* L, double beta, int n_hb, int n_or, const qcd_field_t* field) {
  return sweep_core(L, beta, n_hb, n_or, field, false);
}

int qcd_debug_substep(qcd_lattice_t* L, double beta, int kind, int hit, int parity, int mu, const qcd_field_t* field) {
  if (!L) return fail(QCD_ERR_INVALID_ARG, "lattice is NULL");
  if (!L->has_links) return fail(QCD_ERR_STATE, "no links yet");
  if (!std::isfinite(beta) || beta < 0.0) return fail(QCD_ERR_INVALID_ARG, "beta must be finite and >= 0");
  if ((kind != QCD_KIND_HB && kind != QCD_KIND_OR) || hit < 0 || hit > 65535 || (parity != 0 && parity != 1) || mu < 0 || mu >= L->D)
    return fail(QCD_ERR_INVALID_ARG, "bad kind / hit / parity / mu");
  bool fon;
  int rc = check_field(L, field, &fon);
  if (rc != QCD_OK) return rc;
  uint8_t* trials = nullptr;
  if (L->debug_trials && L->g.sd >= 0) return fail(QCD_ERR_UNSUPPORTED, "trial codes are indexed by the global site: not recorded on a slab");
  if (L->debug_trials && kind == QCD_KIND_HB) {
    if (!L->d_trials) CUDA_TRY(cudaMalloc(&L->d_trials, (size_t)L->g.V * 3));
    CUDA_TRY(cudaMemsetAsync(L->d_trials, 0, (size_t)L->g.V * 3, L->stream));
    trials = L->d_trials;
  }
  return substep(L, beta, kind, hit, parity, mu, field, fon, trials, true);
}

int qcd_debug_get_trials(qcd_lattice_t* L, uint8_t* dst, size_t bytes) {
  if (!L || !dst) return fail(QCD_ERR_INVALID_ARG, "NULL argument");
  if (!L->d_trials) return fail(QCD_ERR_STATE, "no trial codes recorded (set QCD_OPT_DEBUG_TRIALS and run a heatbath qcd_debug_substep)");
  if (bytes != (size_t)L->g.V * 3) return fail(QCD_ERR_INVALID_ARG, "bytes must be V*3");
  CUDA_TRY(cudaMemcpyAsync(dst, L->d_trials, bytes, cudaMemcpyDeviceToHost, L->stream));
  CUDA_TRY(cudaStreamSynchronize(L->stream));
  return QCD_OK;
}

// enqueue the measurement kernels (results land in d_results); no synchronisation
static int enqueue_measure(qcd_lattice_t* L, const qcd_field_t* field, bool want_plaq, bool want_poly, bool fused = false) {
  if (!L) return fail(QCD_ERR_INVALID_ARG, "lattice is NULL");
  if (!L->has_links) return fail(QCD_ERR_STATE, "no links yet");
  bool fon;
  int rc = check_field(L, field, &fon);
  if (rc != QCD_OK) return rc;
  MeasureOp op;
  op.L = L; op.want_plaq = want_plaq; op.want_poly = want_poly; op.fused = fused; op.sums = L->g.sd >= 0;
  memset(&op.mf, 0, sizeof(op.mf));
  FieldArgs fa = make_field_args(field, fon, L->Nc);
  op.mf.enabled = fon ? 1 : 0; op.mf.mu = fa.mu; op.mf.nu = fa.nu;
  for (int c = 0; c < 3; ++c) { op.mf.c[c] = fa.c[c]; op.mf.s[c] = fa.s[c]; }
  if (!op.want_plaq && !op.want_poly) return QCD_OK;
  return dispatch(L, op);
}

// accumulator update: one thread per quantity (npl plane plaquettes, Re L, Im L, |L|), fixed order => deterministic
__global__ void accum_kernel(const double* res, double* acc, int npl) {
  const int k = (int)threadIdx.x, nq = npl + 3;
  if (k >= nq) return;
  const double v = k < npl ? res[k] : k == npl ? res[8] : k == npl + 1 ? res[9] : hypot(res[8], res[9]);
  acc[1 + k] += v;
  acc[1 + nq + k] += v * v;
  if (k == 0) acc[0] += 1.0;
}

int qcd_measure_accumulate(qcd_lattice_t* L, const qcd_field_t* field) {
  if (L && L->g.sd >= 0) return fail(QCD_ERR_UNSUPPORTED, "not available on a slab");
  int rc = enqueue_measure(L, field, true, true);
  if (rc != QCD_OK) return rc;
  accum_kernel<<<1, 32, 0, L->stream>>>(L->d_results, L->d_results + 16, L->D * (L->D - 1) / 2);
  L->launches += 1;
  CUDA_TRY(cudaGetLastError());
  return QCD_OK;
}

int qcd_accum_reset(qcd_lattice_t* L) {
  if (!L) return fail(QCD_ERR_INVALID_ARG, "lattice is NULL");
  CUDA_TRY(cudaMemsetAsync(L->d_results + 16, 0, 32 * sizeof(double), L->stream));
  return QCD_OK;
}

int qcd_accum_get(qcd_lattice_t* L, uint64_t* count, double* sum, double* sumsq, int capacity) {
  if (!L || !count || !sum || !sumsq) return fail(QCD_ERR_INVALID_ARG, "NULL argument");
  const int nq = L->D * (L->D - 1) / 2 + 3;
  if (capacity < nq) return fail(QCD_ERR_INVALID_ARG, "capacity must be >= D(D-1)/2 + 3");
  CUDA_TRY(cudaMemcpyAsync(L->h_results + 16, L->d_results + 16, 32 * sizeof(double), cudaMemcpyDeviceToHost, L->stream));
  CUDA_TRY(cudaStreamSynchronize(L->stream));
  *count = (uint64_t)L->h_results[16];
  for (int k = 0; k < nq; ++k) { sum[k] = L->h_results[17 + k]; sumsq[k] = L->h_results[17 + nq + k]; }
  return QCD_OK;
}

// copy the last measurement to the host and hand it out (synchronises)
static int fetch_results(qcd_lattice_t* L, bool want_plaq, double* plaq_total, double* plaq_planes, double* polyakov) {
  CUDA_TRY(cudaMemcpyAsync(L->h_results, L->d_results, 16 * sizeof(double), cudaMemcpyDeviceToHost, L->stream));
  CUDA_TRY(cudaStreamSynchronize(L->stream));
  const int npl = L->D * (L->D - 1) / 2;
  if (want_plaq) {
    double tot = 0.0;
    for (int k = 0; k < npl; ++k) { tot += L->h_results[k]; if (plaq_planes) plaq_planes[k] = L->h_results[k]; }
    if (plaq_total) *plaq_total = tot / npl;
  }
  if (polyakov) { polyakov[0] = L->h_results[8]; polyakov[1] = L->h_results[9]; }
  return QCD_OK;
}

int qcd_measure(qcd_lattice_t* L, const qcd_field_t* field, double* plaq_total, double* plaq_planes, double* polyakov) {
  if (L && L->g.sd >= 0) return fail(QCD_ERR_UNSUPPORTED, "a slab has sums, not means: qcd_slab_measure_sums / qcd_split_measure");
  const bool want_plaq = plaq_total || plaq_planes, want_poly = polyakov != nullptr;
  int rc = enqueue_measure(L, field, want_plaq, want_poly);
  if (rc != QCD_OK) return rc;
  if (!want_plaq && !want_poly) return QCD_OK;
  return fetch_results(L, want_plaq, plaq_total, plaq_planes, polyakov);
}

// working sweep = update + measurement of the new configuration, the plaquette folded into the last pass
int qcd_sweep_measure(qcd_lattice_t* L, double beta, int n_hb, int n_or, const qcd_field_t* field, double* plaq_total, double* plaq_planes,
                      double* polyakov) {
  const bool want_plaq = plaq_total || plaq_planes, want_poly = polyakov != nullptr;
  const bool fused = want_plaq && n_hb + n_or > 0;
  int rc = sweep_core(L, beta, n_hb, n_or, field, fused);
  if (rc != QCD_OK) return rc;
  rc = enqueue_measure(L, field, want_plaq, want_poly, fused);
  if (rc != QCD_OK) return rc;
  if (!want_plaq && !want_poly) return QCD_OK;
  return fetch_results(L, want_plaq, plaq_total, plaq_planes, polyakov);
}

int qcd_sweep_measure_accumulate(qcd_lattice_t* L, double beta, int n_hb, int n_or, const qcd_field_t* field) {
  const bool fused = n_hb + n_or > 0;
  int rc = sweep_core(L, beta, n_hb, n_or, field, fused);
  if (rc != QCD_OK) return rc;
  rc = enqueue_measure(L, field, true, true, fused);
  if (rc != QCD_OK) return rc;
  accum_kernel<<<1, 32, 0, L->stream>>>(L->d_results, L->d_results + 16, L->D * (L->D - 1) / 2);
  CUDA_TRY(cudaGetLastError());
  L->launches += 1;
  return QCD_OK;
}

// Host transfers go through one bounded device staging buffer (STAGE_BYTES, canonical layout) in chunks of whole sites:
// copy and layout kernel alternate on the lattice's stream, which orders the reuse of the buffer.
static const size_t STAGE_BYTES = (size_t)64 << 20;
static int stage_chunks(qcd_lattice_t* L, char* host, bool to_internal) {
  const size_t site_bytes = canonical_bytes(L) / own_sites(L);
  const size_t per = std::max<size_t>(128, (STAGE_BYTES / site_bytes) / 128 * 128);     // sites per chunk, a multiple of every BL
  if (!L->d_canon && cudaMalloc(&L->d_canon, per * site_bytes) != cudaSuccess) {
    L->d_canon = nullptr; cudaGetLastError();
    return fail(QCD_ERR_ALLOC, "staging buffer");
  }
  for (size_t lex0 = 0; lex0 < own_sites(L); lex0 += per) {
    const size_t lex1 = std::min<size_t>(own_sites(L), lex0 + per), n = (lex1 - lex0) * site_bytes;
    if (to_internal) CUDA_TRY(cudaMemcpyAsync(L->d_canon, host + lex0 * site_bytes, n, cudaMemcpyHostToDevice, L->stream));
    LayoutOp op{L, L->d_canon, to_internal, (uint32_t)lex0, (uint32_t)lex1};
    const int rc = dispatch(L, op);
    if (rc != QCD_OK) return rc;
    if (!to_internal) CUDA_TRY(cudaMemcpyAsync(host + lex0 * site_bytes, L->d_canon, n, cudaMemcpyDeviceToHost, L->stream));
  }
  // host memory: the call returns when the host buffer has been read (set) / filled (get), pinned or not
  CUDA_TRY(cudaStreamSynchronize(L->stream));
  return QCD_OK;
}

int qcd_get_links(qcd_lattice_t* L, void* dst, size_t bytes, int dst_is_device) {
  if (!L || !dst) return fail(QCD_ERR_INVALID_ARG, "NULL argument");
  if (!L->has_links) return fail(QCD_ERR_STATE, "no links yet");
  if (bytes != canonical_bytes(L)) return fail(QCD_ERR_INVALID_ARG, "bytes must equal V*D*N*N*2*sizeof(real) (V*D*2*3*2*sizeof(real) with EXCHANGE_ROWS01)");
  if (dst_is_device && ((uintptr_t)dst & 15u)) return fail(QCD_ERR_INVALID_ARG, "device pointer must be 16-byte aligned");
  if (!dst_is_device) return stage_chunks(L, (char*)dst, false);
  LayoutOp op{L, dst, false, 0u, own_sites(L)};
  return dispatch(L, op);
}

int qcd_set_links(qcd_lattice_t* L, const void* src, size_t bytes, int src_is_device) {
  if (!L || !src) return fail(QCD_ERR_INVALID_ARG, "NULL argument");
  if (bytes != canonical_bytes(L)) return fail(QCD_ERR_INVALID_ARG, "bytes must equal V*D*N*N*2*sizeof(real)");
  if (src_is_device && ((uintptr_t)src & 15u)) return fail(QCD_ERR_INVALID_ARG, "device pointer must be 16-byte aligned");
  int rc;
  if (!src_is_device) {
    rc = stage_chunks(L, (char*)const_cast<void*>(src), true);
  } else {
    LayoutOp op{L, const_cast<void*>(src), true, 0u, own_sites(L)};
    rc = dispatch(L, op);
  }
  if (rc == QCD_OK) L->has_links = true;
  return rc;
}

int qcd_get_sweep_counter(qcd_lattice_t* L, uint32_t* out) {
  if (!L || !out) return fail(QCD_ERR_INVALID_ARG, "NULL argument");
  *out = L->sweep; return QCD_OK;
}
int qcd_set_sweep_counter(qcd_lattice_t* L, uint32_t v) {
  if (!L) return fail(QCD_ERR_INVALID_ARG, "NULL argument");
  L->sweep = v; return QCD_OK;
}
int qcd_get_seed(qcd_lattice_t* L, uint64_t* out) {
  if (!L || !out) return fail(QCD_ERR_INVALID_ARG, "NULL argument");
  *out = L->seed; return QCD_OK;
}
int qcd_set_seed(qcd_lattice_t* L, uint64_t seed) {
  if (!L) return fail(QCD_ERR_INVALID_ARG, "NULL argument");
  L->seed = seed; return QCD_OK;
}

int qcd_set_option(qcd_lattice_t* L, int key, int value) {
  if (!L) return fail(QCD_ERR_INVALID_ARG, "NULL argument");
  switch (key) {
    case QCD_OPT_KP_MAX_TRIALS:
      if (value < 1 || value > 127) return fail(QCD_ERR_INVALID_ARG, "KP_MAX_TRIALS must be in 1..127");
      L->max_trials = value; return QCD_OK;
    case QCD_OPT_DEBUG_TRIALS: L->debug_trials = value != 0; return QCD_OK;
    case QCD_OPT_PROFILE: L->profile = value != 0; return QCD_OK;
    case QCD_OPT_BULK_COPY: L->bulk_copy = value != 0; return QCD_OK;
    case QCD_OPT_ALTERNATE_ORDER: L->alternate_order = value != 0; return QCD_OK;
    case QCD_OPT_EXCHANGE_ROWS01:
      if (value != 0 && !(L->Nc == 3 && L->comp)) return fail(QCD_ERR_UNSUPPORTED, "EXCHANGE_ROWS01 needs SU(3) with COMPRESS12");
      if ((value != 0) != L->exchange_rows01 && L->d_canon) { cudaFree(L->d_canon); L->d_canon = nullptr; }   // chunk geometry changes
      L->exchange_rows01 = value != 0; return QCD_OK;
  }
  return fail(QCD_ERR_INVALID_ARG, "unknown option key");
}

int qcd_get_profile(qcd_lattice_t* L, int kind, double* total_ms, uint64_t* launches) {
  if (!L || (kind != 0 && kind != 1)) return fail(QCD_ERR_INVALID_ARG, "bad argument");
  int rc = drain_profile(L);
  if (rc != QCD_OK) return rc;
  if (total_ms) *total_ms = L->prof_ms[kind];
  if (launches) *launches = L->prof_n[kind];
  return QCD_OK;
}
int qcd_reset_profile(qcd_lattice_t* L) {
  if (!L) return fail(QCD_ERR_INVALID_ARG, "NULL argument");
  int rc = drain_profile(L);
  L->prof_ms[0] = L->prof_ms[1] = 0.0; L->prof_n[0] = L->prof_n[1] = 0;
  return rc;
}
int qcd_get_launch_count(qcd_lattice_t* L, uint64_t* out) {
  if (!L || !out) return fail(QCD_ERR_INVALID_ARG, "NULL argument");
  *out = L->launches; return QCD_OK;
}

int qcd_debug_philox(const uint32_t* ctr, const uint32_t* key, size_t n, uint32_t* out, int impl) {
  if (!ctr || !key || !out || (impl != 0 && impl != 1)) return fail(QCD_ERR_INVALID_ARG, "bad argument");
  if (n == 0) return QCD_OK;
  uint32_t *dc = nullptr, *dk = nullptr, *dout = nullptr;
  cudaError_t e = cudaMalloc(&dc, n * 16);
  if (e == cudaSuccess) e = cudaMalloc(&dk, n * 8);
  if (e == cudaSuccess) e = cudaMalloc(&dout, n * 16);
  if (e == cudaSuccess) e = cudaMemcpy(dc, ctr, n * 16, cudaMemcpyHostToDevice);
  if (e == cudaSuccess) e = cudaMemcpy(dk, key, n * 8, cudaMemcpyHostToDevice);
  if (e == cudaSuccess) {
    philox_debug_kernel<<<(unsigned)((n + 255) / 256), 256>>>(dc, dk, n, dout, impl);
    e = cudaGetLastError();
  }
  if (e == cudaSuccess) e = cudaMemcpy(out, dout, n * 16, cudaMemcpyDeviceToHost);
  cudaFree(dc); cudaFree(dk); cudaFree(dout);
  if (e != cudaSuccess) return fail(QCD_ERR_CUDA, std::string("debug_philox: ") + cudaGetErrorString(e));
  return QCD_OK;
}

int qcd_debug_hb_math(const uint32_t* words, size_t n, double* out) {
  if (!words || !out) return fail(QCD_ERR_INVALID_ARG, "NULL argument");
  if (n == 0) return QCD_OK;
  uint32_t* dw = nullptr;
  double* dout = nullptr;
  cudaError_t e = cudaMalloc(&dw, n * 4);
  if (e == cudaSuccess) e = cudaMalloc(&dout, n * 56);
  if (e == cudaSuccess) e = cudaMemcpy(dw, words, n * 4, cudaMemcpyHostToDevice);
  if (e == cudaSuccess) {
    hb_math_debug_kernel<<<(unsigned)((n + 255) / 256), 256>>>(dw, n, dout);
    e = cudaGetLastError();
  }
  if (e == cudaSuccess) e = cudaMemcpy(out, dout, n * 56, cudaMemcpyDeviceToHost);
  cudaFree(dw); cudaFree(dout);
  if (e != cudaSuccess) return fail(QCD_ERR_CUDA, std::string("debug_hb_math: ") + cudaGetErrorString(e));
  return QCD_OK;
}

int qcd_probe_fma_tflops(int precision, double* tflops) {
  if (!tflops || (precision != QCD_FP32 && precision != QCD_FP64)) return fail(QCD_ERR_INVALID_ARG, "bad argument");
  int dev = 0, sms = 0;
  CUDA_TRY(cudaGetDevice(&dev));
  CUDA_TRY(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
  const int blocks = sms * 8, threads = 256, iters = 4096;
  void* buf = nullptr;
  CUDA_TRY(cudaMalloc(&buf, (size_t)blocks * threads * 8));
  cudaEvent_t a, b;
  cudaEventCreate(&a); cudaEventCreate(&b);
  double best = 0.0;
  for (int rep = 0; rep < 5; ++rep) {
    cudaEventRecord(a);
    if (precision == QCD_FP32) fma_probe_kernel<float><<<blocks, threads>>>((float*)buf, iters, 1.0f);
    else fma_probe_kernel<double><<<blocks, threads>>>((double*)buf, iters, 1.0);
    cudaEventRecord(b);
    cudaError_t e = cudaEventSynchronize(b);
    if (e != cudaSuccess) { cudaFree(buf); return fail(QCD_ERR_CUDA, std::string("fma probe: ") + cudaGetErrorString(e)); }
    float ms = 0.f;
    cudaEventElapsedTime(&ms, a, b);
    const double flops = 2.0 * 64.0 * iters * (double)blocks * threads;
    if (rep > 0) best = std::max(best, flops / (ms * 1e-3) / 1e12);
  }
  cudaEventDestroy(a); cudaEventDestroy(b); cudaFree(buf);
  *tflops = best;
  return QCD_OK;
}

int qcd_probe_copy_gbs(size_t bytes, int reps, double* gbs) {
  if (!gbs || bytes < 16 || reps < 1) return fail(QCD_ERR_INVALID_ARG, "bad argument");
  int dev = 0, sms = 0;
  CUDA_TRY(cudaGetDevice(&dev));
  CUDA_TRY(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
  const size_t n = bytes / 16;
  float4 *src = nullptr, *dst = nullptr;
  CUDA_TRY(cudaMalloc(&src, n * 16));
  cudaError_t e = cudaMalloc(&dst, n * 16);
  if (e != cudaSuccess) { cudaFree(src); return fail(QCD_ERR_ALLOC, "copy probe alloc"); }
  cudaMemset(src, 1, n * 16); cudaMemset(dst, 0, n * 16);
  cudaEvent_t a, b;
  cudaEventCreate(&a); cudaEventCreate(&b);
  double best = 0.0;
  for (int rep = 0; rep < reps + 1; ++rep) {
    cudaEventRecord(a);
    copy_probe_kernel<<<sms * 16, 256>>>(src, dst, n);
    cudaEventRecord(b);
    e = cudaEventSynchronize(b);
    if (e != cudaSuccess) break;
    float ms = 0.f;
    cudaEventElapsedTime(&ms, a, b);
    if (rep > 0) best = std::max(best, 2.0 * n * 16 / (ms * 1e-3) / 1e9);
  }
  cudaEventDestroy(a); cudaEventDestroy(b); cudaFree(src); cudaFree(dst);
  if (e != cudaSuccess) return fail(QCD_ERR_CUDA, std::string("copy probe: ") + cudaGetErrorString(e));
  *gbs = best;
  return QCD_OK;
}


// =====================================================================================
// Slabs and the split driver (sec 4: the lattice divided into parts along one
// spatial direction, boundary values exchanged between the parts)
// =====================================================================================
}  // extern "C"

namespace {

struct HaloOp {
  // mode 0: layer `src_layer` of S -> contiguous buffer; 1: buffer -> layer `dst_layer` of T; 2: layer of S -> layer of T
  int mode; qcd_lattice* S; int src_layer; qcd_lattice* T; int dst_layer; void* buf; int parity, mu; cudaStream_t st;
  template <int NC, int D, typename R, bool COMP> int operator()() {
    typedef typename LinkIO<NC, R, COMP>::Vec Vec;
    constexpr int NP = LinkIO<NC, R, COMP>::T::NP;
    const qcd_lattice* E = mode == 1 ? T : S;
    const uint32_t count = E->g.Vh / (uint32_t)E->g.L[E->g.sd];          // half-indices of one layer
    const dim3 grid((count + 127) / 128);
    if (mode == 0) halo_kernel<Vec, NP, 0><<<grid, 128, 0, st>>>(S->g, (const Vec*)S->mem, src_layer, S->g, (Vec*)buf, 0, parity, mu, D, count);
    else if (mode == 1) halo_kernel<Vec, NP, 1><<<grid, 128, 0, st>>>(T->g, (const Vec*)buf, 0, T->g, (Vec*)T->mem, dst_layer, parity, mu, D, count);
    else halo_kernel<Vec, NP, 2><<<grid, 128, 0, st>>>(S->g, (const Vec*)S->mem, src_layer, T->g, (Vec*)T->mem, dst_layer, parity, mu, D, count);
    CUDA_TRY(cudaGetLastError());
    return QCD_OK;
  }
};

struct HaloPairOp {
  qcd_lattice* S; qcd_lattice* Tprev; int dst_prev; qcd_lattice* Tnext; int dst_next; int last_layer; int parity, mu; cudaStream_t st;
  template <int NC, int D, typename R, bool COMP> int operator()() {
    typedef typename LinkIO<NC, R, COMP>::Vec Vec;
    constexpr int NP = LinkIO<NC, R, COMP>::T::NP;
    const uint32_t count = S->g.Vh / (uint32_t)S->g.L[S->g.sd];          // half-indices of one layer
    HaloTarget<Vec> t0{Tprev->g, (Vec*)Tprev->mem, 0, dst_prev}, t1{Tnext->g, (Vec*)Tnext->mem, last_layer, dst_next};
    CUDA_TRY(launch_pdl(halo_pair_kernel<Vec, NP>, dim3((count + 127) / 128, 2), dim3(128), 0, st, S->g, (const Vec*)S->mem, t0, t1, parity, mu,
                        (int)D, count));
    return QCD_OK;
  }
};

struct DeviceGuard {
  int prev;
  explicit DeviceGuard(int dev) : prev(-1) { cudaGetDevice(&prev); if (dev != prev) cudaSetDevice(dev); else prev = -1; }
  ~DeviceGuard() { if (prev >= 0) cudaSetDevice(prev); }
};

}  // namespace

struct qcd_split {
  int D, Nc, precision, n;
  unsigned flags;
  int dims[4];
  std::vector<qcd_lattice*> part;
  std::vector<int> dev, off, ext;
  std::vector<cudaStream_t> stream;
  std::vector<cudaEvent_t> ev_upd, ev_halo;    // per part: its last update kernel done / its last halo writes done
  uint32_t sweep;
};

namespace {

// refresh, in both neighbours, the copies of part k's boundary layers of the (parity, mu) array.  Part k's stream does the
// copies after (i) its own update (stream order) and (ii) the neighbours' updates of the same sub-step (they may still read
// the old copies); the neighbours' next launches wait for ev_halo[k].
int split_push_halos(qcd_split* S, int k, int parity, int mu) {
  DeviceGuard dg(S->dev[k]);
  const int prev = (k + S->n - 1) % S->n, next = (k + 1) % S->n;
  qcd_lattice* P = S->part[k];
  if (prev != k) CUDA_TRY(cudaStreamWaitEvent(S->stream[k], S->ev_upd[prev], 0));
  if (next != k && next != prev) CUDA_TRY(cudaStreamWaitEvent(S->stream[k], S->ev_upd[next], 0));
  // first own layer -> the previous part's "next" copy (its layer n_int); last own layer -> the next part's "previous" copy
  HaloPairOp op{P, S->part[prev], S->ext[prev], S->part[next], S->ext[next] + 1, S->ext[k] - 1, parity, mu, S->stream[k]};
  const int rc = dispatch(P, op);
  if (rc != QCD_OK) return rc;
  P->launches += 1;
  CUDA_TRY(cudaEventRecord(S->ev_halo[k], S->stream[k]));
  return QCD_OK;
}

// every part waits for the halo writes of its neighbours before its next launch
int split_wait_halos(qcd_split* S, int k) {
  DeviceGuard dg(S->dev[k]);
  const int prev = (k + S->n - 1) % S->n, next = (k + 1) % S->n;
  if (prev != k) CUDA_TRY(cudaStreamWaitEvent(S->stream[k], S->ev_halo[prev], 0));
  if (next != k && next != prev) CUDA_TRY(cudaStreamWaitEvent(S->stream[k], S->ev_halo[next], 0));
  return QCD_OK;
}

int split_refresh_all(qcd_split* S) {
  for (int k = 0; k < S->n; ++k) { DeviceGuard dg(S->dev[k]); CUDA_TRY(cudaEventRecord(S->ev_upd[k], S->stream[k])); }
  for (int p = 0; p < 2; ++p)
    for (int mu = 0; mu < S->D; ++mu)
      for (int k = 0; k < S->n; ++k) { int rc = split_push_halos(S, k, p, mu); if (rc != QCD_OK) return rc; }
  for (int k = 0; k < S->n; ++k) { int rc = split_wait_halos(S, k); if (rc != QCD_OK) return rc; }
  return QCD_OK;
}

// Every part's stream waits for the last update kernels of both neighbours (ev_upd).  A part's halo layers are written by its
// NEIGHBOURS' update kernels, on their streams: whatever reads them next on the part's own stream -- the next sub-step's
// kernel, or a measurement -- has to come behind this wait.
int split_wait_updates(qcd_split* S) {
  for (int k = 0; k < S->n; ++k) {
    DeviceGuard dg(S->dev[k]);
    const int prev = (k + S->n - 1) % S->n, next = (k + 1) % S->n;
    if (prev != k) CUDA_TRY(cudaStreamWaitEvent(S->stream[k], S->ev_upd[prev], 0));
    if (next != k && next != prev) CUDA_TRY(cudaStreamWaitEvent(S->stream[k], S->ev_upd[next], 0));
  }
  return QCD_OK;
}

// One sub-step of every part.  The update kernels write the boundary layers of the array they update into the neighbouring
// parts themselves (HaloPush): there is no separate exchange step, and one event per part and sub-step orders everything --
// a part's kernel of sub-step s+1 starts after both neighbours' kernels of sub-step s, which (i) have then written its halo
// copies of the array they updated and (ii) no longer read the halo copies it is about to overwrite there.  (A sub-step
// reads the array it updates only at its own sites, so kernels of the SAME sub-step never conflict.)
int split_substep(qcd_split* S, double beta, int kind, int hit, int parity, int mu, const qcd_field_t* field) {
  int rc0 = split_wait_updates(S);                                   // the events of the previous sub-step
  if (rc0 != QCD_OK) return rc0;
  for (int k = 0; k < S->n; ++k) {
    DeviceGuard dg(S->dev[k]);
    qcd_lattice* P = S->part[k];
    P->sweep = S->sweep;
    bool fon;
    int rc = check_field(P, field, &fon);
    if (rc != QCD_OK) return rc;
    rc = substep(P, beta, kind, hit, parity, mu, field, fon, nullptr, false);
    if (rc != QCD_OK) return rc;
  }
  for (int k = 0; k < S->n; ++k) { DeviceGuard dg(S->dev[k]); CUDA_TRY(cudaEventRecord(S->ev_upd[k], S->stream[k])); }
  return QCD_OK;
}

// sites per layer of the split direction below it (contiguous run in lex order) and number of such runs
void split_runs(const qcd_split* S, size_t* run_sites, size_t* n_runs) {
  const int sd = S->D - 2;
  size_t lo = 1, hi = 1;
  for (int d = 0; d < sd; ++d) lo *= (size_t)S->dims[d];
  for (int d = sd + 1; d < S->D; ++d) hi *= (size_t)S->dims[d];
  *run_sites = lo; *n_runs = hi;
}

}  // namespace

extern "C" {

size_t qcd_slab_halo_bytes(qcd_lattice_t* L) {
  if (!L || L->g.sd < 0) return 0;
  int nreal, vb, np;
  plane_params(L->Nc, L->precision, L->comp, &nreal, &vb, &np);
  return (size_t)(L->g.Vh / (uint32_t)L->g.L[L->g.sd]) * np * vb;
}

int qcd_slab_halo_pack(qcd_lattice_t* L, int parity, int mu, int side, void* device_buf, size_t bytes) {
  if (!L || !device_buf) return fail(QCD_ERR_INVALID_ARG, "NULL argument");
  if (L->g.sd < 0) return fail(QCD_ERR_STATE, "not a slab");
  if ((parity != 0 && parity != 1) || mu < 0 || mu >= L->D || (side != 0 && side != 1)) return fail(QCD_ERR_INVALID_ARG, "bad parity / mu / side");
  if (bytes != qcd_slab_halo_bytes(L) || ((uintptr_t)device_buf & 15u)) return fail(QCD_ERR_INVALID_ARG, "buffer must hold qcd_slab_halo_bytes() bytes, 16-byte aligned");
  HaloOp op{0, L, side == 0 ? 0 : L->g.Li[L->g.sd] - 1, L, 0, device_buf, parity, mu, L->stream};
  int rc = dispatch(L, op);
  if (rc == QCD_OK) L->launches += 1;
  return rc;
}

int qcd_slab_halo_unpack(qcd_lattice_t* L, int parity, int mu, int side, const void* device_buf, size_t bytes) {
  if (!L || !device_buf) return fail(QCD_ERR_INVALID_ARG, "NULL argument");
  if (L->g.sd < 0) return fail(QCD_ERR_STATE, "not a slab");
  if ((parity != 0 && parity != 1) || mu < 0 || mu >= L->D || (side != 0 && side != 1)) return fail(QCD_ERR_INVALID_ARG, "bad parity / mu / side");
  if (bytes != qcd_slab_halo_bytes(L) || ((uintptr_t)device_buf & 15u)) return fail(QCD_ERR_INVALID_ARG, "buffer must hold qcd_slab_halo_bytes() bytes, 16-byte aligned");
  const int n = L->g.Li[L->g.sd];
  HaloOp op{1, L, 0, L, side == 0 ? n + 1 : n, const_cast<void*>(device_buf), parity, mu, L->stream};
  int rc = dispatch(L, op);
  // the halo layers of the (parity, mu) array were written: an update kernel may not fetch that array early
  if (rc == QCD_OK) { L->launches += 1; if (!(L->last_parity == parity && L->last_mu == mu)) L->last_parity = L->last_mu = -2; }
  return rc;
}

int qcd_slab_measure_sums(qcd_lattice_t* L, const qcd_field_t* field, double* plaq_sums, double* polyakov_sum) {
  if (!L) return fail(QCD_ERR_INVALID_ARG, "lattice is NULL");
  if (L->g.sd < 0) return fail(QCD_ERR_STATE, "not a slab");
  const bool want_plaq = plaq_sums != nullptr, want_poly = polyakov_sum != nullptr;
  int rc = enqueue_measure(L, field, want_plaq, want_poly);
  if (rc != QCD_OK) return rc;
  if (!want_plaq && !want_poly) return QCD_OK;
  CUDA_TRY(cudaMemcpyAsync(L->h_results, L->d_results, 16 * sizeof(double), cudaMemcpyDeviceToHost, L->stream));
  CUDA_TRY(cudaStreamSynchronize(L->stream));
  if (want_plaq) for (int k = 0; k < L->D * (L->D - 1) / 2; ++k) plaq_sums[k] = L->h_results[k];
  if (want_poly) { polyakov_sum[0] = L->h_results[8]; polyakov_sum[1] = L->h_results[9]; }
  return QCD_OK;
}

int qcd_split_create(int D, const int* dims, int Nc, int precision, unsigned flags, int n_parts, const int* extents, const int* devices,
                     qcd_split_t** out) {
  if (!out) return fail(QCD_ERR_INVALID_ARG, "out is NULL");
  *out = nullptr;
  int why;
  if (!valid_shape(D, dims, Nc, precision, flags, &why)) return fail(why, "invalid D / dims / Nc / precision / flags");
  if (D < 3) return fail(QCD_ERR_UNSUPPORTED, "a lattice is split along its slowest spatial direction D-2: D >= 3");
  const int sd = D - 2;
  if (n_parts < 1 || 2 * n_parts > dims[sd]) return fail(QCD_ERR_INVALID_ARG, "n_parts must be in 1 .. dims[D-2] / 2");
  qcd_split* S = new qcd_split();
  S->D = D; S->Nc = Nc; S->precision = precision; S->flags = flags; S->n = n_parts; S->sweep = 0;
  for (int d = 0; d < 4; ++d) S->dims[d] = d < D ? dims[d] : 1;
  int cur = 0;
  cudaGetDevice(&cur);
  int sum = 0;
  for (int k = 0; k < n_parts; ++k) {
    // default: parts as equal as even extents allow (in general the parts are unequal)
    int e = extents ? extents[k] : 2 * ((dims[sd] / 2) / n_parts + (k < (dims[sd] / 2) % n_parts ? 1 : 0));
    S->off.push_back(sum); S->ext.push_back(e); S->dev.push_back(devices ? devices[k] : cur);
    sum += e;
    if (e < 2 || (e & 1)) { delete S; return fail(QCD_ERR_INVALID_ARG, "part extents must be even and >= 2"); }
  }
  if (sum != dims[sd]) { delete S; return fail(QCD_ERR_INVALID_ARG, "part extents must add up to dims[D-2]"); }
  int rc = QCD_OK;
  for (int k = 0; k < n_parts && rc == QCD_OK; ++k) {
    DeviceGuard dg(S->dev[k]);
    cudaStream_t st = nullptr;
    cudaEvent_t eu = nullptr, eh = nullptr;
    if (cudaStreamCreateWithFlags(&st, cudaStreamNonBlocking) != cudaSuccess || cudaEventCreateWithFlags(&eu, cudaEventDisableTiming) != cudaSuccess ||
        cudaEventCreateWithFlags(&eh, cudaEventDisableTiming) != cudaSuccess) {
      rc = fail(QCD_ERR_CUDA, std::string("split: stream / event creation: ") + cudaGetErrorString(cudaGetLastError()));
    }
    S->stream.push_back(st); S->ev_upd.push_back(eu); S->ev_halo.push_back(eh);
    qcd_lattice* P = nullptr;
    if (rc == QCD_OK) rc = qcd_slab_create(D, dims, Nc, precision, flags, S->off[k], S->ext[k], nullptr, 0, st, &P);
    S->part.push_back(P);
  }
  // parts on different devices write each other's halo layers directly: peer access in both directions
  for (int k = 0; k < n_parts && rc == QCD_OK; ++k) {
    const int nb[2] = {(k + n_parts - 1) % n_parts, (k + 1) % n_parts};
    for (int t = 0; t < 2 && rc == QCD_OK; ++t) {
      if (S->dev[nb[t]] == S->dev[k]) continue;
      DeviceGuard dg(S->dev[k]);
      int can = 0;
      cudaDeviceCanAccessPeer(&can, S->dev[k], S->dev[nb[t]]);
      if (!can) { rc = fail(QCD_ERR_UNSUPPORTED, "split: no peer access between the devices of neighbouring parts"); break; }
      cudaError_t e = cudaDeviceEnablePeerAccess(S->dev[nb[t]], 0);
      if (e != cudaSuccess && e != cudaErrorPeerAccessAlreadyEnabled) rc = fail(QCD_ERR_CUDA, std::string("cudaDeviceEnablePeerAccess: ") + cudaGetErrorString(e));
      cudaGetLastError();
    }
  }
  if (rc != QCD_OK) { std::string m = g_err; qcd_split_destroy(S); g_err = m; return rc; }
  // the update kernels of a part write its boundary layers into the neighbours' copies (HaloPush)
  for (int k = 0; k < n_parts; ++k) {
    S->part[k]->push_prev = S->part[(k + n_parts - 1) % n_parts];
    S->part[k]->push_next = S->part[(k + 1) % n_parts];
  }
  *out = S;
  return QCD_OK;
}

int qcd_split_destroy(qcd_split_t* S) {
  if (!S) return QCD_OK;
  // a neighbour's update kernel may still be storing into a part's halo layers (from another stream, or another device,
  // which cudaFree of this device's memory does not wait for): drain every stream before anything is freed
  for (size_t k = 0; k < S->stream.size(); ++k) {
    DeviceGuard dg(S->dev[k]);
    if (S->stream[k]) cudaStreamSynchronize(S->stream[k]);
  }
  for (size_t k = 0; k < S->part.size(); ++k) {
    DeviceGuard dg(S->dev[k]);
    if (S->part[k]) qcd_lattice_destroy(S->part[k]);
    if (k < S->ev_upd.size() && S->ev_upd[k]) cudaEventDestroy(S->ev_upd[k]);
    if (k < S->ev_halo.size() && S->ev_halo[k]) cudaEventDestroy(S->ev_halo[k]);
    if (k < S->stream.size() && S->stream[k]) cudaStreamDestroy(S->stream[k]);
  }
  delete S;
  return QCD_OK;
}

int qcd_split_parts(qcd_split_t* S, int* n_parts, int* offsets, int* extents, int capacity) {
  if (!S || !n_parts) return fail(QCD_ERR_INVALID_ARG, "NULL argument");
  *n_parts = S->n;
  if (offsets || extents) {
    if (capacity < S->n) return fail(QCD_ERR_INVALID_ARG, "capacity < number of parts");
    for (int k = 0; k < S->n; ++k) { if (offsets) offsets[k] = S->off[k]; if (extents) extents[k] = S->ext[k]; }
  }
  return QCD_OK;
}

int qcd_split_halo_bytes(qcd_split_t* S, size_t* per_substep) {
  if (!S || !per_substep) return fail(QCD_ERR_INVALID_ARG, "NULL argument");
  *per_substep = 2 * (size_t)S->n * qcd_slab_halo_bytes(S->part[0]);     // two boundary layers per part and sub-step
  return QCD_OK;
}

int qcd_split_init(qcd_split_t* S, int start, uint64_t seed) {
  if (!S) return fail(QCD_ERR_INVALID_ARG, "split lattice is NULL");
  for (int k = 0; k < S->n; ++k) {
    DeviceGuard dg(S->dev[k]);
    int rc = qcd_init(S->part[k], start, seed);
    if (rc != QCD_OK) return rc;
  }
  S->sweep = 0;
  return split_refresh_all(S);
}

int qcd_split_substep(qcd_split_t* S, double beta, int kind, int hit, int parity, int mu, const qcd_field_t* field) {
  if (!S) return fail(QCD_ERR_INVALID_ARG, "split lattice is NULL");
  if (!S->part[0]->has_links) return fail(QCD_ERR_STATE, "no links yet");
  if (!std::isfinite(beta) || beta < 0.0) return fail(QCD_ERR_INVALID_ARG, "beta must be finite and >= 0");
  if ((kind != QCD_KIND_HB && kind != QCD_KIND_OR) || hit < 0 || hit > 65535 || (parity != 0 && parity != 1) || mu < 0 || mu >= S->D)
    return fail(QCD_ERR_INVALID_ARG, "bad kind / hit / parity / mu");
  return split_substep(S, beta, kind, hit, parity, mu, field);
}

int qcd_split_sweep(qcd_split_t* S, double beta, int n_hb, int n_or, const qcd_field_t* field) {
  if (!S) return fail(QCD_ERR_INVALID_ARG, "split lattice is NULL");
  if (!S->part[0]->has_links) return fail(QCD_ERR_STATE, "qcd_split_sweep before qcd_split_init / qcd_split_set_links");
  if (!std::isfinite(beta) || beta < 0.0) return fail(QCD_ERR_INVALID_ARG, "beta must be finite and >= 0");
  if (n_hb < 0 || n_or < 0 || n_hb > 65535 || n_or > 65535) return fail(QCD_ERR_INVALID_ARG, "n_hb, n_or must be in 0..65535");
  for (int pass = 0; pass < n_hb + n_or; ++pass) {
    const int kind = pass < n_hb ? QCD_KIND_HB : QCD_KIND_OR, hit = pass < n_hb ? pass : 0;
    for (int p = 0; p < 2; ++p)
      for (int mu = 0; mu < S->D; ++mu) {
        int rc = split_substep(S, beta, kind, hit, p, mu, field);
        if (rc != QCD_OK) return rc;
      }
  }
  S->sweep += 1;
  for (int k = 0; k < S->n; ++k) S->part[k]->sweep = S->sweep;
  return QCD_OK;
}

int qcd_split_measure(qcd_split_t* S, const qcd_field_t* field, double* plaq_total, double* plaq_planes, double* polyakov) {
  if (!S) return fail(QCD_ERR_INVALID_ARG, "split lattice is NULL");
  const int npl = S->D * (S->D - 1) / 2;
  double ps[8] = {0, 0, 0, 0, 0, 0, 0, 0}, pl[2] = {0, 0};
  const bool want_plaq = plaq_total || plaq_planes;
  // the plaquette kernel of a part reads its halo copies, which the neighbours' last update kernels may still be writing
  int rcw = split_wait_updates(S);
  if (rcw != QCD_OK) return rcw;
  // enqueue on every part first, then collect: the parts measure concurrently
  for (int k = 0; k < S->n; ++k) {
    DeviceGuard dg(S->dev[k]);
    int rc = enqueue_measure(S->part[k], field, want_plaq, polyakov != nullptr);
    if (rc != QCD_OK) return rc;
    qcd_lattice* P = S->part[k];
    CUDA_TRY(cudaMemcpyAsync(P->h_results, P->d_results, 16 * sizeof(double), cudaMemcpyDeviceToHost, P->stream));
  }
  for (int k = 0; k < S->n; ++k) {                          // fixed order of the parts: deterministic sums
    DeviceGuard dg(S->dev[k]);
    qcd_lattice* P = S->part[k];
    CUDA_TRY(cudaStreamSynchronize(P->stream));
    for (int i = 0; i < npl; ++i) ps[i] += P->h_results[i];
    pl[0] += P->h_results[8]; pl[1] += P->h_results[9];
  }
  double V = 1.0;
  for (int d = 0; d < S->D; ++d) V *= S->dims[d];
  if (want_plaq) {
    double tot = 0.0;
    for (int i = 0; i < npl; ++i) { const double v = ps[i] / V; tot += v; if (plaq_planes) plaq_planes[i] = v; }
    if (plaq_total) *plaq_total = tot / npl;
  }
  if (polyakov) { const double Vs = V / S->dims[S->D - 1]; polyakov[0] = pl[0] / Vs; polyakov[1] = pl[1] / Vs; }
  return QCD_OK;
}

// global canonical layout on the HOST: the parts' own blocks are runs of ext * (sites below the split direction) sites
static int split_links(qcd_split_t* S, char* host, size_t bytes, bool set) {
  if (!S || !host) return fail(QCD_ERR_INVALID_ARG, "NULL argument");
  size_t V = 1;
  for (int d = 0; d < S->D; ++d) V *= (size_t)S->dims[d];
  const size_t site_bytes = (size_t)S->D * S->Nc * S->Nc * 2 * (S->precision == QCD_FP32 ? 4 : 8);
  if (bytes != V * site_bytes) return fail(QCD_ERR_INVALID_ARG, "bytes must equal V*D*N*N*2*sizeof(real)");
  size_t lo, hi;
  split_runs(S, &lo, &hi);
  const size_t grow = (size_t)S->dims[S->D - 2] * lo * site_bytes;      // bytes between runs of the global array
  std::vector<char> tmp;
  for (int k = 0; k < S->n; ++k) {
    DeviceGuard dg(S->dev[k]);
    const size_t run = (size_t)S->ext[k] * lo * site_bytes, goff = (size_t)S->off[k] * lo * site_bytes;
    tmp.resize(run * hi);
    if (set) for (size_t r = 0; r < hi; ++r) memcpy(tmp.data() + r * run, host + r * grow + goff, run);
    int rc = set ? qcd_set_links(S->part[k], tmp.data(), tmp.size(), 0) : qcd_get_links(S->part[k], tmp.data(), tmp.size(), 0);
    if (rc != QCD_OK) return rc;
    if (!set) for (size_t r = 0; r < hi; ++r) memcpy(host + r * grow + goff, tmp.data() + r * run, run);
  }
  return set ? split_refresh_all(S) : QCD_OK;
}
int qcd_split_get_links(qcd_split_t* S, void* dst, size_t bytes) {
  if (S && !S->part[0]->has_links) return fail(QCD_ERR_STATE, "no links yet");
  return split_links(S, (char*)dst, bytes, false);
}
int qcd_split_set_links(qcd_split_t* S, const void* src, size_t bytes) { return split_links(S, (char*)const_cast<void*>(src), bytes, true); }

int qcd_split_set_seed(qcd_split_t* S, uint64_t seed) {
  if (!S) return fail(QCD_ERR_INVALID_ARG, "NULL argument");
  for (int k = 0; k < S->n; ++k) S->part[k]->seed = seed;
  return QCD_OK;
}
int qcd_split_set_sweep_counter(qcd_split_t* S, uint32_t v) {
  if (!S) return fail(QCD_ERR_INVALID_ARG, "NULL argument");
  S->sweep = v;
  for (int k = 0; k < S->n; ++k) S->part[k]->sweep = v;
  return QCD_OK;
}
int qcd_split_get_sweep_counter(qcd_split_t* S, uint32_t* out) {
  if (!S || !out) return fail(QCD_ERR_INVALID_ARG, "NULL argument");
  *out = S->sweep; return QCD_OK;
}
int qcd_split_synchronize(qcd_split_t* S) {
  if (!S) return fail(QCD_ERR_INVALID_ARG, "NULL argument");
  for (int k = 0; k < S->n; ++k) { DeviceGuard dg(S->dev[k]); CUDA_TRY(cudaStreamSynchronize(S->stream[k])); }
  return QCD_OK;
}

}  // extern "C"

// =====================================================================================
// qcd_measure_plaquette_noalloc: the plaquette measurement for callers that must not allocate (include/qcd.h).
//
// qcd_measure keeps the per-CTA partial sums of plaquette_kernel in a buffer it cudaMallocs on first use.  Here the same two
// kernels run with the partials in the array below instead, which is part of the library's device image: every GPU that
// loads the library holds these QCD_NOALLOC_MAX_PARTIALS doubles (8 MiB) until the process exits, whether this entry point
// is ever called or not, and nothing is allocated or freed at call time.
//
// g_noalloc_partials is a device symbol.  In the host code of this file the name only identifies the symbol to the runtime;
// it is not an address a kernel can use, so the device address is looked up with cudaGetSymbolAddress, once per device and
// with that device current, and kept in g_noalloc_ptr.
// =====================================================================================
static __device__ __align__(256) double g_noalloc_partials[QCD_NOALLOC_MAX_PARTIALS];

namespace {

constexpr int NOALLOC_MAX_DEVICES = 64;
std::mutex g_noalloc_mutex;
double* g_noalloc_ptr[NOALLOC_MAX_DEVICES];   // device address of g_noalloc_partials on device i; nullptr: not looked up yet

// device address of the array on the CURRENT device (looked up on this device's first call; no allocation)
int noalloc_scratch(int dev, double** out) {
  if (dev < 0 || dev >= NOALLOC_MAX_DEVICES) return fail(QCD_ERR_UNSUPPORTED, "device ordinal beyond the per-device table of qcd_measure_plaquette_noalloc");
  std::lock_guard<std::mutex> lock(g_noalloc_mutex);
  if (!g_noalloc_ptr[dev]) {
    void* p = nullptr;
    const cudaError_t e = cudaGetSymbolAddress(&p, g_noalloc_partials);
    if (e != cudaSuccess || !p) return fail(QCD_ERR_CUDA, std::string("cudaGetSymbolAddress(g_noalloc_partials): ") + cudaGetErrorString(e));
    g_noalloc_ptr[dev] = (double*)p;
  }
  *out = g_noalloc_ptr[dev];
  return QCD_OK;
}

struct NoAllocPlaquetteOp {
  qcd_lattice* L; MeasureField mf; double* scratch; double* device_out;
  template <int NC, int D, typename R, bool COMP> int operator()() {
    typedef typename LinkIO<NC, R, COMP>::Vec Vec;
    constexpr int NPL = D * (D - 1) / 2;
    const MeasLayout m = meas_layout(L);
    mf.boxed = m.boxed ? 1 : 0;
    if (mf.boxed) {
      mf.n0 = make_fastdiv((uint32_t)(L->g.Lh0 / 8)); mf.n1 = make_fastdiv((uint32_t)(L->g.Li[1] / 2)); mf.n2 = make_fastdiv((uint32_t)(L->g.Li[2] / 2));
    }
    const dim3 plaq_grid = mf.boxed ? dim3(own_sites(L) / 128, 1) : dim3((L->g.Vh_int + 127) / 128, 2);
    // Every CTA of plaquette_kernel stores all NPL of its partials and final_reduce_kernel reads exactly those
    // NPL x nb_plaq entries: nothing in the array has to start at zero, and what an earlier call left beyond them is not read.
    plaquette_kernel<NC, D, R, COMP><<<plaq_grid, 128, 0, L->stream>>>(L->g, (const Vec*)L->mem, mf, scratch);
    final_reduce_kernel<<<NPL, 256, 0, L->stream>>>(scratch, m.nb_plaq, device_out, 1.0 / ((double)L->g.V * NC));
    CUDA_TRY(cudaGetLastError());
    L->launches += 2;
    L->last_parity = L->last_mu = -1;
    return QCD_OK;
  }
};

}  // namespace

extern "C" int qcd_measure_plaquette_noalloc(qcd_lattice_t* L, const qcd_field_t* field, double* device_out) {
  if (!L || !device_out) return fail(QCD_ERR_INVALID_ARG, "NULL argument");
  if (((uintptr_t)device_out) & 7u) return fail(QCD_ERR_INVALID_ARG, "device_out must be 8-byte aligned");
  if (!L->has_links) return fail(QCD_ERR_STATE, "no links yet");
  if (L->g.sd >= 0) return fail(QCD_ERR_UNSUPPORTED, "a slab has sums, not means: qcd_slab_measure_sums / qcd_split_measure");
  bool fon;
  int rc = check_field(L, field, &fon);
  if (rc != QCD_OK) return rc;
  const MeasLayout m = meas_layout(L);
  const size_t need = (size_t)m.npl * m.nb_plaq;
  if (need > (size_t)QCD_NOALLOC_MAX_PARTIALS) {
    char msg[256];
    snprintf(msg, sizeof(msg), "lattice too large for qcd_measure_plaquette_noalloc: it needs %zu partial sums (planes x sites/128), the "
             "built-in scratch array holds QCD_NOALLOC_MAX_PARTIALS = %d; use qcd_measure", need, (int)QCD_NOALLOC_MAX_PARTIALS);
    return fail(QCD_ERR_UNSUPPORTED, msg);
  }
  // the array's address is per device: the lattice's device must be the current one
  int dev = -1;
  CUDA_TRY(cudaGetDevice(&dev));
  cudaPointerAttributes attr;
  CUDA_TRY(cudaPointerGetAttributes(&attr, L->mem));
  if ((attr.type != cudaMemoryTypeDevice && attr.type != cudaMemoryTypeManaged) || (attr.type == cudaMemoryTypeDevice && attr.device != dev))
    return fail(QCD_ERR_STATE, "qcd_measure_plaquette_noalloc: the lattice's device must be the current device");
  double* scratch = nullptr;
  rc = noalloc_scratch(dev, &scratch);
  if (rc != QCD_OK) return rc;
  NoAllocPlaquetteOp op;
  op.L = L; op.scratch = scratch; op.device_out = device_out;
  memset(&op.mf, 0, sizeof(op.mf));
  const FieldArgs fa = make_field_args(field, fon, L->Nc);
  op.mf.enabled = fon ? 1 : 0; op.mf.mu = fa.mu; op.mf.nu = fa.nu;
  for (int c = 0; c < 3; ++c) { op.mf.c[c] = fa.c[c]; op.mf.s[c] = fa.s[c]; }
  return dispatch(L, op);
}
