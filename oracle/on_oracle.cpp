// =====================================================================================
// on_oracle.cpp -- TEST INFRASTRUCTURE ONLY.  Plain, slow, obviously-correct CPU oracle for the
// second workload of QCDGPU (arxiv 1310.7087): the O(N) scalar model updated by multi-hit
// ("improved") Metropolis on a checkerboard.
//
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline leg may build, load or call
// this file; it shares no code, header, table or constant generator with paper_1310_7087_b200/.
//
// What the paper fixes (PAPER.md = /root/reference/PAPER.md):
//   * "In case of O(N) models the fields are set with N-vectors, which are associated with
//      lattice sites"                                                  (sec 3.3)
//   * checkerboard: "lattice is traditionally divided into even and odd sites"
//   * "Improved Metropolis algorithm [7] is used for O(N) update"
//   * "For O(4) model NHIT=100 tries were used to update each lattice site (this provides
//      acceptance rate up to 50%)"                                     (sec 5)
//   * ref [7] is Bordag, Demchik, Gulov, Skalozub, "The type of the phase
//     transition and coupling values in lambda phi^4 model": the model is the N-component
//     lambda phi^4 scalar field.  The reference itself is NOT in the container; the paper prints
//     no action and no algorithm.  Readings taken (R16..R19):
//   R16 action (standard lattice parametrisation of the N-component phi^4 model):
//         S = sum_x [ -2 kappa sum_{mu<D} phi(x).phi(x+mu) + phi(x).phi(x) + lambda (phi(x).phi(x) - 1)^2 ]
//   R17 "improved Metropolis" = multi-hit Metropolis: every visit of a site makes NHIT tries, each
//       from the site's CURRENT value: phi' = phi + delta * s, s_a = 2 u_a - 1 uniform in (-1, 1)
//       per component, accepted iff u_acc < exp(-(S(phi') - S(phi))).  ALL NHIT tries are made (an
//       accepted try does not end the visit: stopping at the first acceptance would break detailed
//       balance, because the rejection probability depends on the current value).
//   R18 Philox keying: one Philox4x32-10 block per try, counter (lex site, sweep counter,
//       parity<<4 | hit<<8 | domain<<24 with domain 2, 0), key = seed.  The block's 128 bits give
//       five 23-bit numbers k: k_a = w_a & 0x7FFFFF (a = 0..3: components), k_acc = (w0>>23) |
//       (w1>>23)<<9 | ((w2>>23) & 31)<<18; uniform u = (k + 1/2) 2^-23 (exactly representable in
//       float and double, strictly inside (0,1)); N <= 4.
//   R19 hot start: phi_a = 2u - 1 from Philox domain 3 (same 23-bit numbers of one block per site);
//       cold start: phi = (1, 0, .., 0).  Observables: <phi^2> = (1/V) sum phi.phi, link energy
//       (1/(V D)) sum_x sum_mu phi(x).phi(x+mu), magnetisation vector (1/V) sum phi(x).
// Arithmetic: always double.  fp32 shadow mode (for the fp32 GPU kernels): the stored field is
// rounded to float after every accepted try, everything else stays double.
// Pins (tests/test_oracle_on.py): brute-force action difference, O(N) invariance of the action,
// decoupled sites (kappa = 0) against radial quadrature, free field (lambda = 0) against the exact
// lattice propagator, lambda -> infinity (|phi| -> 1), uniformity of the 23-bit numbers, trial
// bookkeeping, resume, and the Philox function itself against the known-answer vectors.
// "parity unpinned": the absolute values of observables at interacting couplings in D >= 2 (no closed
// form); every term of the action is pinned separately by the limits above and the brute-force test.
// =====================================================================================
#ifdef _OPENMP
#include <omp.h>
#endif
#include <cmath>
#include <cstdint>
#include <cstring>
#include <vector>

namespace {

// Philox4x32-10 (Salmon et al., SC'11), restated from the round description of SURVEY.md sec 8(c)-3
void philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
  uint32_t c[4] = {ctr[0], ctr[1], ctr[2], ctr[3]}, k[2] = {key[0], key[1]};
  for (int round = 0; round < 10; ++round) {
    const uint64_t p0 = (uint64_t)0xD2511F53u * c[0], p1 = (uint64_t)0xCD9E8D57u * c[2];
    const uint32_t n[4] = {(uint32_t)(p1 >> 32) ^ c[1] ^ k[0], (uint32_t)p1, (uint32_t)(p0 >> 32) ^ c[3] ^ k[1], (uint32_t)p0};
    for (int i = 0; i < 4; ++i) c[i] = n[i];
    if (round < 9) { k[0] += 0x9E3779B9u; k[1] += 0xBB67AE85u; }
  }
  for (int i = 0; i < 4; ++i) out[i] = c[i];
}

struct Lattice {
  int D, N, dims[4];
  long V;
  std::vector<double> phi;      // V * N, canonical layout [lex][component]
  uint64_t seed;
  uint32_t sweep;
  int store_fp32;
  unsigned long long accepted, tried;
};

inline void lex_to_coord(const Lattice& L, long lex, int x[4]) {
  for (int d = 0; d < L.D; ++d) { x[d] = (int)(lex % L.dims[d]); lex /= L.dims[d]; }
  for (int d = L.D; d < 4; ++d) x[d] = 0;
}
inline long coord_to_lex(const Lattice& L, const int x[4]) {
  long lex = 0;
  for (int d = L.D - 1; d >= 0; --d) lex = lex * L.dims[d] + x[d];
  return lex;
}
inline long neighbour(const Lattice& L, const int x[4], int d, int step) {
  int y[4] = {x[0], x[1], x[2], x[3]};
  y[d] = (y[d] + step + L.dims[d]) % L.dims[d];
  return coord_to_lex(L, y);
}

// R18: the five 23-bit numbers of one block
void block_numbers(uint64_t seed, long lex, uint32_t sweep, int parity, int hit, int domain, uint32_t k[5]) {
  const uint32_t key[2] = {(uint32_t)(seed & 0xFFFFFFFFull), (uint32_t)(seed >> 32)};
  const uint32_t ctr[4] = {(uint32_t)lex, sweep, ((uint32_t)parity << 4) | ((uint32_t)hit << 8) | ((uint32_t)domain << 24), 0u};
  uint32_t w[4];
  philox4x32_10(ctr, key, w);
  for (int a = 0; a < 4; ++a) k[a] = w[a] & 0x7FFFFFu;
  k[4] = (w[0] >> 23) | ((w[1] >> 23) << 9) | (((w[2] >> 23) & 31u) << 18);
}
inline double uniform23(uint32_t k) { return ((double)k + 0.5) * (1.0 / 8388608.0); }

// the part of the action (R16) that depends on phi(x): -2 kappa phi.h + phi.phi + lambda (phi.phi - 1)^2,
// h = sum over the 2D neighbours
double local_action(const double* p, const double* h, int N, double kappa, double lambda) {
  double ph = 0.0, pp = 0.0;
  for (int a = 0; a < N; ++a) { ph += p[a] * h[a]; pp += p[a] * p[a]; }
  return -2.0 * kappa * ph + pp + lambda * (pp - 1.0) * (pp - 1.0);
}

// one visit of site lex (R17): NHIT tries; returns the number of accepted tries
int visit_site(Lattice& L, long lex, int parity, double kappa, double lambda, double delta, int nhit) {
  const int N = L.N;
  int x[4];
  lex_to_coord(L, lex, x);
  double h[4] = {0, 0, 0, 0};
  for (int d = 0; d < L.D; ++d)
    for (int step = -1; step <= 1; step += 2) {
      const double* q = &L.phi[(size_t)neighbour(L, x, d, step) * N];
      for (int a = 0; a < N; ++a) h[a] += q[a];
    }
  double p[4] = {0, 0, 0, 0};
  for (int a = 0; a < N; ++a) p[a] = L.phi[(size_t)lex * N + a];
  if (L.store_fp32) delta = (double)(float)delta;                  // the fp32 kernels hold the step as a float
  int acc = 0;
  for (int t = 0; t < nhit; ++t) {
    uint32_t k[5];
    block_numbers(L.seed, lex, L.sweep, parity, t, /*domain=*/2, k);
    double q[4];
    for (int a = 0; a < N; ++a) {
      q[a] = p[a] + delta * (2.0 * uniform23(k[a]) - 1.0);
      if (L.store_fp32) q[a] = (double)(float)q[a];
    }
    const double dS = local_action(q, h, N, kappa, lambda) - local_action(p, h, N, kappa, lambda);
    if (uniform23(k[4]) < std::exp(-dS)) {
      for (int a = 0; a < N; ++a) p[a] = q[a];
      ++acc;
    }
  }
  for (int a = 0; a < N; ++a) L.phi[(size_t)lex * N + a] = p[a];
  return acc;
}

}  // namespace

extern "C" {

void* on_oracle_create(int D, const int* dims, int N) {
  if (D < 2 || D > 4 || N < 1 || N > 4) return nullptr;
  Lattice* L = new Lattice();
  L->D = D; L->N = N; L->V = 1;
  for (int d = 0; d < 4; ++d) L->dims[d] = 1;
  for (int d = 0; d < D; ++d) {
    if (dims[d] < 2 || (dims[d] & 1)) { delete L; return nullptr; }
    L->dims[d] = dims[d]; L->V *= dims[d];
  }
  L->phi.assign((size_t)L->V * N, 0.0);
  L->seed = 0; L->sweep = 0; L->store_fp32 = 0; L->accepted = 0; L->tried = 0;
  return L;
}
void on_oracle_destroy(void* h) { delete (Lattice*)h; }
void on_oracle_set_fp32(void* h, int on) { ((Lattice*)h)->store_fp32 = on ? 1 : 0; }
void on_oracle_set_seed(void* h, uint64_t s) { ((Lattice*)h)->seed = s; }
void on_oracle_set_sweep_counter(void* h, uint32_t s) { ((Lattice*)h)->sweep = s; }
uint32_t on_oracle_get_sweep_counter(void* h) { return ((Lattice*)h)->sweep; }
void on_oracle_get_field(void* h, double* dst) { Lattice* L = (Lattice*)h; std::memcpy(dst, L->phi.data(), L->phi.size() * sizeof(double)); }
void on_oracle_set_field(void* h, const double* src) { Lattice* L = (Lattice*)h; std::memcpy(L->phi.data(), src, L->phi.size() * sizeof(double)); }
void on_oracle_counts(void* h, unsigned long long* accepted, unsigned long long* tried) {
  Lattice* L = (Lattice*)h; *accepted = L->accepted; *tried = L->tried;
}

// start 0: cold, phi = (1,0,..,0); 1: hot, phi_a = 2u - 1 from Philox domain 3 (R19).  Sets seed, sweep counter = 0.
void on_oracle_init(void* h, int start, uint64_t seed) {
  Lattice* L = (Lattice*)h;
  L->seed = seed; L->sweep = 0; L->accepted = 0; L->tried = 0;
  for (long lex = 0; lex < L->V; ++lex) {
    int x[4]; lex_to_coord(*L, lex, x);
    const int parity = (x[0] + x[1] + x[2] + x[3]) & 1;
    uint32_t k[5];
    block_numbers(seed, lex, 0u, parity, 0, /*domain=*/3, k);
    for (int a = 0; a < L->N; ++a) {
      double v = start == 0 ? (a == 0 ? 1.0 : 0.0) : 2.0 * uniform23(k[a]) - 1.0;
      if (L->store_fp32) v = (double)(float)v;
      L->phi[(size_t)lex * L->N + a] = v;
    }
  }
}

// one parity of one sweep: every site of that parity is visited once (sites of one parity do not interact)
void on_oracle_half_sweep(void* h, int parity, double kappa, double lambda, double delta, int nhit) {
  Lattice* L = (Lattice*)h;
  unsigned long long acc = 0;
#pragma omp parallel for schedule(static) reduction(+ : acc)
  for (long lex = 0; lex < L->V; ++lex) {
    int x[4]; lex_to_coord(*L, lex, x);
    if (((x[0] + x[1] + x[2] + x[3]) & 1) != parity) continue;
    acc += (unsigned long long)visit_site(*L, lex, parity, kappa, lambda, delta, nhit);
  }
  L->accepted += acc; L->tried += (unsigned long long)(L->V / 2) * (unsigned long long)nhit;
}

// one sweep: even sites, then odd sites; the sweep counter is incremented at the end
void on_oracle_sweep(void* h, double kappa, double lambda, double delta, int nhit) {
  on_oracle_half_sweep(h, 0, kappa, lambda, delta, nhit);
  on_oracle_half_sweep(h, 1, kappa, lambda, delta, nhit);
  ((Lattice*)h)->sweep += 1;
}

// total action (R16) of the current configuration
double on_oracle_action(void* h, double kappa, double lambda) {
  Lattice* L = (Lattice*)h;
  double S = 0.0;
  for (long lex = 0; lex < L->V; ++lex) {
    int x[4]; lex_to_coord(*L, lex, x);
    const double* p = &L->phi[(size_t)lex * L->N];
    double pp = 0.0;
    for (int a = 0; a < L->N; ++a) pp += p[a] * p[a];
    S += pp + lambda * (pp - 1.0) * (pp - 1.0);
    for (int d = 0; d < L->D; ++d) {
      const double* q = &L->phi[(size_t)neighbour(*L, x, d, +1) * L->N];
      double pq = 0.0;
      for (int a = 0; a < L->N; ++a) pq += p[a] * q[a];
      S -= 2.0 * kappa * pq;
    }
  }
  return S;
}

// observables (R19): phi2 = (1/V) sum phi.phi ; link = (1/(V D)) sum_x sum_mu phi(x).phi(x+mu) ; mag[a] = (1/V) sum phi_a
void on_oracle_measure(void* h, double* phi2, double* link, double* mag) {
  Lattice* L = (Lattice*)h;
  double s2 = 0.0, sl = 0.0, m[4] = {0, 0, 0, 0};
  for (long lex = 0; lex < L->V; ++lex) {
    int x[4]; lex_to_coord(*L, lex, x);
    const double* p = &L->phi[(size_t)lex * L->N];
    for (int a = 0; a < L->N; ++a) { s2 += p[a] * p[a]; m[a] += p[a]; }
    for (int d = 0; d < L->D; ++d) {
      const double* q = &L->phi[(size_t)neighbour(*L, x, d, +1) * L->N];
      for (int a = 0; a < L->N; ++a) sl += p[a] * q[a];
    }
  }
  *phi2 = s2 / (double)L->V;
  *link = sl / ((double)L->V * L->D);
  for (int a = 0; a < L->N; ++a) mag[a] = m[a] / (double)L->V;
}

// the five 23-bit numbers of the block of (site, sweep, parity, hit, domain) -- for the pins of R18
void on_oracle_block_numbers(uint64_t seed, long lex, uint32_t sweep, int parity, int hit, int domain, uint32_t* out) {
  block_numbers(seed, lex, sweep, parity, hit, domain, out);
}
void on_oracle_philox(const uint32_t* ctr, const uint32_t* key, uint32_t* out) { philox4x32_10(ctr, key, out); }

int on_oracle_num_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

}  // extern "C"
