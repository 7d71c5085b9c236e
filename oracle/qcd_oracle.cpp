// =====================================================================================
// qcd_oracle.cpp -- TEST INFRASTRUCTURE ONLY.  Plain, slow, obviously-correct CPU oracle
// for the checkerboard SU(N) Monte Carlo sweep of QCDGPU (arxiv 1310.7087).
//
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg
// may build, load or call this file.  The product (paper_1310_7087_b200/, include/) never
// does, and shares no code, header, table or constant generator with it.
//
// What the paper fixes (PAPER.md = /root/reference/PAPER.md):
//   * links are N x N complex matrices on lattice links, N = 2,3   (sec 3.3)
//   * even/odd "checkerboard" update                               (sec 3.3)
//   * "(Pseudo)heat-bath algorithm is used for SU(N)"
//   * "NHIT=10 and reunitarization"                                (sec 5)
//   * run-time dimension D, single/double precision                (PAPER.md:31,  sec 1)
//   * external (chromo)magnetic field, finite temperature          (PAPER.md:11,  abstract)
//   * one seed reproduces the run                                  (sec 3.4)
// The paper prints no formulas ("we did not bring attention to the details of realized
// algorithms").  Every formula below is the textbook definition named by
// BASELINE.json's north_star, in the reading recorded in SURVEY.md sec 8(c) and DESIGN.md
// ("readings R1..R15").  Each function cites the reading it follows.
//
// Arithmetic: always double.  Storage: AoS std::complex<double>, canonical layout
//   U[lex][mu][row][col],  lex = x0 + L0*(x1 + L1*(x2 + L2*x3)),  dims[0] fastest,
//   dims[D-1] = time (Polyakov direction).
// Parity pins (what this file is checked against, tests/test_oracle_*.py): Philox
// known-answer vectors; cold plaquette = 1; brute-force action difference for the staples
// (with and without field); chi-square and Bessel-ratio mean of the Kennedy-Pendleton draw;
// overrelaxation conserves the action; unitarity/det = 1; 2-D SU(2) <P> = I2(beta)/I1(beta);
// 2-D SU(3) Weyl integral; strong coupling beta/18, beta/4; Haar moments of the hot start;
// centre transformation of the Polyakov loop; gauge and translation invariance.
// "parity unpinned": absolute 4-D plaquette values at production beta (5.7, 6.0, 6.2, 2.5)
// have no closed form; only relative GPU-vs-oracle parity is checked there.
// =====================================================================================
#ifdef _OPENMP
#include <omp.h>
#endif
#include <algorithm>
#include <cmath>
#include <complex>
#include <cstdint>
#include <cstring>
#include <vector>

typedef std::complex<double> cplx;

namespace {

// ------------------------------------------------------------------ small N x N matrices
struct Mat {            // N x N complex, N <= 3, row major; entries beyond N unused
  cplx m[3][3];
};

Mat mat_zero() { Mat r; for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) r.m[i][j] = 0.0; return r; }
Mat mat_identity(int N) { Mat r = mat_zero(); for (int i = 0; i < N; ++i) r.m[i][i] = 1.0; return r; }
Mat mat_mul(const Mat& a, const Mat& b, int N) {
  Mat r = mat_zero();
  for (int i = 0; i < N; ++i) for (int j = 0; j < N; ++j) for (int k = 0; k < N; ++k) r.m[i][j] += a.m[i][k] * b.m[k][j];
  return r;
}
Mat mat_dag(const Mat& a, int N) {
  Mat r = mat_zero();
  for (int i = 0; i < N; ++i) for (int j = 0; j < N; ++j) r.m[i][j] = std::conj(a.m[j][i]);
  return r;
}
Mat mat_add(const Mat& a, const Mat& b, int N) {
  Mat r = mat_zero();
  for (int i = 0; i < N; ++i) for (int j = 0; j < N; ++j) r.m[i][j] = a.m[i][j] + b.m[i][j];
  return r;
}
cplx mat_trace(const Mat& a, int N) { cplx t = 0.0; for (int i = 0; i < N; ++i) t += a.m[i][i]; return t; }

// ------------------------------------------------------------------ field description
// F = diag(exp(i*theta_c)) multiplies every plaquette of plane (mu,nu), mu<nu  (reading R12).
struct Field {
  int enabled;
  int mu, nu;
  double theta[3];
};
Mat field_matrix(const Field& f, int N) {
  Mat r = mat_zero();
  for (int c = 0; c < N; ++c) r.m[c][c] = std::polar(1.0, f.theta[c]);
  return r;
}

// ------------------------------------------------------------------ the lattice
struct Lattice {
  int D;
  int dims[4];
  int N;
  long V;
  std::vector<cplx> U;        // V * D * N * N
  uint64_t seed;
  uint32_t sweep;             // sweep counter s (Philox counter word c1)
  int max_trials;             // Kennedy-Pendleton trial cap T_max (reading R5: NHIT=10)
  int uniform_mode;           // 0: u=(w+0.5)*2^-32 ; 1: u=((w>>9)+0.5)*2^-23   (reading R8)
  int store_fp32;             // 1: every stored link is rounded to float (fp32 storage shadow, R15)
  int has_links;
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
inline int site_parity(const Lattice& L, const int x[4]) {
  int s = 0; for (int d = 0; d < L.D; ++d) s += x[d]; return s & 1;
}
// site x shifted by `step` (+1/-1) in direction d, periodic (checkerboard needs even extents)
inline long shifted(const Lattice& L, const int x[4], int d, int step) {
  int y[4] = {x[0], x[1], x[2], x[3]};
  y[d] = (y[d] + step + L.dims[d]) % L.dims[d];
  return coord_to_lex(L, y);
}
inline long shifted2(const Lattice& L, const int x[4], int d1, int s1, int d2, int s2) {
  int y[4] = {x[0], x[1], x[2], x[3]};
  y[d1] = (y[d1] + s1 + L.dims[d1]) % L.dims[d1];
  y[d2] = (y[d2] + s2 + L.dims[d2]) % L.dims[d2];
  return coord_to_lex(L, y);
}
inline Mat get_link(const Lattice& L, long lex, int mu) {
  Mat r = mat_zero();
  const cplx* p = &L.U[((size_t)lex * L.D + mu) * L.N * L.N];
  for (int i = 0; i < L.N; ++i) for (int j = 0; j < L.N; ++j) r.m[i][j] = p[i * L.N + j];
  return r;
}
inline void put_link(Lattice& L, long lex, int mu, const Mat& a) {
  cplx* p = &L.U[((size_t)lex * L.D + mu) * L.N * L.N];
  for (int i = 0; i < L.N; ++i) for (int j = 0; j < L.N; ++j) {
    cplx z = a.m[i][j];
    if (L.store_fp32) z = cplx((double)(float)z.real(), (double)(float)z.imag());
    p[i * L.N + j] = z;
  }
}

// ------------------------------------------------------------------ Philox4x32-10
// Salmon, Moraes, Dror, Shaw, "Parallel random numbers: as easy as 1, 2, 3" (SC'11);
// mandated by BASELINE.json north_star; round description as in SURVEY.md sec 8(c)-3.
void philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
  const uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u, W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;
  uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3], k0 = key[0], k1 = key[1];
  for (int round = 0; round < 10; ++round) {
    uint64_t p0 = (uint64_t)M0 * c0, p1 = (uint64_t)M1 * c2;
    uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
    uint32_t n1 = (uint32_t)p1;
    uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
    uint32_t n3 = (uint32_t)p0;
    c0 = n0; c1 = n1; c2 = n2; c3 = n3;
    if (round < 9) { k0 += W0; k1 += W1; }
  }
  out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// Keying (reading R7): key = seed; c0 = lex site, c1 = sweep counter,
// c2 = mu | parity<<4 | subgroup<<5 | hit<<8 | domain<<24, c3 = draw.
void keyed_block(uint64_t seed, long lex, uint32_t sweep, int mu, int parity, int sg, int hit, int domain, int draw,
                 uint32_t out[4]) {
  uint32_t key[2] = {(uint32_t)(seed & 0xFFFFFFFFull), (uint32_t)(seed >> 32)};
  uint32_t ctr[4] = {(uint32_t)lex, sweep,
                     (uint32_t)mu | ((uint32_t)parity << 4) | ((uint32_t)sg << 5) | ((uint32_t)hit << 8) | ((uint32_t)domain << 24),
                     (uint32_t)draw};
  philox4x32_10(ctr, key, out);
}

// Word -> uniform strictly inside (0,1) (reading R8).
double word_to_uniform(uint32_t w, int mode) {
  if (mode == 0) return ((double)w + 0.5) * (1.0 / 4294967296.0);
  return ((double)(w >> 9) + 0.5) * (1.0 / 8388608.0);
}

// ------------------------------------------------------------------ staples
// A(x,mu) = sum_{nu != mu} [ U_nu(x+mu) U_mu(x+nu)^+ U_nu(x)^+  +  U_nu(x+mu-nu)^+ U_mu(x-nu)^+ U_nu(x-nu) ]
// so that the U_mu(x)-dependent part of sum_P Re Tr P is Re Tr[U_mu(x) A].  With a field in plane (m,n), m<n:
//   link along m (mu=m, nu=n): upper * F ,  lower: ... U_mu(x-nu)^+ * F^+ * U_nu(x-nu)
//   link along n (mu=n, nu=m): upper * F^+, lower: ... U_mu(x-nu)^+ * F   * U_nu(x-nu)
Mat staple_sum(const Lattice& L, long lex, int mu, const Field* field) {
  const int N = L.N;
  int x[4]; lex_to_coord(L, lex, x);
  Mat A = mat_zero();
  for (int nu = 0; nu < L.D; ++nu) {
    if (nu == mu) continue;
    Mat up_fac = mat_identity(N), low_fac = mat_identity(N);
    if (field && field->enabled) {
      Mat F = field_matrix(*field, N);
      if (mu == field->mu && nu == field->nu) { up_fac = F; low_fac = mat_dag(F, N); }
      else if (mu == field->nu && nu == field->mu) { up_fac = mat_dag(F, N); low_fac = F; }
    }
    long xpmu = shifted(L, x, mu, +1), xpnu = shifted(L, x, nu, +1), xmnu = shifted(L, x, nu, -1);
    long xpmumnu = shifted2(L, x, mu, +1, nu, -1);
    // upper: U_nu(x+mu) U_mu(x+nu)^+ U_nu(x)^+ [* F or F^+]
    Mat up = mat_mul(mat_mul(get_link(L, xpmu, nu), mat_dag(get_link(L, xpnu, mu), N), N), mat_dag(get_link(L, lex, nu), N), N);
    up = mat_mul(up, up_fac, N);
    // lower: U_nu(x+mu-nu)^+ U_mu(x-nu)^+ [F^+ or F] U_nu(x-nu)
    Mat lo = mat_mul(mat_dag(get_link(L, xpmumnu, nu), N), mat_dag(get_link(L, xmnu, mu), N), N);
    lo = mat_mul(mat_mul(lo, low_fac, N), get_link(L, xmnu, nu), N);
    A = mat_add(A, mat_add(up, lo, N), N);
  }
  return A;
}

// ------------------------------------------------------------------ quaternions
// a=(a0,a1,a2,a3) <-> [[a0+i a3, a2+i a1],[-a2+i a1, a0-i a3]] = a0 + i a.sigma
struct Quat { double q[4]; };
Quat quat_mul(const Quat& a, const Quat& b) {
  Quat r;
  r.q[0] = a.q[0] * b.q[0] - a.q[1] * b.q[1] - a.q[2] * b.q[2] - a.q[3] * b.q[3];
  // vector part: a0 b + b0 a - a x b
  r.q[1] = a.q[0] * b.q[1] + b.q[0] * a.q[1] - (a.q[2] * b.q[3] - a.q[3] * b.q[2]);
  r.q[2] = a.q[0] * b.q[2] + b.q[0] * a.q[2] - (a.q[3] * b.q[1] - a.q[1] * b.q[3]);
  r.q[3] = a.q[0] * b.q[3] + b.q[0] * a.q[3] - (a.q[1] * b.q[2] - a.q[2] * b.q[1]);
  return r;
}
Quat quat_conj(const Quat& a) { Quat r = {{a.q[0], -a.q[1], -a.q[2], -a.q[3]}}; return r; }
// embed(a; i, j): identity with the 2x2 block at rows/cols (i,j) replaced by a's matrix
Mat quat_embed(const Quat& a, int i, int j, int N) {
  Mat r = mat_identity(N);
  r.m[i][i] = cplx(a.q[0], a.q[3]);
  r.m[i][j] = cplx(a.q[2], a.q[1]);
  r.m[j][i] = cplx(-a.q[2], a.q[1]);
  r.m[j][j] = cplx(a.q[0], -a.q[3]);
  return r;
}

// ------------------------------------------------------------------ reunitarisation (reading R6)
Mat reunitarise(const Mat& in, int N) {
  Mat r = in;
  if (N == 2) {
    // quaternion from the first row, normalised, rebuilt
    double a0 = in.m[0][0].real(), a3 = in.m[0][0].imag(), a2 = in.m[0][1].real(), a1 = in.m[0][1].imag();
    double n = std::sqrt(a0 * a0 + a1 * a1 + a2 * a2 + a3 * a3);
    Quat a = {{a0 / n, a1 / n, a2 / n, a3 / n}};
    return quat_embed(a, 0, 1, 2);
  }
  // SU(3): Gram-Schmidt on rows 0,1; row 2 = conj(row0 x row1)
  double n0 = 0.0; for (int c = 0; c < 3; ++c) n0 += std::norm(r.m[0][c]);
  n0 = std::sqrt(n0); for (int c = 0; c < 3; ++c) r.m[0][c] /= n0;
  cplx d = 0.0; for (int c = 0; c < 3; ++c) d += std::conj(r.m[0][c]) * r.m[1][c];
  for (int c = 0; c < 3; ++c) r.m[1][c] -= d * r.m[0][c];
  double n1 = 0.0; for (int c = 0; c < 3; ++c) n1 += std::norm(r.m[1][c]);
  n1 = std::sqrt(n1); for (int c = 0; c < 3; ++c) r.m[1][c] /= n1;
  r.m[2][0] = std::conj(r.m[0][1] * r.m[1][2] - r.m[0][2] * r.m[1][1]);
  r.m[2][1] = std::conj(r.m[0][2] * r.m[1][0] - r.m[0][0] * r.m[1][2]);
  r.m[2][2] = std::conj(r.m[0][0] * r.m[1][1] - r.m[0][1] * r.m[1][0]);
  return r;
}

// ------------------------------------------------------------------ Kennedy-Pendleton draw
// g0 with density ~ sqrt(1-g0^2) exp(alpha g0); at most max_trials trials; trial t uses Philox draw 1+t.
// Returns true when accepted.  *code: t+1 when accepted at trial t; 0x80|max_trials when exhausted.
bool kennedy_pendleton(double alpha, uint64_t seed, long lex, uint32_t sweep, int mu, int parity, int sg, int hit,
                       int max_trials, int uniform_mode, double* g0, int* code) {
  for (int t = 0; t < max_trials; ++t) {
    uint32_t w[4];
    keyed_block(seed, lex, sweep, mu, parity, sg, hit, /*domain=*/0, /*draw=*/1 + t, w);
    double r1 = word_to_uniform(w[0], uniform_mode), r2 = word_to_uniform(w[1], uniform_mode);
    double r3 = word_to_uniform(w[2], uniform_mode), r4 = word_to_uniform(w[3], uniform_mode);
    double c = std::cos(2.0 * M_PI * r2);
    double delta = -(std::log(r1) + c * c * std::log(r3)) / alpha;
    if (r4 * r4 <= 1.0 - 0.5 * delta) { *g0 = 1.0 - delta; *code = t + 1; return true; }
  }
  *code = 0x80 | max_trials;
  return false;
}

// ------------------------------------------------------------------ Cabibbo-Marinari update of one link
// kind 0: heatbath hit `hit`; kind 1: overrelaxation.  trial_codes[sg] receives the KP code (0 if skipped / OR).
// *kmin (optional) receives the smallest subgroup projection norm k met (conditioning of the update, test diagnostics).
Mat cm_update(const Lattice& L, const Mat& U_in, const Mat& A, double beta, int kind, int hit, long lex, int mu, int parity,
              int trial_codes[3], double* kmin = nullptr) {
  const int N = L.N;
  static const int sub_i[3] = {0, 0, 1}, sub_j[3] = {1, 2, 2};       // reading R3
  const int n_sub = (N == 2) ? 1 : 3;
  Mat U = U_in;
  for (int sg = 0; sg < 3; ++sg) trial_codes[sg] = 0;
  for (int sg = 0; sg < n_sub; ++sg) {
    const int i = sub_i[sg], j = sub_j[sg];
    Mat W = mat_mul(U, A, N);                                        // with the *current* U
    cplx M00 = W.m[i][i], M01 = W.m[i][j], M10 = W.m[j][i], M11 = W.m[j][j];
    Quat v;
    v.q[0] = 0.5 * (M00 + M11).real();
    v.q[1] = 0.5 * (M01 + M10).imag();
    v.q[2] = 0.5 * (M01 - M10).real();
    v.q[3] = 0.5 * (M00 - M11).imag();
    double k2 = v.q[0] * v.q[0] + v.q[1] * v.q[1] + v.q[2] * v.q[2] + v.q[3] * v.q[3];
    if (kmin && (sg == 0 || std::sqrt(k2) < *kmin)) *kmin = std::sqrt(k2);
    if (k2 < 1e-30) continue;                                        // reading R4
    double k = std::sqrt(k2);
    Quat vt = {{v.q[0] / k, v.q[1] / k, v.q[2] / k, v.q[3] / k}};
    Quat a;
    if (kind == 1) {
      // overrelaxation: a = (vt^+)^2
      a = quat_mul(quat_conj(vt), quat_conj(vt));
    } else {
      double alpha = 2.0 * beta * k / N;
      double g0; int code;
      bool ok = kennedy_pendleton(alpha, L.seed, lex, L.sweep, mu, parity, sg, hit, L.max_trials, L.uniform_mode, &g0, &code);
      trial_codes[sg] = code;
      if (!ok) continue;                                             // reading R5: keep the old subgroup part
      uint32_t w[4];
      keyed_block(L.seed, lex, L.sweep, mu, parity, sg, hit, /*domain=*/0, /*draw=*/0, w);
      double u1 = word_to_uniform(w[0], L.uniform_mode), u2 = word_to_uniform(w[1], L.uniform_mode);
      double ct = 1.0 - 2.0 * u1, st = std::sqrt(1.0 - ct * ct), phi = 2.0 * M_PI * u2;
      double r = std::sqrt(std::max(0.0, 1.0 - g0 * g0));
      Quat g = {{g0, r * st * std::cos(phi), r * st * std::sin(phi), r * ct}};
      a = quat_mul(g, quat_conj(vt));
    }
    U = mat_mul(quat_embed(a, i, j, N), U, N);
  }
  return reunitarise(U, N);                                          // once per link-hit, before the store
}

void update_one_link(Lattice& L, long lex, int mu, double beta, int kind, int hit, const Field* field, Mat* out, int codes[3],
                     double* kmin = nullptr) {
  int x[4]; lex_to_coord(L, lex, x);
  Mat A = staple_sum(L, lex, mu, field);
  *out = cm_update(L, get_link(L, lex, mu), A, beta, kind, hit, lex, mu, site_parity(L, x), codes, kmin);
}

// one (parity, mu) sub-step over all sites of that parity (any order: sites are independent)
void substep(Lattice& L, double beta, int kind, int hit, int parity, int mu, const Field* field, uint8_t* trials,
             double* kmin = nullptr) {
#pragma omp parallel for schedule(static)
  for (long lex = 0; lex < L.V; ++lex) {
    int x[4]; lex_to_coord(L, lex, x);
    if (site_parity(L, x) != parity) continue;
    Mat Unew; int codes[3];
    update_one_link(L, lex, mu, beta, kind, hit, field, &Unew, codes, kmin ? &kmin[lex] : nullptr);
    put_link(L, lex, mu, Unew);        // writes U_mu on parity p only; nobody else reads it in this sub-step
    if (trials) for (int sg = 0; sg < 3; ++sg) trials[(size_t)lex * 3 + sg] = (uint8_t)codes[sg];
  }
}

// hot start (reading R9): Gaussians by Box-Muller on consecutive 32-bit-mode uniforms
void hot_link(const Lattice& L, long lex, int mu, int parity, Mat* out) {
  const int N = L.N;
  const int n_draws = (N == 2) ? 1 : 3;
  double z[12];
  for (int d = 0; d < n_draws; ++d) {
    uint32_t w[4];
    keyed_block(L.seed, lex, /*sweep=*/0, mu, parity, /*sg=*/0, /*hit=*/0, /*domain=*/1, d, w);
    for (int pair = 0; pair < 2; ++pair) {
      double ua = word_to_uniform(w[2 * pair], 0), ub = word_to_uniform(w[2 * pair + 1], 0);
      double rad = std::sqrt(-2.0 * std::log(ua));
      z[4 * d + 2 * pair] = rad * std::cos(2.0 * M_PI * ub);
      z[4 * d + 2 * pair + 1] = rad * std::sin(2.0 * M_PI * ub);
    }
  }
  if (N == 2) {
    double n = std::sqrt(z[0] * z[0] + z[1] * z[1] + z[2] * z[2] + z[3] * z[3]);
    Quat a = {{z[0] / n, z[1] / n, z[2] / n, z[3] / n}};
    *out = quat_embed(a, 0, 1, 2);
    return;
  }
  Mat r = mat_zero();
  for (int c = 0; c < 3; ++c) { r.m[0][c] = cplx(z[2 * c], z[2 * c + 1]); r.m[1][c] = cplx(z[6 + 2 * c], z[6 + 2 * c + 1]); }
  *out = reunitarise(r, 3);
}

}  // namespace

// =====================================================================================
// C interface for ctypes (tests, smoke, bench cpu_baseline).  Names carry the oracle_ prefix.
// =====================================================================================
extern "C" {

void oracle_philox4x32_10(const uint32_t* ctr, const uint32_t* key, uint32_t* out) { philox4x32_10(ctr, key, out); }

void oracle_philox4x32_10_batch(const uint32_t* ctr, const uint32_t* key, long n, uint32_t* out) {
  for (long i = 0; i < n; ++i) philox4x32_10(ctr + 4 * i, key + 2 * i, out + 4 * i);
}

void oracle_keyed_block(uint64_t seed, long lex, uint32_t sweep, int mu, int parity, int sg, int hit, int domain, int draw,
                        uint32_t* out) {
  keyed_block(seed, lex, sweep, mu, parity, sg, hit, domain, draw, out);
}

double oracle_word_to_uniform(uint32_t w, int mode) { return word_to_uniform(w, mode); }

void* oracle_create(int D, const int* dims, int N) {
  if (D < 2 || D > 4 || (N != 2 && N != 3)) return nullptr;
  Lattice* L = new Lattice();
  L->D = D; L->N = N; L->V = 1;
  for (int d = 0; d < 4; ++d) L->dims[d] = 1;
  for (int d = 0; d < D; ++d) {
    if (dims[d] < 2 || (dims[d] & 1)) { delete L; return nullptr; }
    L->dims[d] = dims[d]; L->V *= dims[d];
  }
  L->U.assign((size_t)L->V * D * N * N, cplx(0.0, 0.0));
  L->seed = 0; L->sweep = 0; L->max_trials = 10; L->uniform_mode = 0; L->store_fp32 = 0; L->has_links = 0;
  return L;
}
void oracle_destroy(void* h) { delete (Lattice*)h; }

// key 0: max_trials, key 1: uniform_mode, key 2: store_fp32
int oracle_set_option(void* h, int key, int value) {
  Lattice* L = (Lattice*)h;
  if (key == 0) { if (value < 1 || value > 127) return 1; L->max_trials = value; return 0; }
  if (key == 1) { L->uniform_mode = value ? 1 : 0; return 0; }
  if (key == 2) { L->store_fp32 = value ? 1 : 0; return 0; }
  return 1;
}
void oracle_set_seed(void* h, uint64_t seed) { ((Lattice*)h)->seed = seed; }
void oracle_set_sweep_counter(void* h, uint32_t s) { ((Lattice*)h)->sweep = s; }
uint32_t oracle_get_sweep_counter(void* h) { return ((Lattice*)h)->sweep; }

// start 0: cold (all links identity), 1: hot (Haar random from Philox domain 1).  Sets seed, sweep counter = 0.
int oracle_init(void* h, int start, uint64_t seed) {
  Lattice* L = (Lattice*)h;
  L->seed = seed; L->sweep = 0;
#pragma omp parallel for schedule(static)
  for (long lex = 0; lex < L->V; ++lex) {
    int x[4]; lex_to_coord(*L, lex, x);
    for (int mu = 0; mu < L->D; ++mu) {
      Mat u;
      if (start == 0) u = mat_identity(L->N); else hot_link(*L, lex, mu, site_parity(*L, x), &u);
      put_link(*L, lex, mu, u);
    }
  }
  L->has_links = 1;
  return 0;
}

// canonical layout, complex128: [lex][mu][row][col]
void oracle_get_links(void* h, double* dst) {
  Lattice* L = (Lattice*)h; std::memcpy(dst, L->U.data(), L->U.size() * sizeof(cplx));
}
void oracle_set_links(void* h, const double* src) {
  Lattice* L = (Lattice*)h; std::memcpy((void*)L->U.data(), src, L->U.size() * sizeof(cplx)); L->has_links = 1;
}

// field may be NULL.  trials: NULL or V*3 bytes indexed [lex][subgroup] (only sites of `parity` written).
void oracle_substep(void* h, double beta, int kind, int hit, int parity, int mu, const Field* field, uint8_t* trials) {
  substep(*(Lattice*)h, beta, kind, hit, parity, mu, field, trials);
}
// same, and kmin[lex] (V doubles, only sites of `parity` written) = smallest subgroup projection norm of that link update
void oracle_substep_diag(void* h, double beta, int kind, int hit, int parity, int mu, const Field* field, uint8_t* trials,
                         double* kmin) {
  substep(*(Lattice*)h, beta, kind, hit, parity, mu, field, trials, kmin);
}

// One qcd_sweep: passes outermost (R1), then parity, then direction (R2); counter += 1 at the end.
void oracle_sweep(void* h, double beta, int n_hb, int n_or, const Field* field) {
  Lattice* L = (Lattice*)h;
  for (int pass = 0; pass < n_hb + n_or; ++pass) {
    int kind = (pass < n_hb) ? 0 : 1, hit = (pass < n_hb) ? pass : 0;
    for (int p = 0; p < 2; ++p)
      for (int mu = 0; mu < L->D; ++mu) substep(*L, beta, kind, hit, p, mu, field, nullptr);
  }
  L->sweep += 1;
}

// new value of the single link (lex, mu) from the CURRENT configuration (does not store it).
void oracle_update_one_link(void* h, double beta, int kind, int hit, long lex, int mu, const Field* field, double* out_link,
                            uint8_t* codes_out, double* kmin_out) {
  Lattice* L = (Lattice*)h;
  Mat u; int codes[3];
  update_one_link(*L, lex, mu, beta, kind, hit, field, &u, codes, kmin_out);
  for (int i = 0; i < L->N; ++i) for (int j = 0; j < L->N; ++j) {
    out_link[2 * (i * L->N + j)] = u.m[i][j].real(); out_link[2 * (i * L->N + j) + 1] = u.m[i][j].imag();
  }
  if (codes_out) for (int sg = 0; sg < 3; ++sg) codes_out[sg] = (uint8_t)codes[sg];
}

void oracle_staple(void* h, long lex, int mu, const Field* field, double* out) {
  Lattice* L = (Lattice*)h;
  Mat A = staple_sum(*L, lex, mu, field);
  for (int i = 0; i < L->N; ++i) for (int j = 0; j < L->N; ++j) {
    out[2 * (i * L->N + j)] = A.m[i][j].real(); out[2 * (i * L->N + j) + 1] = A.m[i][j].imag();
  }
}

// Observables.  plaq_planes: D(D-1)/2 values, order (0,1),(0,2),..,(D-2,D-1); dressed with F (R10).
// polyakov: (Re L, Im L), direction D-1, (1/N) Tr of the ordered product in increasing t (R11).
void oracle_measure(void* h, const Field* field, double* plaq_total, double* plaq_planes, double* polyakov) {
  Lattice* Lp = (Lattice*)h; const Lattice& L = *Lp; const int N = L.N, D = L.D;
  int plane = 0; double total = 0.0;
  for (int mu = 0; mu < D; ++mu) for (int nu = mu + 1; nu < D; ++nu, ++plane) {
    Mat F = mat_identity(N);
    if (field && field->enabled && field->mu == mu && field->nu == nu) F = field_matrix(*field, N);
    double sum = 0.0;
#pragma omp parallel for schedule(static) reduction(+ : sum)
    for (long lex = 0; lex < L.V; ++lex) {
      int x[4]; lex_to_coord(L, lex, x);
      Mat P = mat_mul(F, get_link(L, lex, mu), N);
      P = mat_mul(P, get_link(L, shifted(L, x, mu, +1), nu), N);
      P = mat_mul(P, mat_dag(get_link(L, shifted(L, x, nu, +1), mu), N), N);
      P = mat_mul(P, mat_dag(get_link(L, lex, nu), N), N);
      sum += mat_trace(P, N).real() / N;
    }
    double mean = sum / (double)L.V;
    if (plaq_planes) plaq_planes[plane] = mean;
    total += mean;
  }
  if (plaq_total) *plaq_total = total / plane;
  if (polyakov) {
    const int Lt = L.dims[D - 1]; const long Vs = L.V / Lt;
    double re = 0.0, im = 0.0;
#pragma omp parallel for schedule(static) reduction(+ : re, im)
    for (long s = 0; s < Vs; ++s) {
      Mat P = mat_identity(N);
      for (int t = 0; t < Lt; ++t) P = mat_mul(P, get_link(L, s + (long)t * Vs, D - 1), N);
      cplx tr = mat_trace(P, N) / (double)N;
      re += tr.real(); im += tr.imag();
    }
    polyakov[0] = re / (double)Vs; polyakov[1] = im / (double)Vs;
  }
}

// Stand-alone Kennedy-Pendleton draws for the chi-square pin: n draws at fixed alpha, draw i keyed by site index i.
// g0_out[i] = accepted g0 or NaN when all trials failed; codes_out[i] = trial code.
void oracle_kp_samples(double alpha, uint64_t seed, long n, int max_trials, int uniform_mode, double* g0_out, uint8_t* codes_out) {
  for (long i = 0; i < n; ++i) {
    double g0 = NAN; int code = 0;
    kennedy_pendleton(alpha, seed, i, 0, 0, 0, 0, 0, max_trials, uniform_mode, &g0, &code);
    g0_out[i] = g0; codes_out[i] = (uint8_t)code;
  }
}

// threads the OpenMP loops of substep / measure use (reported by bench.py's cpu_baseline as "cores")
int oracle_num_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

}  // extern "C"
