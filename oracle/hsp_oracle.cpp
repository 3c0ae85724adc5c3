// hsp_oracle.cpp -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
//
// A plain, slow, single-threaded CPU Gibbs sampler for the Horseshoe Probit model of
// Terenin, Dong & Draper (arXiv 1608.04329), written from /root/reference/PAPER.md only.
// It is the oracle the CUDA path (paper_1608_04329_b200/) is compared against.  It shares no
// source, header, table or helper with the CUDA path and neither includes the other.
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg
// may load this library.
//
// What it computes (one sweep, in the paper's order, "Our algorithm performs
// the following updates: (i) z and lambda^-2 in parallel, followed by tau^-2; (ii) beta, nu^-1,
// xi^-1 in parallel"), with the six full conditionals of eq. (12), PAPER.md:174-184:
//   1. eta_i   = sum_j x_ij beta_j                                  (z step i)
//   2. z_i     ~ TN(eta_i, 1, y_i)
//   3. g_j     = sum_i x_ij z_i   (X^T z)                           (beta step vi)
//   4. lam_j^-2 ~ Exp(nu_j^-1 + tau^-2 beta_j^2 / 2)
//   5. tau^-2  ~ Gamma((p+1)/2, rate xi^-1 + 1/2 sum lam_j^-2 beta_j^2)   (
//                DESIGN.md reading R1: Gamma, not IG, for the precision tau^-2)
//   6. Q = X^T X + diag(tau^-2 lam_j^-2);  Q = L L^T
//   7. beta = Q^-1 g + L^-T e,  e ~ N(0, I)
//   8. nu_j^-1 ~ Exp(1 + lam_j^-2);  xi^-1 ~ Exp(1 + tau^-2)
// All arithmetic is fp64; the special-function inversions run in long double.  Loops are the
// textbook ones (i ascending, j ascending); nothing is blocked, fused or reordered.
//
// TIMING-ONLY mode FLAG_ROW_CHUNKS (never used by a parity test as the reference): steps 1-3 run over FIXED
// chunks of 4096 rows, the chunks dealt to the host cores by OpenMP, each chunk keeping its own partial of
// X^T z, and the partials are added in chunk order -- the same row arithmetic, the analogue of the paper's
// 16-thread workstation code (SURVEY.md 8(d) "oracle timing (ii)").  The result does not
// depend on the number of threads; it differs from the default path by the summation order of g only
// (pinned by tests/test_oracle_chain.py::test_row_chunk_mode_matches_default).
//
// Random numbers: the paper says only "use Philox".  The contract (DESIGN.md
// "Random-number contract") is Philox-4x32-10 with counter (idx_lo, idx_hi, sweep, tag) and key
// (seed_lo, seed_hi); one Philox call per variate.  This file has its own implementation.
//
// Pins (tests/test_oracle_*.py, all "-m 'not gpu'"):
//   philox4x32_10   : the CUDA toolkit's cuRAND *host* Philox generator (library, CPU)
//   qinv / norm_inv : scipy.special.ndtri, mpmath round trip
//   tnpos           : sign invariant, mpmath round trip Q(t)/Q(a)=u, closed-form moments,
//                     KS against the paper's own rejection samplers
//   exponential     : closed-form CDF
//   cheng_gamma     : scipy.stats.gamma KS, mean=var=alpha, acceptance
//   cholesky/solves : numpy.linalg
//   beta step       : mean/covariance of 1e5 draws vs Q^-1 X^T z and Q^-1
//   scale steps     : brute-force quadrature of p(lambda_j | .), p(tau | .) for p <= 3
//   whole chain     : 3-D quadrature (p=1), planted-beta recovery
// No function here is "parity unpinned".

#include <cfloat>
#include <chrono>
#include <cmath>
#include <cstdint>
#include <cstdlib>
#include <cstring>
#include <algorithm>
#include <new>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

// ----------------------------------------------------------------------------------------
// Philox-4x32-10 (Salmon et al. 2011).
// ----------------------------------------------------------------------------------------
constexpr uint32_t kMul0 = 0xD2511F53u, kMul1 = 0xCD9E8D57u;
constexpr uint32_t kWeyl0 = 0x9E3779B9u, kWeyl1 = 0xBB67AE85u;

void philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
  uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
  uint32_t k0 = key[0], k1 = key[1];
  for (int round = 0; round < 10; ++round) {
    if (round > 0) { k0 += kWeyl0; k1 += kWeyl1; }
    const uint64_t prod0 = (uint64_t)kMul0 * c0;
    const uint64_t prod1 = (uint64_t)kMul1 * c2;
    const uint32_t hi0 = (uint32_t)(prod0 >> 32), lo0 = (uint32_t)prod0;
    const uint32_t hi1 = (uint32_t)(prod1 >> 32), lo1 = (uint32_t)prod1;
    const uint32_t n0 = hi1 ^ c1 ^ k0;
    const uint32_t n1 = lo1;
    const uint32_t n2 = hi0 ^ c3 ^ k1;
    const uint32_t n3 = lo0;
    c0 = n0; c1 = n1; c2 = n2; c3 = n3;
  }
  out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

enum Tag : uint32_t { TAG_Z = 0, TAG_LAMBDA = 1, TAG_TAU = 2, TAG_E = 3, TAG_NU = 4, TAG_XI = 5,
                      TAG_LITERAL = 6 };

// 52 random bits + 1/2, scaled by 2^-52: strictly inside (0,1); u and 1-u are both exact.
inline double bits_to_unit(uint32_t hi, uint32_t lo) {
  const uint64_t n = ((uint64_t)hi << 20) | (uint64_t)(lo >> 12);
  return ((double)n + 0.5) * 0x1.0p-52;
}

void uniforms(uint64_t seed, uint64_t idx, uint32_t sweep, uint32_t tag, double* ua, double* ub) {
  const uint32_t ctr[4] = {(uint32_t)idx, (uint32_t)(idx >> 32), sweep, tag};
  const uint32_t key[2] = {(uint32_t)seed, (uint32_t)(seed >> 32)};
  uint32_t r[4];
  philox4x32_10(ctr, key, r);
  if (ua) *ua = bits_to_unit(r[0], r[1]);
  if (ub) *ub = bits_to_unit(r[2], r[3]);
}

// ----------------------------------------------------------------------------------------
// Normal tail Q(x) = P(N(0,1) > x) = erfc(x/sqrt 2)/2 and its inverse, long double.
// ----------------------------------------------------------------------------------------
const long double kSqrt1_2 = 0.70710678118654752440084436210484903928L;
const long double kSqrt2OverPi = 0.79788456080286535587989211986876373695L;  // sqrt(2/pi)

inline long double upper_tail(long double x) { return 0.5L * erfcl(x * kSqrt1_2); }

// Solve Q(x) = q for q in (0, 1/2]  (so x >= 0).  Safeguarded Newton on log Q, which is concave
// and decreasing: after the first step the iterates approach the root from the right.
long double qinv_half(long double q) {
  if (!(q > 0.0L)) return INFINITY;
  if (q >= 0.5L) return 0.0L;
  const long double target = logl(q);
  long double lo = 0.0L, hi = 160.0L;      // Q(160) ~ 1e-5561 is below any q we can form
  long double x = sqrtl(-2.0L * target);   // crude start (exact leading order in the tail)
  if (x > hi) x = hi;
  for (int it = 0; it < 200; ++it) {
    const long double Qx = upper_tail(x);
    const long double f = logl(Qx) - target;
    if (f > 0.0L) lo = x; else hi = x;
    // d/dx log Q(x) = -phi(x)/Q(x)
    const long double phi = 0.5L * kSqrt2OverPi * expl(-0.5L * x * x);
    long double xn = x + f * Qx / phi;
    if (!(xn > lo && xn < hi)) xn = 0.5L * (lo + hi);
    const long double dx = fabsl(xn - x);
    x = xn;
    if (dx <= 2e-19L * (1.0L + fabsl(x))) break;
  }
  return x;
}

// Phi^-1(u), u in (0,1).  1-u is exact for the uniforms produced by bits_to_unit.
double norm_inv(double u) {
  if (u <= 0.5) return (double)(-qinv_half((long double)u));
  return (double)qinv_half(1.0L - (long double)u);
}

// TNpos(m, u): the draw from N(m,1) truncated to (0, inf) by inverse survival function:
//   t = Q^-1(u Q(-m)),  w = m + t,  clamped to the smallest positive normal double so that the
//   sign invariant holds exactly even when rounding would give w <= 0.
double tnpos(double m, double u) {
  const long double a = -(long double)m;
  const long double Qa = upper_tail(a);
  const long double q = (long double)u * Qa;
  long double t;
  if (q <= 0.5L) {
    t = qinv_half(q);
  } else {
    // 1 - u Q(a) = (1-u) + u Q(-a), free of cancellation
    const long double pc = (1.0L - (long double)u) + (long double)u * upper_tail(-a);
    t = -qinv_half(pc);
  }
  double w = (double)((long double)m + t);
  if (!(w >= DBL_MIN)) w = DBL_MIN;
  return w;
}

// ----------------------------------------------------------------------------------------
// The paper's own truncated-normal samplers, used only as a cross-check of
// the target law (they consume a sequential private Philox stream, tag TAG_LITERAL).
// ----------------------------------------------------------------------------------------
struct SeqStream {
  uint64_t seed, idx; uint32_t sweep; uint64_t n = 0;
  double next() { double u; uniforms(seed ^ 0x5bf03635d1f4b7a1ull, idx + (n++ << 40), sweep, TAG_LITERAL, &u, nullptr); return u; }
};

double tnpos_rejection(double m, SeqStream& rs, long long* trials) {
  long long n = 0;
  if (m > 0.47) {                         // Gaussian rejection sampler
    for (;;) {
      ++n;
      const double prop = norm_inv(rs.next()) + m;
      if (prop > 0.0) { if (trials) *trials = n; return prop; }
    }
  }
  // exponential rejection sampler of Robert (1995), shifted to mean m and
  // truncation at 0 (reading R6): theta = (-m + sqrt(m^2+4))/2,
  // rho(w) = exp(-(w - m - theta)^2 / 2).
  const double theta = 0.5 * (-m + std::sqrt(m * m + 4.0));
  for (;;) {
    ++n;
    const double u1 = rs.next(), u2 = rs.next();
    const double prop = -std::log(u1) / theta;
    const double d = prop - m - theta;
    if (u2 < std::exp(-0.5 * d * d)) { if (trials) *trials = n; return prop; }
  }
}

// ----------------------------------------------------------------------------------------
// Gamma(alpha, 1), alpha > 1, by Cheng (1977) algorithm GB.  Trial t uses
// the two uniforms of Philox(idx=t, sweep, TAG_TAU); the result is the proposal of the smallest
// accepted t, which is what "32 lanes try, thread 1 scans for the first accepted" returns.
// ----------------------------------------------------------------------------------------
double cheng_gamma(double alpha, uint64_t seed, uint32_t sweep, long long* accepted_trial) {
  const double a = 1.0 / std::sqrt(2.0 * alpha - 1.0);
  const double b = alpha - std::log(4.0);
  const double c = alpha + 1.0 / a;
  for (uint64_t t = 0;; ++t) {
    double u1, u2;
    uniforms(seed, t, sweep, TAG_TAU, &u1, &u2);
    const double V = a * std::log(u1 / (1.0 - u1));
    const double X = alpha * std::exp(V);
    if (b + c * V - X >= 2.0 * std::log(u1) + std::log(u2)) {
      if (accepted_trial) *accepted_trial = (long long)t;
      return X;
    }
  }
}

// ----------------------------------------------------------------------------------------
// Dense linear algebra, textbook loops, row-major, lower triangle.
// ----------------------------------------------------------------------------------------
// In-place Cholesky A = L L^T (only the lower triangle is read and written).
// Returns 0, or j+1 if pivot j is not positive.
int cholesky_lower(double* A, int p) {
  for (int j = 0; j < p; ++j) {
    double d = A[(size_t)j * p + j];
    for (int k = 0; k < j; ++k) d -= A[(size_t)j * p + k] * A[(size_t)j * p + k];
    if (!(d > 0.0)) return j + 1;
    const double ljj = std::sqrt(d);
    A[(size_t)j * p + j] = ljj;
    for (int i = j + 1; i < p; ++i) {
      double s = A[(size_t)i * p + j];
      for (int k = 0; k < j; ++k) s -= A[(size_t)i * p + k] * A[(size_t)j * p + k];
      A[(size_t)i * p + j] = s / ljj;
    }
  }
  return 0;
}

void solve_lower(const double* L, int p, double* b) {       // L x = b, forward substitution
  for (int i = 0; i < p; ++i) {
    double s = b[i];
    for (int k = 0; k < i; ++k) s -= L[(size_t)i * p + k] * b[k];
    b[i] = s / L[(size_t)i * p + i];
  }
}

void solve_lower_t(const double* L, int p, double* b) {     // L^T x = b, back substitution
  for (int i = p - 1; i >= 0; --i) {
    double s = b[i];
    for (int k = i + 1; k < p; ++k) s -= L[(size_t)k * p + i] * b[k];
    b[i] = s / L[(size_t)i * p + i];
  }
}

enum { F32 = 0, F64 = 1 };
enum { FLAG_STORE_Z = 1u, FLAG_FREEZE_SCALES = 2u, FLAG_FREEZE_Z = 4u, FLAG_LITERAL_Z = 8u,
       FLAG_FREEZE_BETA = 16u, FLAG_ROW_CHUNKS = 32u };
constexpr int64_t kRowChunk = 4096;

struct Chain {
  const void* X; int dtype; const uint8_t* y; int64_t N; int p; uint64_t seed;
  unsigned flags = FLAG_STORE_Z;
  int64_t sweep = 0;
  std::vector<double> G, Lmat, beta, lam_inv2, nu_inv, z, g, eta;
  double tau_inv2 = 1.0, xi_inv = 1.0;
  std::vector<double> h_beta, h_lambda, h_tau;   // draws of the last sweep() call
  int64_t h_n = 0;
  double t_rows = 0.0, t_rest = 0.0;             // seconds spent in steps 1-3 / the rest
  long long literal_trials = 0;
  inline double x(int64_t i, int j) const {
    return dtype == F32 ? (double)((const float*)X)[(size_t)i * p + j]
                        : ((const double*)X)[(size_t)i * p + j];
  }
};

double now_s() {
  return std::chrono::duration<double>(std::chrono::steady_clock::now().time_since_epoch()).count();
}

int sweep_once(Chain& c) {
  const int p = c.p; const int64_t N = c.N;
  const uint32_t k = (uint32_t)(++c.sweep);
  const double t0 = now_s();
  if (!(c.flags & FLAG_FREEZE_Z) && (c.flags & FLAG_ROW_CHUNKS) && !(c.flags & FLAG_LITERAL_Z)) {
    // timing-only: steps 1-3 over fixed row chunks on all cores (see the header); same row arithmetic as below
    const int64_t n_chunks = (N + kRowChunk - 1) / kRowChunk;
    std::vector<double> part((size_t)n_chunks * p, 0.0);
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t ch = 0; ch < n_chunks; ++ch) {
      const int64_t i0 = ch * kRowChunk, i1 = std::min(N, i0 + kRowChunk);
      double* gp = part.data() + (size_t)ch * p;
      for (int64_t i = i0; i < i1; ++i) {
        double s = 0.0;
        for (int j = 0; j < p; ++j) s += c.x(i, j) * c.beta[j];
        c.eta[i] = s;
        const double ystar = 2.0 * (double)c.y[i] - 1.0;
        double u;
        uniforms(c.seed, (uint64_t)i, k, TAG_Z, &u, nullptr);
        const double zi = ystar * tnpos(ystar * s, u);
        c.z[i] = zi;
        for (int j = 0; j < p; ++j) gp[j] += c.x(i, j) * zi;
      }
    }
    for (int j = 0; j < p; ++j) c.g[j] = 0.0;
    for (int64_t ch = 0; ch < n_chunks; ++ch)
      for (int j = 0; j < p; ++j) c.g[j] += part[(size_t)ch * p + j];
  } else if (!(c.flags & FLAG_FREEZE_Z)) {
    // 1. eta = X beta
    for (int64_t i = 0; i < N; ++i) {
      double s = 0.0;
      for (int j = 0; j < p; ++j) s += c.x(i, j) * c.beta[j];
      c.eta[i] = s;
    }
    // 2. z_i = y*_i TNpos(y*_i eta_i)  with y* = 2y - 1
    for (int64_t i = 0; i < N; ++i) {
      const double ystar = 2.0 * (double)c.y[i] - 1.0;
      const double mstar = ystar * c.eta[i];
      double w;
      if (c.flags & FLAG_LITERAL_Z) {
        SeqStream rs{c.seed, (uint64_t)i, k};
        long long n = 0;
        w = tnpos_rejection(mstar, rs, &n);
        c.literal_trials += n;
      } else {
        double u;
        uniforms(c.seed, (uint64_t)i, k, TAG_Z, &u, nullptr);
        w = tnpos(mstar, u);
      }
      c.z[i] = ystar * w;
    }
    // 3. g = X^T z
    for (int j = 0; j < p; ++j) c.g[j] = 0.0;
    for (int64_t i = 0; i < N; ++i) {
      const double zi = c.z[i];
      for (int j = 0; j < p; ++j) c.g[j] += c.x(i, j) * zi;
    }
  }
  const double t1 = now_s();
  if (!(c.flags & FLAG_FREEZE_SCALES)) {
    // 4. local precisions from the previous beta, tau^-2, nu^-1
    for (int j = 0; j < p; ++j) {
      double u;
      uniforms(c.seed, (uint64_t)j, k, TAG_LAMBDA, &u, nullptr);
      const double rate = c.nu_inv[j] + 0.5 * c.tau_inv2 * c.beta[j] * c.beta[j];
      c.lam_inv2[j] = -std::log(u) / rate;
    }
    // 5. global precision
    double S = 0.0;
    for (int j = 0; j < p; ++j) S += c.lam_inv2[j] * c.beta[j] * c.beta[j];
    S *= 0.5;
    const double gam = cheng_gamma(0.5 * ((double)p + 1.0), c.seed, k, nullptr);
    c.tau_inv2 = gam / (c.xi_inv + S);
  }
  if (!(c.flags & FLAG_FREEZE_BETA)) {
  // 6. Q = G + diag(tau^-2 lam^-2), Cholesky
  for (int i = 0; i < p; ++i)
    for (int j = 0; j <= i; ++j) c.Lmat[(size_t)i * p + j] = c.G[(size_t)i * p + j];
  for (int j = 0; j < p; ++j) c.Lmat[(size_t)j * p + j] += c.tau_inv2 * c.lam_inv2[j];
  if (cholesky_lower(c.Lmat.data(), p) != 0) return -4;
  // 7. beta = Q^-1 g + L^-T e (reading R5)
  std::vector<double> v(c.g);
  solve_lower(c.Lmat.data(), p, v.data());
  for (int j = 0; j < p; ++j) {
    double u;
    uniforms(c.seed, (uint64_t)j, k, TAG_E, &u, nullptr);
    v[j] += norm_inv(u);
  }
  solve_lower_t(c.Lmat.data(), p, v.data());
  for (int j = 0; j < p; ++j) c.beta[j] = v[j];
  }
  if (!(c.flags & FLAG_FREEZE_SCALES)) {
    // 8. auxiliaries from the new lam^-2, tau^-2
    for (int j = 0; j < p; ++j) {
      double u;
      uniforms(c.seed, (uint64_t)j, k, TAG_NU, &u, nullptr);
      c.nu_inv[j] = -std::log(u) / (1.0 + c.lam_inv2[j]);
    }
    double u;
    uniforms(c.seed, 0, k, TAG_XI, &u, nullptr);
    c.xi_inv = -std::log(u) / (1.0 + c.tau_inv2);
  }
  const double t2 = now_s();
  c.t_rows += t1 - t0; c.t_rest += t2 - t1;
  for (int j = 0; j < p; ++j)
    if (!std::isfinite(c.beta[j]) || !std::isfinite(c.lam_inv2[j]) || !std::isfinite(c.nu_inv[j])) return -5;
  if (!std::isfinite(c.tau_inv2) || !std::isfinite(c.xi_inv)) return -5;
  return 0;
}

}  // namespace

extern "C" {

void hspo_philox4x32_10(const uint32_t* ctr, const uint32_t* key, uint32_t* out) { philox4x32_10(ctr, key, out); }
void hspo_uniforms(uint64_t seed, uint64_t idx, uint32_t sweep, uint32_t tag, double* ua, double* ub) { uniforms(seed, idx, sweep, tag, ua, ub); }
void hspo_philox_many(const uint32_t* ctr, const uint32_t* key, uint32_t* out, long long n) {
  for (long long i = 0; i < n; ++i) philox4x32_10(ctr + 4 * i, key + 2 * i, out + 4 * i);
}
void hspo_uniforms_many(uint64_t seed, const uint64_t* idx, uint32_t sweep, uint32_t tag, double* ua, double* ub, long long n) {
  for (long long i = 0; i < n; ++i) uniforms(seed, idx[i], sweep, tag, ua ? ua + i : nullptr, ub ? ub + i : nullptr);
}
void hspo_norm_inv_many(const double* u, double* x, long long n) { for (long long i = 0; i < n; ++i) x[i] = norm_inv(u[i]); }
double hspo_qinv(double q) { return q <= 0.5 ? (double)qinv_half(q) : (double)(-qinv_half(1.0L - (long double)q)); }
double hspo_norm_inv(double u) { return norm_inv(u); }
double hspo_tnpos(double m, double u) { return tnpos(m, u); }
void hspo_tnpos_many(const double* m, const double* u, double* w, long long n) { for (long long i = 0; i < n; ++i) w[i] = tnpos(m[i], u[i]); }
double hspo_tnpos_rejection(double m, uint64_t seed, uint64_t idx, uint32_t sweep, long long* trials) {
  SeqStream rs{seed, idx, sweep};
  return tnpos_rejection(m, rs, trials);
}
double hspo_cheng_gamma(double alpha, uint64_t seed, uint32_t sweep, long long* accepted_trial) { return cheng_gamma(alpha, seed, sweep, accepted_trial); }
int hspo_cholesky_lower(double* A, int p) { return cholesky_lower(A, p); }
void hspo_solve_lower(const double* L, int p, double* b) { solve_lower(L, p, b); }
void hspo_solve_lower_t(const double* L, int p, double* b) { solve_lower_t(L, p, b); }

// X, y are HOST pointers, borrowed.  gram: optional HOST p*p row-major X^T X (lower triangle
// read); if NULL it is computed here by the triple loop.
void* hspo_create(const void* X, int dtype, const unsigned char* y, long long N, int p,
                  unsigned long long seed, const double* gram) {
  if (!X || !y || N < 2 || p < 1 || (dtype != F32 && dtype != F64)) return nullptr;
  for (long long i = 0; i < N; ++i) if (y[i] > 1) return nullptr;
  Chain* c = new (std::nothrow) Chain();
  if (!c) return nullptr;
  c->X = X; c->dtype = dtype; c->y = y; c->N = N; c->p = p; c->seed = seed;
  c->G.assign((size_t)p * p, 0.0); c->Lmat.assign((size_t)p * p, 0.0);
  c->beta.assign(p, 0.0); c->lam_inv2.assign(p, 1.0); c->nu_inv.assign(p, 1.0);
  c->z.assign(N, 0.0); c->g.assign(p, 0.0); c->eta.assign(N, 0.0);
  if (gram) {
    for (int i = 0; i < p; ++i) for (int j = 0; j <= i; ++j) c->G[(size_t)i * p + j] = gram[(size_t)i * p + j];
  } else {
    for (long long i = 0; i < N; ++i)
      for (int a = 0; a < p; ++a) {
        const double xa = c->x(i, a);
        for (int b = 0; b <= a; ++b) c->G[(size_t)a * p + b] += xa * c->x(i, b);
      }
  }
  return c;
}

void hspo_destroy(void* s) { delete (Chain*)s; }

int hspo_set_flags(void* s, unsigned flags) { ((Chain*)s)->flags = flags; return 0; }

int hspo_sweep(void* s, long long n_iter) {
  Chain& c = *(Chain*)s;
  if (n_iter < 0) return -1;
  c.h_n = n_iter;
  c.h_beta.assign((size_t)n_iter * c.p, 0.0); c.h_lambda.assign((size_t)n_iter * c.p, 0.0); c.h_tau.assign(n_iter, 0.0);
  for (long long it = 0; it < n_iter; ++it) {
    const int rc = sweep_once(c);
    if (rc != 0) return rc;
    // 9. emit beta, lambda_j = (lam_j^-2)^-1/2, tau = (tau^-2)^-1/2
    for (int j = 0; j < c.p; ++j) {
      c.h_beta[(size_t)it * c.p + j] = c.beta[j];
      c.h_lambda[(size_t)it * c.p + j] = 1.0 / std::sqrt(c.lam_inv2[j]);
    }
    c.h_tau[it] = 1.0 / std::sqrt(c.tau_inv2);
  }
  return 0;
}

int hspo_get_draws(const void* s, double* beta, double* lambda, double* tau) {
  const Chain& c = *(const Chain*)s;
  if (beta) std::memcpy(beta, c.h_beta.data(), c.h_beta.size() * sizeof(double));
  if (lambda) std::memcpy(lambda, c.h_lambda.data(), c.h_lambda.size() * sizeof(double));
  if (tau) std::memcpy(tau, c.h_tau.data(), c.h_tau.size() * sizeof(double));
  return 0;
}

int hspo_get_latent(const void* s, double* z, signed char* side) {
  const Chain& c = *(const Chain*)s;
  if (z) std::memcpy(z, c.z.data(), c.z.size() * sizeof(double));
  if (side) for (long long i = 0; i < c.N; ++i) side[i] = (signed char)(2 * (int)c.y[i] - 1);
  return 0;
}

int hspo_set_latent(void* s, const double* z) {     // also refreshes g = X^T z
  Chain& c = *(Chain*)s;
  std::memcpy(c.z.data(), z, c.z.size() * sizeof(double));
  for (int j = 0; j < c.p; ++j) c.g[j] = 0.0;
  for (long long i = 0; i < c.N; ++i) for (int j = 0; j < c.p; ++j) c.g[j] += c.x(i, j) * c.z[i];
  return 0;
}

int hspo_get_xtz(const void* s, double* g) { const Chain& c = *(const Chain*)s; std::memcpy(g, c.g.data(), c.p * sizeof(double)); return 0; }
int hspo_get_eta(const void* s, double* eta) { const Chain& c = *(const Chain*)s; std::memcpy(eta, c.eta.data(), c.N * sizeof(double)); return 0; }
int hspo_get_gram(const void* s, double* G) { const Chain& c = *(const Chain*)s; std::memcpy(G, c.G.data(), c.G.size() * sizeof(double)); return 0; }
int hspo_get_chol(const void* s, double* L) { const Chain& c = *(const Chain*)s; std::memcpy(L, c.Lmat.data(), c.Lmat.size() * sizeof(double)); return 0; }

int hspo_get_state(const void* s, double* beta, double* lam_inv2, double* nu_inv, double* tau_inv2,
                   double* xi_inv, long long* sweep) {
  const Chain& c = *(const Chain*)s;
  if (beta) std::memcpy(beta, c.beta.data(), c.p * sizeof(double));
  if (lam_inv2) std::memcpy(lam_inv2, c.lam_inv2.data(), c.p * sizeof(double));
  if (nu_inv) std::memcpy(nu_inv, c.nu_inv.data(), c.p * sizeof(double));
  if (tau_inv2) *tau_inv2 = c.tau_inv2;
  if (xi_inv) *xi_inv = c.xi_inv;
  if (sweep) *sweep = c.sweep;
  return 0;
}

int hspo_set_state(void* s, const double* beta, const double* lam_inv2, const double* nu_inv,
                   const double* tau_inv2, const double* xi_inv, long long sweep) {
  Chain& c = *(Chain*)s;
  if (beta) std::memcpy(c.beta.data(), beta, c.p * sizeof(double));
  if (lam_inv2) std::memcpy(c.lam_inv2.data(), lam_inv2, c.p * sizeof(double));
  if (nu_inv) std::memcpy(c.nu_inv.data(), nu_inv, c.p * sizeof(double));
  if (tau_inv2) c.tau_inv2 = *tau_inv2;
  if (xi_inv) c.xi_inv = *xi_inv;
  if (sweep >= 0) c.sweep = sweep;
  return 0;
}

// seconds accumulated in steps 1-3 (the O(N p) row work) and in the rest (O(p^3) and O(p))
int hspo_get_timing(const void* s, double* t_rows, double* t_rest) {
  const Chain& c = *(const Chain*)s;
  if (t_rows) *t_rows = c.t_rows;
  if (t_rest) *t_rest = c.t_rest;
  return 0;
}
long long hspo_get_literal_trials(const void* s) { return ((const Chain*)s)->literal_trials; }
// threads the FLAG_ROW_CHUNKS mode uses (1 when built without OpenMP)
int hspo_max_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

}  // extern "C"
