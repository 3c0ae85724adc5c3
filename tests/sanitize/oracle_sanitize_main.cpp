// Driver for tests/test_oracle_sanitizers.py: the oracle (oracle/hsp_oracle.cpp, included as one translation unit) under
// AddressSanitizer + UndefinedBehaviorSanitizer on a small synthetic problem -- every sweep mode, the getters, the
// special functions at the ends of their ranges, a non-positive-definite factorisation.  Holds no arithmetic of the method:
// the inputs come from a linear congruential generator.
#include "../../oracle/hsp_oracle.cpp"
#include <cstdio>
#include <vector>

static unsigned long long lcg_state = 12345;
static double lcg_unit() { lcg_state = lcg_state * 6364136223846793005ull + 1442695040888963407ull; return ((lcg_state >> 11) + 0.5) / 9007199254740992.0; }

template <typename T>
static int run(int dtype, long long N, int p, unsigned flags, int sweeps) {
  std::vector<T> X((size_t)N * p);
  std::vector<unsigned char> y(N);
  for (auto& v : X) v = (T)(2.0 * lcg_unit() - 1.0);
  for (long long i = 0; i < N; ++i) y[i] = (X[(size_t)i * p] + 0.3 * (2.0 * lcg_unit() - 1.0)) > 0;
  void* c = hspo_create(X.data(), dtype, y.data(), N, p, 7, nullptr);
  if (!c) return 1;
  hspo_set_flags(c, flags | 1u);
  if (hspo_sweep(c, sweeps) != 0) return 2;
  std::vector<double> b((size_t)sweeps * p), l((size_t)sweeps * p), t(sweeps), z(N), g(p), eta(N), G((size_t)p * p), L((size_t)p * p);
  std::vector<signed char> side(N);
  hspo_get_draws(c, b.data(), l.data(), t.data());
  hspo_get_latent(c, z.data(), side.data());
  hspo_get_xtz(c, g.data()); hspo_get_eta(c, eta.data()); hspo_get_gram(c, G.data()); hspo_get_chol(c, L.data());
  std::vector<double> sb(p), sl(p), sn(p); double ti, xi; long long k;
  hspo_get_state(c, sb.data(), sl.data(), sn.data(), &ti, &xi, &k);
  hspo_set_state(c, sb.data(), sl.data(), sn.data(), &ti, &xi, k);
  hspo_set_latent(c, z.data());
  if (hspo_sweep(c, 2) != 0) return 3;
  for (long long i = 0; i < N; ++i) if (!(z[i] * side[i] > 0.0)) return 4;
  hspo_destroy(c);
  return 0;
}

int main() {
  int rc = 0;
  rc |= run<double>(1, 257, 7, 0u, 6);            // default (inverse-CDF) mode, fp64 X
  rc |= run<float>(0, 300, 5, 0u, 5);             // fp32 X
  rc |= run<double>(1, 129, 3, 8u, 5);            // the paper's rejection samplers
  rc |= run<float>(0, 9000, 4, 32u, 3);           // row chunks (OpenMP), more than two chunks of 4096 rows
  rc |= run<double>(1, 2, 1, 0u, 3);              // smallest problem
  // special functions at the ends of their ranges
  const double ms[] = {-100.0, -37.0, -8.0, 0.0, 0.47, 8.0, 100.0};
  const double us[] = {1.1102230246251565e-16, 1e-9, 0.5, 1.0 - 1e-9, 1.0 - 1.1102230246251565e-16};
  for (double m : ms) for (double u : us) if (!(hspo_tnpos(m, u) > 0.0)) rc |= 16;
  for (double u : us) { volatile double x = hspo_norm_inv(u); (void)x; }
  long long tr = 0;
  for (double a : {1.5, 5.5, 500.5, 2000.5}) if (!(hspo_cheng_gamma(a, 3, 1, &tr) > 0.0)) rc |= 32;
  for (double m : {-3.0, 0.2, 0.47, 0.9, 4.0}) if (!(hspo_tnpos_rejection(m, 5, 11, 2, &tr) > 0.0)) rc |= 64;
  double A[4] = {1.0, 2.0, 2.0, 1.0};             // not positive definite: must be reported, not crash
  if (hspo_cholesky_lower(A, 2) == 0) rc |= 128;
  std::printf(rc == 0 ? "ok\n" : "FAILED rc=%d\n", rc);
  return rc;
}
