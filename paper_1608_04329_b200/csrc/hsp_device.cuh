// hsp_device.cuh -- device-side random numbers and variate maps of the Horseshoe-Probit sweep.
//
// Random-number contract (the paper only says "use Philox"):
// Philox-4x32-10, counter = (idx_lo, idx_hi, sweep, tag), key = (seed_lo, seed_hi); one call per
// variate.  U_A = (52 bits of (r0,r1) + 1/2) * 2^-52, U_B likewise from (r2,r3).
#pragma once
#include <cstdint>
#include <cfloat>

namespace hsp {

enum : uint32_t { TAG_Z = 0, TAG_LAMBDA = 1, TAG_TAU = 2, TAG_E = 3, TAG_NU = 4, TAG_XI = 5 };

struct U4 { uint32_t x, y, z, w; };

__device__ __forceinline__ U4 philox4x32_10(U4 c, uint32_t k0, uint32_t k1) {
#pragma unroll
  for (int r = 0; r < 10; ++r) {
    const uint32_t hi0 = __umulhi(0xD2511F53u, c.x), lo0 = 0xD2511F53u * c.x;
    const uint32_t hi1 = __umulhi(0xCD9E8D57u, c.z), lo1 = 0xCD9E8D57u * c.z;
    U4 n;
    n.x = hi1 ^ c.y ^ k0;
    n.y = lo1;
    n.z = hi0 ^ c.w ^ k1;
    n.w = lo0;
    c = n;
    k0 += 0x9E3779B9u;
    k1 += 0xBB67AE85u;
  }
  return c;
}

__device__ __forceinline__ double bits_to_unit(uint32_t hi, uint32_t lo) {
  const unsigned long long n = ((unsigned long long)hi << 20) | (unsigned long long)(lo >> 12);
  return ((double)n + 0.5) * 0x1.0p-52;     // exact: (2n+1) * 2^-53
}

__device__ __forceinline__ U4 variate_bits(unsigned long long seed, unsigned long long idx, uint32_t sweep,
                                           uint32_t tag) {
  U4 c;
  c.x = (uint32_t)idx; c.y = (uint32_t)(idx >> 32); c.z = sweep; c.w = tag;
  return philox4x32_10(c, (uint32_t)seed, (uint32_t)(seed >> 32));
}

__device__ __forceinline__ double uniform_a(unsigned long long seed, unsigned long long idx, uint32_t sweep,
                                            uint32_t tag) {
  const U4 r = variate_bits(seed, idx, sweep, tag);
  return bits_to_unit(r.x, r.y);
}

// Phi^-1(u) for u in (0,1); 1-u is exact for our uniforms, so the upper half mirrors the lower.
__device__ __forceinline__ double norm_inv(double u) {
  const bool up = u > 0.5;
  const double x = normcdfinv(up ? 1.0 - u : u);
  return up ? -x : x;
}

// Exponential-tail form of TNpos for a = -m large (Q(a) would underflow): solve
//   log Q(a+w) - log Q(a) = log u   for w > 0
// with Q(x) = erfcx(x/sqrt2) exp(-x^2/2) / 2, by Newton from w0 = L/(sqrt(a^2+L)+a), L = -2 ln u.
// d/dw log Q(a+w) = -sqrt(2/pi)/erfcx((a+w)/sqrt2).  Start error is O(1/a^2) relative and the
// iteration converges quadratically: 4 steps reach fp64 for a >= 8.
__device__ __forceinline__ double tnpos_tail(double a, double u) {
  const double lnu = log(u);
  const double L = -2.0 * lnu;
  const double ea = erfcx(a * 0.70710678118654752440);
  const double lea = log(ea);
  double w = L / (sqrt(fma(a, a, L)) + a);
#pragma unroll
  for (int it = 0; it < 4; ++it) {
    const double ex = erfcx((a + w) * 0.70710678118654752440);
    const double h = -w * fma(0.5, w, a) + (log(ex) - lea) - lnu;
    w = fma(h, ex * 1.2533141373155002512, w);   // w - h/h', 1/h' = -erfcx*sqrt(pi/2)
    w = fmax(w, 0.0);
  }
  return w;
}

// TNpos(m,u): N(m,1) truncated to (0,inf) by inverse survival function, t = Q^-1(u Q(-m)),
// w = m + t, clamped to DBL_MIN.  Branch-free except for a warp-uniform vote
// that skips the tail form when no lane needs it.
#define HSP_TN_TAIL_A 30.0
__device__ __forceinline__ double tnpos(double m, double u) {
  const double a = -m;
  const double he = 0.5 * erfc(fabs(a) * 0.70710678118654752440);   // Q(|a|) in (0, 1/2]
  const bool neg = a < 0.0;
  const double Qa = neg ? 1.0 - he : he;
  const double q = u * Qa;
  const double pc = (1.0 - u) + u * he;            // 1 - q when a < 0, free of cancellation
  const bool lower = neg && (q > 0.5);
  const double t0 = normcdfinv(lower ? pc : q);    // <= 0
  double w = m + (lower ? t0 : -t0);
  const bool tail = a > HSP_TN_TAIL_A;
  if (__any_sync(__activemask(), tail)) {
    const double wt = tnpos_tail(tail ? a : HSP_TN_TAIL_A + 1.0, u);
    w = tail ? wt : w;
  }
  return fmax(w, DBL_MIN);
}

// Gamma(alpha,1), alpha > 1, Cheng (1977) GB with the first accepted trial.
// Must be called by all 32 lanes of a warp; lane l of round r evaluates trial 32 r + l.
__device__ __forceinline__ double cheng_gamma_warp(double alpha, unsigned long long seed, uint32_t sweep) {
  const int lane = threadIdx.x & 31;
  const double a = 1.0 / sqrt(2.0 * alpha - 1.0);
  const double b = alpha - 1.3862943611198906188;   // ln 4
  const double c = alpha + 1.0 / a;
  for (unsigned long long round = 0;; ++round) {
    const U4 r = variate_bits(seed, round * 32ull + lane, sweep, TAG_TAU);
    const double u1 = bits_to_unit(r.x, r.y), u2 = bits_to_unit(r.z, r.w);
    const double V = a * log(u1 / (1.0 - u1));
    const double X = alpha * exp(V);
    const bool ok = b + c * V - X >= 2.0 * log(u1) + log(u2);
    const unsigned m = __ballot_sync(0xffffffffu, ok);
    if (m) return __shfl_sync(0xffffffffu, X, __ffs(m) - 1);
  }
}

}  // namespace hsp
