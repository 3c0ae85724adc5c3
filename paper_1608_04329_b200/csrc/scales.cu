// scales.cu -- rows e1, e2, e3 and g of the hot-path table: the horseshoe scale conditionals of
// eq. (12) exactly as PAPER.md:174-184 states them (with reading R1: tau^-2 is Gamma), by the
// inversion -ln(u)/rate and Cheng's gamma sampler, plus the
// append of (lambda, tau) to the device history (beta is appended by beta_gemv2_kernel).
#include <cuda_runtime.h>
#include <cstdint>
#include "hsp_device.cuh"
#include "hsp_internal.h"

namespace hsp {

constexpr int kScaleThreads = 1024;

// e1, e2 ("z and lambda^-2 in parallel, followed by tau^-2"; both use the OLD beta), then e3
// (nu^-1 and xi^-1 "in parallel" with beta: they depend on the NEW lambda^-2, tau^-2 only, not
// on beta, so they are drawn here, off the critical path), then row g for lambda and tau.  One CTA.
__global__ void __launch_bounds__(kScaleThreads)
scales_kernel(const double* __restrict__ beta, double* __restrict__ lam_inv2, double* __restrict__ nu_inv,
              Ctl* __restrict__ ctl, int p, unsigned long long seed, int freeze_scales) {
  __shared__ double red[kScaleThreads];
  const int tid = threadIdx.x;
  const unsigned long long k = ctl->sweep + 1ull;
  const uint32_t sweep = (uint32_t)k;
  double* __restrict__ h_lambda = ctl->h_lambda;
  double* __restrict__ h_tau = ctl->h_tau;
  const unsigned long long hrow = k - 1ull - ctl->hist_base;
  const double tau_old = ctl->tau_inv2;
  double s = 0.0;
  bool bad = false;
  for (int j = tid; j < p; j += kScaleThreads) {
    double l = lam_inv2[j];
    if (!freeze_scales) {
      const double u = uniform_a(seed, (unsigned long long)j, sweep, TAG_LAMBDA);
      const double b = beta[j];
      const double rate = nu_inv[j] + 0.5 * tau_old * b * b;
      l = -log(u) / rate;
      lam_inv2[j] = l;
      s += l * b * b;
      const double un = uniform_a(seed, (unsigned long long)j, sweep, TAG_NU);
      const double n = -log(un) / (1.0 + l);
      nu_inv[j] = n;
      bad |= !isfinite(l) || !isfinite(n);
    }
    if (h_lambda != nullptr) h_lambda[hrow * (unsigned long long)p + j] = 1.0 / sqrt(l);
  }
  double tau_new = tau_old;
  if (!freeze_scales) {
    red[tid] = s;
    __syncthreads();
    for (int off = kScaleThreads / 2; off > 0; off >>= 1) {      // fixed tree: deterministic
      if (tid < off) red[tid] += red[tid + off];
      __syncthreads();
    }
    if (tid < 32) {
      const double gam = cheng_gamma_warp(0.5 * ((double)p + 1.0), seed, sweep);
      if (tid == 0) {
        tau_new = gam / (ctl->xi_inv + 0.5 * red[0]);
        ctl->tau_inv2 = tau_new;
        const double u = uniform_a(seed, 0ull, sweep, TAG_XI);
        const double x = -log(u) / (1.0 + tau_new);
        ctl->xi_inv = x;
        if (!isfinite(tau_new) || !isfinite(x)) bad = true;
      }
    }
  }
  if (tid == 0 && h_tau != nullptr) h_tau[hrow] = 1.0 / sqrt(tau_new);
  if (bad) atomicCAS(&ctl->status, 0, -5);
}

__global__ void set_history_kernel(Ctl* ctl, unsigned long long hist_base, double* hb, double* hl, double* ht) {
  ctl->hist_base = hist_base; ctl->h_beta = hb; ctl->h_lambda = hl; ctl->h_tau = ht;
}

__global__ void validate_y_kernel(const unsigned char* __restrict__ y, long long N, int* __restrict__ bad) {
  const long long stride = (long long)gridDim.x * blockDim.x;
  bool b = false;
  for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < N; i += stride) b |= y[i] > 1;
  if (b) *bad = 1;
}

__global__ void side_kernel(const unsigned char* __restrict__ y, long long N, signed char* __restrict__ side) {
  const long long stride = (long long)gridDim.x * blockDim.x;
  for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < N; i += stride)
    side[i] = (signed char)(2 * (int)y[i] - 1);
}

cudaError_t scales_launch(const double* beta, double* lam_inv2, double* nu_inv, Ctl* ctl, int p, unsigned long long seed,
                          int freeze_scales, cudaStream_t st) {
  scales_kernel<<<1, kScaleThreads, 0, st>>>(beta, lam_inv2, nu_inv, ctl, p, seed, freeze_scales);
  return cudaGetLastError();
}

cudaError_t set_history_launch(Ctl* ctl, unsigned long long hist_base, double* hb, double* hl, double* ht, cudaStream_t st) {
  set_history_kernel<<<1, 1, 0, st>>>(ctl, hist_base, hb, hl, ht);
  return cudaGetLastError();
}

cudaError_t validate_y_launch(const unsigned char* y, long long N, int* bad, cudaStream_t st) {
  validate_y_kernel<<<296, 256, 0, st>>>(y, N, bad);
  return cudaGetLastError();
}

cudaError_t side_launch(const unsigned char* y, long long N, signed char* side, cudaStream_t st) {
  side_kernel<<<296, 256, 0, st>>>(y, N, side);
  return cudaGetLastError();
}

}  // namespace hsp
