// paper_design.cu -- SURVEY.md 8(f) NEXT-2: the PAPER'S OWN decomposition of rows a1-a3, written as plain CUDA so
// that the fused pass can be measured against it on the same box (an A/B, selected by the flag HSP_PAPER_DESIGN):
//   1. mu = X beta                      one matrix-vector product (the paper: cublasSgemv)
//   2. z_i by rejection, thread per row the paper's two samplers split at mu* = 0.47, with its warp
//                                       divergence (Gaussian proposal / Robert's exponential proposal)
//   3. g = X^T z                        a second matrix-vector product: X is read from HBM TWICE
// The rejection sampler consumes a private sequential Philox stream per row (counter layout of the oracle's
// paper-literal mode: key seed ^ C, idx = i + (n << 40), tag LITERAL), so the draws differ from the fused pass
// (inverse CDF) but have the same law (R6, R16).  mu and z are materialised in HBM (fp64), as in the paper.
#include <cuda_runtime.h>
#include <cstdint>
#include "hsp_device.cuh"
#include "hsp_internal.h"

namespace hsp {

constexpr uint32_t TAG_LITERAL = 6;
constexpr unsigned long long kLiteralKeyXor = 0x5bf03635d1f4b7a1ull;

// 1. mu_i = x_i . beta: one warp per row, 16-byte loads; fp32 X: fp32 chains of 4 added in fp64, fp64 X: DFMA.
template <typename XT>
__global__ void __launch_bounds__(256)
pd_gemv_kernel(const XT* __restrict__ X, long long N, int p, const double* __restrict__ beta, double* __restrict__ mu) {
  constexpr int V = 16 / sizeof(XT);
  const int lane = threadIdx.x & 31;
  const long long warp0 = (long long)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
  const long long nwarps = (long long)gridDim.x * (blockDim.x >> 5);
  const bool vec = (p % V == 0) && ((reinterpret_cast<uintptr_t>(X) & 15) == 0);
  for (long long i = warp0; i < N; i += nwarps) {
    const XT* xr = X + (size_t)i * p;
    double s = 0.0;
    if (vec) {
      for (int j = lane * V; j < p; j += 32 * V) {
        if constexpr (sizeof(XT) == 4) {
          // fp32 chain of 4, converted once (the arithmetic of the fused pass's eta phase)
          const float4 x = *reinterpret_cast<const float4*>(xr + j);
          float c = x.x * (float)beta[j];
          c = fmaf(x.y, (float)beta[j + 1], c); c = fmaf(x.z, (float)beta[j + 2], c); c = fmaf(x.w, (float)beta[j + 3], c);
          s += (double)c;
        } else {
          const double2 x = *reinterpret_cast<const double2*>(xr + j);
          s = fma(x.x, beta[j], s); s = fma(x.y, beta[j + 1], s);
        }
      }
    } else {
      for (int j = lane; j < p; j += 32) s = fma((double)xr[j], beta[j], s);
    }
#pragma unroll
    for (int off = 16; off >= 1; off >>= 1) s += __shfl_xor_sync(0xffffffffu, s, off);
    if (lane == 0) mu[i] = s;
  }
}

__device__ __forceinline__ double literal_next(unsigned long long key, unsigned long long i, unsigned long long& n, uint32_t sweep) {
  const double u = uniform_a(key, i + (n << 40), sweep, TAG_LITERAL);
  ++n;
  return u;
}

// 2. the paper's rejection samplers (divergent loops, one thread per row).
__global__ void __launch_bounds__(256)
pd_tn_rejection_kernel(const double* __restrict__ mu, const unsigned char* __restrict__ y, long long N,
                       unsigned long long seed, const Ctl* __restrict__ ctl, double* __restrict__ z) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= N) return;
  const uint32_t sweep = (uint32_t)(ctl->sweep + 1ull);
  const unsigned long long key = seed ^ kLiteralKeyXor;
  const double ystar = 2.0 * (double)y[i] - 1.0;
  const double m = ystar * mu[i];
  unsigned long long n = 0;
  double w;
  if (m > 0.47) {                                    // Gaussian proposal
    for (;;) {
      w = norm_inv(literal_next(key, (unsigned long long)i, n, sweep)) + m;
      if (w > 0.0) break;
    }
  } else {                                           // Robert's exponential proposal (reading R6)
    const double theta = 0.5 * (-m + sqrt(m * m + 4.0));
    for (;;) {
      const double u1 = literal_next(key, (unsigned long long)i, n, sweep);
      const double u2 = literal_next(key, (unsigned long long)i, n, sweep);
      w = -log(u1) / theta;
      const double d = w - m - theta;
      if (u2 < exp(-0.5 * d * d)) break;
    }
  }
  z[i] = ystar * w;
}

// 3. g = X^T z: CTA c owns the row range [c R, (c+1) R); thread t owns the columns t, t+256, ... (coalesced
// across the CTA), fp64 accumulation; per-CTA partials are summed by reduce_partials_kernel (fixed order).
constexpr int kPdMaxC = 4, kPdRows = 8;
template <typename XT>
__global__ void __launch_bounds__(256)
pd_gemvt_kernel(const XT* __restrict__ X, long long N, int p, const double* __restrict__ z, double* __restrict__ partial,
                long long rows_per_cta) {
  const long long r0 = (long long)blockIdx.x * rows_per_cta;
  const long long r1 = (r0 + rows_per_cta < N) ? r0 + rows_per_cta : N;
  for (int j0 = 0; j0 < p; j0 += 256 * kPdMaxC) {
    double acc[kPdMaxC];
    bool on[kPdMaxC];
#pragma unroll
    for (int c = 0; c < kPdMaxC; ++c) { acc[c] = 0.0; on[c] = j0 + c * 256 + (int)threadIdx.x < p; }
    const XT* xc = X + j0 + threadIdx.x;
    for (long long i = r0; i < r1; i += kPdRows) {
      XT x[kPdRows][kPdMaxC];
      double zi[kPdRows];
#pragma unroll
      for (int r = 0; r < kPdRows; ++r) {            // all loads of 8 rows first: 32 independent loads in flight
        const bool live = i + r < r1;
        zi[r] = live ? z[i + r] : 0.0;
        const XT* xr = xc + (size_t)(live ? i + r : r0) * p;
#pragma unroll
        for (int c = 0; c < kPdMaxC; ++c) x[r][c] = on[c] ? xr[c * 256] : (XT)0;
      }
#pragma unroll
      for (int r = 0; r < kPdRows; ++r)
#pragma unroll
        for (int c = 0; c < kPdMaxC; ++c) acc[c] = fma((double)x[r][c], zi[r], acc[c]);
    }
#pragma unroll
    for (int c = 0; c < kPdMaxC; ++c)
      if (on[c]) partial[(size_t)blockIdx.x * p + j0 + c * 256 + threadIdx.x] = acc[c];
  }
}

int paper_design_ctas(long long N, int num_sms) {
  long long c = (long long)num_sms * 8;
  if (c > (N + 63) / 64) c = (N + 63) / 64;
  return (int)(c < 1 ? 1 : c);
}

cudaError_t paper_design_launch(const void* X, int dtype, const unsigned char* y, long long N, int p, unsigned long long seed,
                                const double* beta, const Ctl* ctl, double* mu, double* z, double* partial, int n_part,
                                int num_sms, cudaStream_t st) {
  const int gemv_grid = num_sms * 8;
  const long long rows_per_cta = (N + n_part - 1) / n_part;
  if (dtype == kF32) pd_gemv_kernel<float><<<gemv_grid, 256, 0, st>>>(static_cast<const float*>(X), N, p, beta, mu);
  else pd_gemv_kernel<double><<<gemv_grid, 256, 0, st>>>(static_cast<const double*>(X), N, p, beta, mu);
  pd_tn_rejection_kernel<<<(unsigned)((N + 255) / 256), 256, 0, st>>>(mu, y, N, seed, ctl, z);
  if (dtype == kF32)
    pd_gemvt_kernel<float><<<n_part, 256, 0, st>>>(static_cast<const float*>(X), N, p, z, partial, rows_per_cta);
  else
    pd_gemvt_kernel<double><<<n_part, 256, 0, st>>>(static_cast<const double*>(X), N, p, z, partial, rows_per_cta);
  return cudaGetLastError();
}

}  // namespace hsp
