// gram.cu -- row c0 of the hot-path table: G = X^T X, computed once at create (PAPER.md:195,
// "Precompute X^T X before starting the algorithm").  fp64 accumulation of exact products
// (an fp32 x fp32 product is exact in fp64), lower-triangular 64x64 tiles, split over row ranges
// with a fixed-order reduction of the splits (deterministic).
#include <cuda_runtime.h>
#include <cstdint>
#include "hsp_internal.h"

namespace hsp {

constexpr int kGT = 64;   // tile edge
constexpr int kGK = 16;   // rows per smem chunk

template <typename XT>
__global__ void __launch_bounds__(256)
gram_kernel(const XT* __restrict__ X, long long N, int p, double* __restrict__ out, int slot0,
            long long rows_per_split) {
  __shared__ double As[kGK][kGT + 4];
  __shared__ double Bs[kGK][kGT + 4];
  // linear lower-triangular tile index -> (ti >= tj)
  int t = blockIdx.x, ti = 0;
  while (t >= ti + 1) { t -= ti + 1; ++ti; }
  const int tj = t;
  const int tid = threadIdx.x, tx = tid & 15, ty = tid >> 4;
  const long long r_begin = (long long)(slot0 + blockIdx.y) * rows_per_split;     // slot q owns rows [q rps, (q+1) rps)
  const long long r_end = (r_begin + rows_per_split < N) ? r_begin + rows_per_split : N;
  double acc[4][4];
#pragma unroll
  for (int i = 0; i < 4; ++i)
#pragma unroll
    for (int j = 0; j < 4; ++j) acc[i][j] = 0.0;
  const int lc = tid & 63, lr = tid >> 6;            // loader: 64 columns x 4 rows per pass
  const int ca = ti * kGT + lc, cb = tj * kGT + lc;
  for (long long r0 = r_begin; r0 < r_end; r0 += kGK) {
#pragma unroll
    for (int q = 0; q < kGK / 4; ++q) {
      const int kk = q * 4 + lr;
      const long long r = r0 + kk;
      const bool ok = r < r_end;
      As[kk][lc] = (ok && ca < p) ? (double)X[(size_t)r * p + ca] : 0.0;
      Bs[kk][lc] = (ok && cb < p) ? (double)X[(size_t)r * p + cb] : 0.0;
    }
    __syncthreads();
#pragma unroll
    for (int kk = 0; kk < kGK; ++kk) {
      double a[4], b[4];
#pragma unroll
      for (int i = 0; i < 4; ++i) { a[i] = As[kk][ty * 4 + i]; b[i] = Bs[kk][tx * 4 + i]; }
#pragma unroll
      for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) acc[i][j] = fma(a[i], b[j], acc[i][j]);
    }
    __syncthreads();
  }
  double* dst = out + (size_t)(slot0 + blockIdx.y) * p * p;
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const int a = ti * kGT + ty * 4 + i;
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      const int b = tj * kGT + tx * 4 + j;
      if (a < p && b < p && b <= a) dst[(size_t)a * p + b] = acc[i][j];
    }
  }
}

__global__ void gram_reduce_kernel(const double* __restrict__ part, int splits, int p, double* __restrict__ G) {
  const size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= (size_t)p * p) return;
  const int a = (int)(idx / p), b = (int)(idx % p);
  if (b > a) { G[idx] = 0.0; return; }
  double s = 0.0;
  for (int q = 0; q < splits; ++q) s += part[(size_t)q * p * p + idx];
  G[idx] = s;
}

__global__ void gram_mirror_kernel(double* __restrict__ G, int p) {
  const size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= (size_t)p * p) return;
  const int a = (int)(idx / p), b = (int)(idx % p);
  if (b > a) G[idx] = G[(size_t)b * p + a];
}

// Row partition of the Gram: `slots` equal row ranges (a multiple of 16 rows each), each accumulated on its own and
// summed in slot order.  Enough slots to fill the SMs; and, for large X, at least 16 so that hsp_create_host can
// overlap the upload of row chunk c+1 with the Gram of chunk c.  The partition depends only on (N, p, dtype, SMs):
// the device and the host entry points give bit-identical G.
GramPlan gram_plan(long long N, int p, int dtype, int num_sms, bool tensor_core) {
  GramPlan g{};
  g.tensor_core = tensor_core;
  const int tile = tensor_core ? 128 : kGT;
  const int ts = (p + tile - 1) / tile;
  const long long tiles = (long long)ts * (ts + 1) / 2;
  long long per_chunk = (2LL * num_sms + tiles - 1) / tiles;            // slots launched together
  if (tensor_core) per_chunk = tiles <= num_sms ? num_sms / tiles : 1;   // one CTA per SM (TMEM, 128 registers x 512): one wave
  if (per_chunk > 64) per_chunk = 64;
  const double x_bytes = (double)N * p * (dtype == kF32 ? 4.0 : 8.0);
  long long chunks = (long long)(x_bytes / (128.0 * 1024 * 1024));
  chunks = chunks < 1 ? 1 : chunks > 16 ? 16 : chunks;
  long long slots = per_chunk * chunks;
  const long long max_by_rows = (N + 4095) / 4096;
  if (slots > max_by_rows) { slots = max_by_rows < 1 ? 1 : max_by_rows; chunks = 1; per_chunk = slots; }
  g.slots = (int)slots; g.chunks = (int)chunks; g.slots_per_chunk = (int)per_chunk;
  g.rows_per_slot = ((N + slots - 1) / slots + kGK - 1) / kGK * kGK;
  return g;
}

// Gram of the row chunk c (its slots_per_chunk slots) into scratch.
cudaError_t gram_chunk_launch(const GramPlan& g, int chunk, const void* X, int dtype, long long N, int p, double* scratch,
                              cudaStream_t st) {
  const int ts = (p + kGT - 1) / kGT;
  const int tiles = ts * (ts + 1) / 2;
  dim3 grid(tiles, g.slots_per_chunk);
  const int slot0 = chunk * g.slots_per_chunk;
  if (dtype == kF32)
    gram_kernel<float><<<grid, 256, 0, st>>>(static_cast<const float*>(X), N, p, scratch, slot0, g.rows_per_slot);
  else
    gram_kernel<double><<<grid, 256, 0, st>>>(static_cast<const double*>(X), N, p, scratch, slot0, g.rows_per_slot);
  return cudaGetLastError();
}

// G = sum of the slots in slot order, mirrored to the upper triangle.
cudaError_t gram_finish_launch(const GramPlan& g, int p, const double* scratch, double* G, cudaStream_t st) {
  const size_t n = (size_t)p * p;
  gram_reduce_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(scratch, g.slots, p, G);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return e;
  gram_mirror_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(G, p);
  return cudaGetLastError();
}

}  // namespace hsp
