// cholesky.cu -- rows c, d1, d2 of the hot-path table:
//   c   Q = G + diag(tau^-2 lam_j^-2)
//   d1  Q = L L^T, blocked right-looking fp64 Cholesky
//   d2  beta = Q^-1 g + L^-T e  via  L v = g,  L^T beta = v + e,  e_j = Phi^-1(u_j)
//                                                            PAPER.md:180, 198-202, 239 (reading R5)
// Storage: row-major p x p, lower triangle.
#include <cuda_runtime.h>
#include <cstdint>
#include "hsp_device.cuh"
#include "hsp_internal.h"

namespace hsp {

constexpr int NB = 32;   // panel width

__global__ void build_q_kernel(const double* __restrict__ G, const double* __restrict__ lam_inv2,
                               const Ctl* __restrict__ ctl, double* __restrict__ L, int p) {
  const size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= (size_t)p * p) return;
  const int i = (int)(idx / p), j = (int)(idx % p);
  if (j > i) return;
  double v = G[idx];
  if (i == j) v += ctl->tau_inv2 * lam_inv2[j];
  L[idx] = v;
}

// Panel step at column k0: every CTA factors the NB x NB diagonal block (warp 0, rows in
// registers, shuffles) redundantly, CTA 0 writes it back, and each CTA then solves its 128 rows of
// the block column below:  L21 = A21 L11^-T  (thread per row, forward substitution).
constexpr int kPanelRows = 128;
__global__ void __launch_bounds__(kPanelRows)
chol_panel_kernel(double* __restrict__ A, int p, int k0, Ctl* __restrict__ ctl) {
  __shared__ double D[NB][NB + 1];
  __shared__ double invd[NB];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int nb = (p - k0) < NB ? (p - k0) : NB;
  if (warp == 0) {
    double a[NB];
    const int i = lane;
#pragma unroll
    for (int j = 0; j < NB; ++j) {
      double v = (i == j) ? 1.0 : 0.0;                       // identity padding past nb
      if (i < nb && j <= i) v = A[(size_t)(k0 + i) * p + k0 + j];
      a[j] = v;
    }
    bool bad = false;
#pragma unroll
    for (int j = 0; j < NB; ++j) {
      double d = __shfl_sync(0xffffffffu, a[j], j);
      if (!(d > 0.0)) { bad = true; d = 1.0; }
      const double inv = rsqrt(d);
      const double l = d * inv;
      a[j] = (i == j) ? l : a[j] * inv;
#pragma unroll
      for (int k = j + 1; k < NB; ++k) {
        const double lkj = __shfl_sync(0xffffffffu, a[j], k);
        a[k] = fma(-a[j], lkj, a[k]);
      }
      if (i == j) invd[j] = 1.0 / l;
    }
    if (bad && lane == 0 && blockIdx.x == 0) atomicCAS(&ctl->status, 0, -4);
#pragma unroll
    for (int j = 0; j < NB; ++j) {
      D[i][j] = (j <= i) ? a[j] : 0.0;
      if (blockIdx.x == 0 && i < nb && j <= i) A[(size_t)(k0 + i) * p + k0 + j] = a[j];
    }
  }
  __syncthreads();
  const int r = k0 + nb + blockIdx.x * kPanelRows + tid;
  if (r < p) {
    double a[NB];
    double* row = A + (size_t)r * p + k0;
#pragma unroll
    for (int j = 0; j < NB; ++j) a[j] = (j < nb) ? row[j] : 0.0;
#pragma unroll
    for (int j = 0; j < NB; ++j) {
      double s = a[j];
#pragma unroll
      for (int k = 0; k < j; ++k) s = fma(-a[k], D[j][k], s);
      a[j] = s * invd[j];
    }
#pragma unroll
    for (int j = 0; j < NB; ++j)
      if (j < nb) row[j] = a[j];
  }
}

// Trailing update after panel k0:  A22 -= L21 L21^T on lower 64x64 tiles (K = NB).
constexpr int kUT = 64;
__global__ void __launch_bounds__(256)
chol_update_kernel(double* __restrict__ A, int p, int k0) {
  __shared__ double As[NB][kUT + 4];
  __shared__ double Bs[NB][kUT + 4];
  int t = blockIdx.x, ti = 0;
  while (t >= ti + 1) { t -= ti + 1; ++ti; }
  const int tj = t;
  const int base = k0 + NB;
  const int tid = threadIdx.x, tx = tid & 15, ty = tid >> 4;
  // load L21 rows of tile ti and tj: 64 rows x NB columns each, transposed into [k][row]
  for (int e = tid; e < kUT * NB; e += 256) {
    const int rr = e / NB, kk = e % NB;
    const int ra = base + ti * kUT + rr, rb = base + tj * kUT + rr;
    As[kk][rr] = (ra < p) ? A[(size_t)ra * p + k0 + kk] : 0.0;
    Bs[kk][rr] = (rb < p) ? A[(size_t)rb * p + k0 + kk] : 0.0;
  }
  __syncthreads();
  double acc[4][4];
#pragma unroll
  for (int i = 0; i < 4; ++i)
#pragma unroll
    for (int j = 0; j < 4; ++j) acc[i][j] = 0.0;
#pragma unroll
  for (int kk = 0; kk < NB; ++kk) {
    double a[4], b[4];
#pragma unroll
    for (int i = 0; i < 4; ++i) { a[i] = As[kk][ty * 4 + i]; b[i] = Bs[kk][tx * 4 + i]; }
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
      for (int j = 0; j < 4; ++j) acc[i][j] = fma(a[i], b[j], acc[i][j]);
  }
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const int r = base + ti * kUT + ty * 4 + i;
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      const int c = base + tj * kUT + tx * 4 + j;
      if (r < p && c <= r) A[(size_t)r * p + c] -= acc[i][j];
    }
  }
}

cudaError_t build_q_launch(const double* G, const double* lam_inv2, const Ctl* ctl, double* L, int p, cudaStream_t st) {
  const size_t n = (size_t)p * p;
  build_q_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(G, lam_inv2, ctl, L, p);
  return cudaGetLastError();
}

cudaError_t cholesky_launch(double* L, int p, Ctl* ctl, cudaStream_t st, long long* launches) {
  for (int k0 = 0; k0 < p; k0 += NB) {
    const int below = p - k0 - NB;
    const int grid = below > 0 ? (below + kPanelRows - 1) / kPanelRows : 1;
    chol_panel_kernel<<<grid, kPanelRows, 0, st>>>(L, p, k0, ctl);
    if (launches) ++*launches;
    if (below > 0) {
      const int ts = (below + kUT - 1) / kUT;
      chol_update_kernel<<<ts * (ts + 1) / 2, 256, 0, st>>>(L, p, k0);
      if (launches) ++*launches;
    }
  }
  return cudaGetLastError();
}

// d2: single-CTA blocked substitutions.  v = L^-1 g; beta = L^-T (v + e).
constexpr int kSolveThreads = 512;
__global__ void __launch_bounds__(kSolveThreads)
beta_draw_kernel(const double* __restrict__ L, const double* __restrict__ g, double* __restrict__ beta, int p,
                 unsigned long long seed, Ctl* __restrict__ ctl) {
  extern __shared__ double v[];               // p doubles
  __shared__ double xb[NB];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const uint32_t sweep = (uint32_t)(ctl->sweep + 1ull);
  for (int j = tid; j < p; j += kSolveThreads) v[j] = g[j];
  __syncthreads();
  // forward: L v = g
  for (int k0 = 0; k0 < p; k0 += NB) {
    const int nb = (p - k0) < NB ? (p - k0) : NB;
    if (warp == 0) {
      const int i = lane;
      double a[NB];
#pragma unroll
      for (int j = 0; j < NB; ++j) a[j] = (i < nb && j < i) ? L[(size_t)(k0 + i) * p + k0 + j] : 0.0;
      const double dinv = (i < nb) ? 1.0 / L[(size_t)(k0 + i) * p + k0 + i] : 1.0;
      double r = (i < nb) ? v[k0 + i] : 0.0;
#pragma unroll
      for (int j = 0; j < NB; ++j) {
        const double xj = __shfl_sync(0xffffffffu, r * dinv, j);
        if (i == j) r = xj; else if (i > j) r = fma(-a[j], xj, r);
      }
      if (i < nb) { v[k0 + i] = r; }
      xb[i] = (i < nb) ? r : 0.0;
    }
    __syncthreads();
    for (int r = k0 + nb + tid; r < p; r += kSolveThreads) {
      const double* row = L + (size_t)r * p + k0;
      double s = v[r];
#pragma unroll 8
      for (int j = 0; j < nb; ++j) s = fma(-row[j], xb[j], s);
      v[r] = s;
    }
    __syncthreads();
  }
  // add e ~ N(0, I): one Philox call per coordinate
  for (int j = tid; j < p; j += kSolveThreads) v[j] += norm_inv(uniform_a(seed, (unsigned long long)j, sweep, TAG_E));
  __syncthreads();
  // backward: L^T beta = v
  const int nblk = (p + NB - 1) / NB;
  for (int b = nblk - 1; b >= 0; --b) {
    const int k0 = b * NB;
    const int nb = (p - k0) < NB ? (p - k0) : NB;
    if (warp == 0) {
      const int i = lane;                     // unknown k0 + i; needs column i of the diagonal block
      double a[NB];
#pragma unroll
      for (int j = 0; j < NB; ++j) a[j] = (j < nb && i < nb && j > i) ? L[(size_t)(k0 + j) * p + k0 + i] : 0.0;
      const double dinv = (i < nb) ? 1.0 / L[(size_t)(k0 + i) * p + k0 + i] : 1.0;
      double r = (i < nb) ? v[k0 + i] : 0.0;
#pragma unroll
      for (int j = NB - 1; j >= 0; --j) {
        const double xj = __shfl_sync(0xffffffffu, r * dinv, j);
        if (i == j) r = xj; else if (i < j) r = fma(-a[j], xj, r);
      }
      if (i < nb) v[k0 + i] = r;
      xb[i] = (i < nb) ? r : 0.0;
    }
    __syncthreads();
    for (int r = tid; r < k0; r += kSolveThreads) {
      double s = v[r];
#pragma unroll 8
      for (int j = 0; j < nb; ++j) s = fma(-L[(size_t)(k0 + j) * p + r], xb[j], s);
      v[r] = s;
    }
    __syncthreads();
  }
  bool bad = false;
  for (int j = tid; j < p; j += kSolveThreads) {
    const double b = v[j];
    beta[j] = b;
    if (!isfinite(b)) bad = true;
  }
  if (bad) atomicCAS(&ctl->status, 0, -5);
}

cudaError_t beta_draw_launch(const double* L, const double* g, double* beta, int p, unsigned long long seed,
                             Ctl* ctl, cudaStream_t st) {
  const size_t smem = (size_t)p * sizeof(double);
  static size_t configured = 0;
  if (smem > 48 * 1024 && smem > configured) {
    cudaError_t e = cudaFuncSetAttribute(beta_draw_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    configured = smem;
  }
  if (L == nullptr) return cudaSuccess;   // prepare-only call
  beta_draw_kernel<<<1, kSolveThreads, smem, st>>>(L, g, beta, p, seed, ctl);
  return cudaGetLastError();
}

}  // namespace hsp
