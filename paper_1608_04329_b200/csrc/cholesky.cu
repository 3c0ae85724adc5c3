// cholesky.cu -- rows c, d1, d2 of the hot-path table:
//   c   Q = G + diag(tau^-2 lam_j^-2)
//   d1  Q = L L^T, tiled fp64 Cholesky
//   d2  beta = Q^-1 g + L^-T e,  e_j = Phi^-1(u_j)           PAPER.md:180, 198-202, 239 (reading R5)
//
// One persistent kernel (`chol_dataflow_kernel`) does c and d1 and, in the same task graph, the inverse
// factor W = L^-1 (and its transpose Wt = L^-T): d2 then needs no substitution on the critical path
// after X^T z arrives -- it is two triangular matrix-vector products, t = W g + e and beta = Wt t,
// i.e. L t = g + L e and L^T beta = t, exactly the two solves of PAPER.md:199-201.
//
// Task graph on 64x64 tiles (nt = ceil(p/64) tile rows; matrices padded to P = 64 nt with the identity):
//   L(i,j), i >= j :  A = Q_ij - sum_{k<j} L_ik L_jk^T ;  i == j: L_jj = chol(A), W_jj = L_jj^-1 ;
//                                                         i >  j: L_ij = A W_jj^T
//   B(i,j), i <  j :  A = - sum_{k=i}^{j-1} L_jk Wt_ik^T ; W_ji = W_jj A  (stored in W and, transposed, in Wt)
// Tasks are numbered column by column and dealt round-robin to the CTAs; every task depends only on
// lower-numbered tasks, each CTA runs its tasks in order, and all CTAs are co-resident (cooperative
// launch), so spinning on the per-tile "done" flags cannot deadlock.  Every tile is computed by one
// CTA with a fixed summation order: the result does not depend on the number of CTAs.
//
// Storage: row-major, leading dimension P; L lower, W lower, Wt upper.
#include <cuda_runtime.h>
#include <cstdint>
#include <cstdlib>
#include "hsp_device.cuh"
#include "hsp_internal.h"

namespace hsp {

constexpr int CT = 64;                 // tile edge
constexpr int KC = 16;                 // k-columns per pipeline chunk
constexpr int CLD = KC + 2;            // chunk row stride in doubles (144 B): conflict-free LDS.128
constexpr int TLD = CT + 2;            // full-tile row stride in shared memory (528 B)
constexpr int NST = 4;                 // cp.async pipeline stages
constexpr int kCholThreads = 256;
constexpr int kStageDoubles = 2 * CT * CLD;                       // A chunk + B chunk
constexpr size_t kCholSmem = (size_t)NST * kStageDoubles * sizeof(double) + 1024;   // 73728 + scratch
static_assert((size_t)NST * kStageDoubles >= 2 * (size_t)CT * TLD, "finalize tiles must fit in the pipeline pool");

int chol_tiles(int p) { return (p + CT - 1) / CT; }
int chol_ld(int p) { return chol_tiles(p) * CT; }
size_t chol_flag_count(int p) { const size_t nt = chol_tiles(p); return 2 * nt * nt; }

__device__ __forceinline__ void cp_async16(void* dst_smem, const void* src) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"((uint32_t)__cvta_generic_to_shared(dst_smem)), "l"(src)
               : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

__device__ __forceinline__ int ld_acquire(const int* p) {
  int v;
  asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ void st_release(int* p, int v) {
  asm volatile("st.release.gpu.global.s32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}
__device__ __forceinline__ void wait_flag(const int* f) {
  while (ld_acquire(f) == 0) __nanosleep(32);
}

// acc[a][b] (rows ty+16a, cols tx+16b) += sgn * sum_k A[row][k] B[col][k],  k in [0, K), K even.
template <int LDA, int LDB, int K, bool NEG>
__device__ __forceinline__ void tile_mac(const double* __restrict__ A, const double* __restrict__ B, int ty, int tx,
                                         double (&acc)[4][4]) {
#pragma unroll
  for (int kk = 0; kk < K; kk += 2) {
    double2 av[4], bv[4];
#pragma unroll
    for (int a = 0; a < 4; ++a) av[a] = *reinterpret_cast<const double2*>(A + (ty + 16 * a) * LDA + kk);
#pragma unroll
    for (int b = 0; b < 4; ++b) bv[b] = *reinterpret_cast<const double2*>(B + (tx + 16 * b) * LDB + kk);
#pragma unroll
    for (int a = 0; a < 4; ++a)
#pragma unroll
      for (int b = 0; b < 4; ++b) {
        if (NEG) {
          acc[a][b] = fma(-av[a].x, bv[b].x, acc[a][b]);
          acc[a][b] = fma(-av[a].y, bv[b].y, acc[a][b]);
        } else {
          acc[a][b] = fma(av[a].x, bv[b].x, acc[a][b]);
          acc[a][b] = fma(av[a].y, bv[b].y, acc[a][b]);
        }
      }
  }
}

// In-place Cholesky of the 64x64 tile S (stride TLD, lower triangle used), all 256 threads.  On return
// S holds L (lower, diagonal included; the strict upper triangle is zeroed).  One barrier per pivot:
// the trailing update uses the unscaled column, S[r][c] -= S[r][j] S[c][j] / d_j, and the columns are
// scaled by 1/sqrt(d_j) at the end.  Returns false if a pivot is not positive (then d_j := 1).
__device__ __forceinline__ bool tile_potrf(double* __restrict__ S, double* __restrict__ dsq, int tid, int ty, int tx) {
  bool ok = true;
  for (int j = 0; j < CT; ++j) {
    __syncthreads();
    double d = S[j * TLD + j];
    if (!(d > 0.0)) { ok = false; d = 1.0; }
    const double inv = 1.0 / d;
#pragma unroll
    for (int a = 0; a < 4; ++a) {
      const int r = ty + 16 * a;
      if (r > j) {
        const double lr = S[r * TLD + j] * inv;
#pragma unroll
        for (int b = 0; b < 4; ++b) {
          const int c = tx + 16 * b;
          if (c > j && c <= r) S[r * TLD + c] = fma(-lr, S[c * TLD + j], S[r * TLD + c]);
        }
      }
    }
  }
  __syncthreads();
  if (tid < CT) {
    double d = S[tid * TLD + tid];
    if (!(d > 0.0)) d = 1.0;
    dsq[tid] = 1.0 / sqrt(d);
  }
  __syncthreads();
  double v[4][4];
#pragma unroll
  for (int a = 0; a < 4; ++a)
#pragma unroll
    for (int b = 0; b < 4; ++b) {
      const int r = ty + 16 * a, c = tx + 16 * b;
      double x = 0.0;
      if (r > c) x = S[r * TLD + c] * dsq[c];
      else if (r == c) { double d = S[r * TLD + r]; if (!(d > 0.0)) d = 1.0; x = d * dsq[r]; }
      v[a][b] = x;
    }
  __syncthreads();
#pragma unroll
  for (int a = 0; a < 4; ++a)
#pragma unroll
    for (int b = 0; b < 4; ++b) S[(ty + 16 * a) * TLD + tx + 16 * b] = v[a][b];
  __syncthreads();
  return ok;
}

// X = S^-1 for the lower-triangular 64x64 tile S (stride TLD); X (stride TLD) gets the full tile
// (zeros above the diagonal).  16x16 diagonal blocks by substitution (one thread per column, registers),
// then two merge levels  [A 0; B C]^-1 = [A^-1 0; -C^-1 B A^-1  C^-1].
__device__ __forceinline__ void tile_trinv(const double* __restrict__ S, const double* __restrict__ dsq,
                                           double* __restrict__ X, int tid) {
  for (int e = tid; e < CT * TLD; e += kCholThreads) X[e] = 0.0;
  __syncthreads();
  if (tid < CT) {
    const int b0 = (tid >> 4) * 16, c = tid & 15;
    double x[16];
#pragma unroll
    for (int r = 0; r < 16; ++r) {
      double s = (r == c) ? 1.0 : 0.0;
#pragma unroll
      for (int m = 0; m < r; ++m) s = fma(-S[(b0 + r) * TLD + b0 + m], x[m], s);
      x[r] = (r >= c) ? s * dsq[b0 + r] : 0.0;          // 1 / L_rr = 1 / sqrt(d_r)
    }
#pragma unroll
    for (int r = 0; r < 16; ++r) X[(b0 + r) * TLD + b0 + c] = x[r];
  }
  __syncthreads();
  for (int h = 16; h < CT; h <<= 1) {
    const int nblk = CT / (2 * h);
    // T = B A^-1 into the (zero) upper-right block of X
    for (int e = tid; e < nblk * h * h; e += kCholThreads) {
      const int blk = e / (h * h), r = (e / h) % h, c = e % h, off = blk * 2 * h;
      double s = 0.0;
      for (int m = c; m < h; ++m) s = fma(S[(off + h + r) * TLD + off + m], X[(off + m) * TLD + off + c], s);
      X[(off + r) * TLD + off + h + c] = s;
    }
    __syncthreads();
    // lower-left block = -C^-1 T
    for (int e = tid; e < nblk * h * h; e += kCholThreads) {
      const int blk = e / (h * h), r = (e / h) % h, c = e % h, off = blk * 2 * h;
      double s = 0.0;
      for (int m = 0; m <= r; ++m) s = fma(X[(off + h + r) * TLD + off + h + m], X[(off + m) * TLD + off + h + c], s);
      X[(off + h + r) * TLD + off + c] = -s;
    }
    __syncthreads();
    for (int e = tid; e < nblk * h * h; e += kCholThreads) {
      const int blk = e / (h * h), r = (e / h) % h, c = e % h, off = blk * 2 * h;
      X[(off + r) * TLD + off + h + c] = 0.0;
    }
    __syncthreads();
  }
}

__global__ void __launch_bounds__(kCholThreads, 1)
chol_dataflow_kernel(const double* __restrict__ G, const double* __restrict__ lam_inv2, Ctl* __restrict__ ctl,
                     double* __restrict__ L, double* __restrict__ W, double* __restrict__ Wt, int* __restrict__ flags,
                     int p, int nt) {
  extern __shared__ __align__(16) double pool[];
  double* dsq = pool + (size_t)NST * kStageDoubles;          // 64 doubles of scratch after the pool
  const int P = nt * CT;
  const int tid = threadIdx.x, ty = tid >> 4, tx = tid & 15;
  int* fL = flags;
  int* fB = flags + (size_t)nt * nt;
  const double tau_inv2 = ctl->tau_inv2;
  const long long ntasks = (long long)nt * nt;

  for (long long t = blockIdx.x; t < ntasks; t += gridDim.x) {
    const int j = (int)(t / nt), rr = (int)(t % nt);
    const bool isL = rr < nt - j;
    const int i = isL ? j + rr : rr - (nt - j);
    // operands of the k loop: acc -= MA(ra,k) MB(rb,k)^T, k in [kbeg, kend)
    const double* MA = L;
    const double* MB = isL ? L : Wt;
    const int ra = isL ? i : j, rb = isL ? j : i;
    const int kbeg = isL ? 0 : i, kend = j;

    double acc[4][4];
#pragma unroll
    for (int a = 0; a < 4; ++a)
#pragma unroll
      for (int b = 0; b < 4; ++b) {
        double v = 0.0;
        if (isL) {                                   // c: Q tile, padded with the identity
          const int gr = i * CT + ty + 16 * a, gc = j * CT + tx + 16 * b;
          if (gr < p && gc < p) {
            v = G[(size_t)gr * p + gc];
            if (gr == gc) v = fma(tau_inv2, lam_inv2[gr], v);
          } else if (gr == gc) v = 1.0;
        }
        acc[a][b] = v;
      }

    const int nchunks = (kend - kbeg) * (CT / KC);
    auto issue = [&](int c) {
      const int k = kbeg + c / (CT / KC), kc = c % (CT / KC);
      if (kc == 0) {                                 // first chunk of a k tile: its producers must be done
        wait_flag(&fL[(size_t)ra * nt + k]);
        if (isL) { if (rb != ra) wait_flag(&fL[(size_t)rb * nt + k]); }
        else wait_flag(k == rb ? &fL[(size_t)rb * nt + rb] : &fB[(size_t)rb * nt + k]);
      }
      double* sa = pool + (size_t)(c % NST) * kStageDoubles;
      double* sb = sa + CT * CLD;
      const double* ga = MA + (size_t)ra * CT * P + (size_t)k * CT + kc * KC;
      const double* gb = MB + (size_t)rb * CT * P + (size_t)k * CT + kc * KC;
#pragma unroll
      for (int q = tid; q < CT * (KC / 2); q += kCholThreads) {
        const int row = q / (KC / 2), pc = q % (KC / 2);
        cp_async16(sa + row * CLD + pc * 2, ga + (size_t)row * P + pc * 2);
        cp_async16(sb + row * CLD + pc * 2, gb + (size_t)row * P + pc * 2);
      }
    };
    __syncthreads();                                 // the pool is free (previous task's finalize is over)
    for (int c = 0; c < NST - 1; ++c) {
      if (c < nchunks) issue(c);
      cp_async_commit();
    }
    for (int c = 0; c < nchunks; ++c) {
      cp_async_wait<NST - 2>();
      __syncthreads();
      if (c + NST - 1 < nchunks) issue(c + NST - 1);
      cp_async_commit();
      const double* sa = pool + (size_t)(c % NST) * kStageDoubles;
      tile_mac<CLD, CLD, KC, true>(sa, sa + CT * CLD, ty, tx, acc);
    }
    cp_async_wait<0>();
    __syncthreads();

    double* S = pool;                                // 64 x TLD
    double* X = pool + CT * TLD;                     // 64 x TLD
    if (isL && i == j) {
      // ---- diagonal: L_jj = chol(acc), W_jj = L_jj^-1
#pragma unroll
      for (int a = 0; a < 4; ++a)
#pragma unroll
        for (int b = 0; b < 4; ++b) S[(ty + 16 * a) * TLD + tx + 16 * b] = acc[a][b];
      const bool ok = tile_potrf(S, dsq, tid, ty, tx);
      if (!ok && tid == 0) atomicCAS(&ctl->status, 0, -4);
      tile_trinv(S, dsq, X, tid);
      for (int e = tid; e < CT * CT; e += kCholThreads) {
        const int r = e / CT, c = e % CT;
        const size_t g = (size_t)(j * CT + r) * P + j * CT + c;
        L[g] = S[r * TLD + c];
        W[g] = X[r * TLD + c];
        Wt[g] = X[c * TLD + r];
      }
      __threadfence();
      __syncthreads();
      if (tid == 0) st_release(&fL[(size_t)j * nt + j], 1);
    } else {
      // ---- off-diagonal: multiply by W_jj (from global; written by the diagonal task of column j)
      wait_flag(&fL[(size_t)j * nt + j]);
      const double* wjj = W + (size_t)j * CT * P + (size_t)j * CT;
      for (int q = tid; q < CT * (CT / 2); q += kCholThreads) {
        const int row = q / (CT / 2), pc = q % (CT / 2);
        cp_async16(X + row * TLD + pc * 2, wjj + (size_t)row * P + pc * 2);
      }
      cp_async_commit();
      double out[4][4];
#pragma unroll
      for (int a = 0; a < 4; ++a)
#pragma unroll
        for (int b = 0; b < 4; ++b) out[a][b] = 0.0;
      if (isL) {
#pragma unroll
        for (int a = 0; a < 4; ++a)
#pragma unroll
          for (int b = 0; b < 4; ++b) S[(ty + 16 * a) * TLD + tx + 16 * b] = acc[a][b];
        cp_async_wait<0>();
        __syncthreads();
        tile_mac<TLD, TLD, CT, false>(S, X, ty, tx, out);          // L_ij = A W_jj^T
#pragma unroll
        for (int a = 0; a < 4; ++a)
#pragma unroll
          for (int b = 0; b < 4; ++b) L[(size_t)(i * CT + ty + 16 * a) * P + j * CT + tx + 16 * b] = out[a][b];
        __threadfence();
        __syncthreads();
        if (tid == 0) st_release(&fL[(size_t)i * nt + j], 1);
      } else {
#pragma unroll
        for (int a = 0; a < 4; ++a)
#pragma unroll
          for (int b = 0; b < 4; ++b) S[(tx + 16 * b) * TLD + ty + 16 * a] = acc[a][b];   // transposed
        cp_async_wait<0>();
        __syncthreads();
        tile_mac<TLD, TLD, CT, false>(X, S, ty, tx, out);          // W_ji = W_jj A
#pragma unroll
        for (int a = 0; a < 4; ++a)
#pragma unroll
          for (int b = 0; b < 4; ++b) {
            const int r = j * CT + ty + 16 * a, c = i * CT + tx + 16 * b;
            W[(size_t)r * P + c] = out[a][b];
            Wt[(size_t)c * P + r] = out[a][b];
          }
        __threadfence();
        __syncthreads();
        if (tid == 0) st_release(&fB[(size_t)i * nt + j], 1);
      }
    }
  }
}

// d2, first half: t = W g + e (L t = g + L e), one warp per row; e_j = Phi^-1(U_A(j, k, E)).
constexpr int kGemvWarps = 8;
__global__ void __launch_bounds__(kGemvWarps * 32)
beta_gemv1_kernel(const double* __restrict__ W, const double* __restrict__ g, double* __restrict__ tv, int p, int P,
                  unsigned long long seed, const Ctl* __restrict__ ctl) {
  const int row = blockIdx.x * kGemvWarps + (threadIdx.x >> 5), lane = threadIdx.x & 31;
  if (row >= p) return;
  const double* w = W + (size_t)row * P;
  const int end = (row / CT + 1) * CT;               // W is zero right of the diagonal inside its tile
  double s0 = 0.0, s1 = 0.0;
  for (int c = 2 * lane; c < end; c += 64) {
    const double2 a = *reinterpret_cast<const double2*>(w + c);
    const double2 b = *reinterpret_cast<const double2*>(g + c);
    s0 = fma(a.x, b.x, s0);
    s1 = fma(a.y, b.y, s1);
  }
  double s = s0 + s1;
#pragma unroll
  for (int off = 16; off >= 1; off >>= 1) s += __shfl_xor_sync(0xffffffffu, s, off);
  if (lane == 0) {
    const uint32_t sweep = (uint32_t)(ctl->sweep + 1ull);
    tv[row] = s + norm_inv(uniform_a(seed, (unsigned long long)row, sweep, TAG_E));
  }
}

// d2, second half: beta = Wt t (L^T beta = t), one warp per row.
__global__ void __launch_bounds__(kGemvWarps * 32)
beta_gemv2_kernel(const double* __restrict__ Wt, const double* __restrict__ tv, double* __restrict__ beta, int p, int P,
                  Ctl* __restrict__ ctl) {
  const int row = blockIdx.x * kGemvWarps + (threadIdx.x >> 5), lane = threadIdx.x & 31;
  if (row >= p) return;
  const double* w = Wt + (size_t)row * P;
  const int begin = (row / CT) * CT;                 // Wt is zero left of the diagonal inside its tile
  double s0 = 0.0, s1 = 0.0;
  for (int c = begin + 2 * lane; c < P; c += 64) {
    const double2 a = *reinterpret_cast<const double2*>(w + c);
    const double2 b = *reinterpret_cast<const double2*>(tv + c);
    s0 = fma(a.x, b.x, s0);
    s1 = fma(a.y, b.y, s1);
  }
  double s = s0 + s1;
#pragma unroll
  for (int off = 16; off >= 1; off >>= 1) s += __shfl_xor_sync(0xffffffffu, s, off);
  if (lane == 0) {
    beta[row] = s;
    if (!isfinite(s)) atomicCAS(&ctl->status, 0, -5);
  }
}

static int env_int2(const char* name, int dflt) {
  const char* v = getenv(name);
  return (v && *v) ? atoi(v) : dflt;
}

// Number of CTAs for the Cholesky branch.  When the branch is expected to hide behind the fused pass
// it gets `k` SMs of its own and the fused pass the other num_sms - k; otherwise every SM.
int chol_plan_ctas(int p, int num_sms, double fused_ms_estimate, bool* overlap) {
  const int nt = chol_tiles(p);
  const double flops = 2.0 * (double)p * p * p / 3.0;             // Cholesky + inverse factor
  const double per_sm = 0.5 * 2.0 * 64.0 * 1.9e9;                 // ~50 % of 64 DFMA/clk/SM
  int k = env_int2("HSP_CHOL_CTAS", 0);
  bool ov;
  if (k > 0) {
    ov = k < num_sms;
  } else {
    // measured on B200 (profiles/r01_b): the left-looking task chain costs ~35 us per tile column, and the
    // kernel takes ~2.6x the time the flop count at 50 % of the DFMA rate suggests
    const double critical_ms = nt * 0.035;
    k = 8;
    while (k < 48 && 2.6 * (flops / (k * per_sm)) * 1e3 > 0.85 * fused_ms_estimate) k += 4;
    const double t = 2.6 * (flops / (k * per_sm)) * 1e3;
    ov = t <= 0.9 * fused_ms_estimate && critical_ms <= 0.9 * fused_ms_estimate;
    if (!ov) k = num_sms;
  }
  const long long ntasks = (long long)nt * nt;
  if (k > ntasks) k = (int)ntasks;
  if (k > num_sms) k = num_sms;
  if (overlap) *overlap = ov;
  return k;
}

cudaError_t chol_prepare() {
  return cudaFuncSetAttribute(chol_dataflow_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kCholSmem);
}

cudaError_t cholesky_launch(const double* G, const double* lam_inv2, Ctl* ctl, double* L, double* W, double* Wt,
                            int* flags, int p, int ctas, cudaStream_t st, long long* launches) {
  int nt = chol_tiles(p);
  cudaError_t e = cudaMemsetAsync(flags, 0, chol_flag_count(p) * sizeof(int), st);
  if (e != cudaSuccess) return e;
  void* args[] = {(void*)&G, (void*)&lam_inv2, (void*)&ctl, (void*)&L, (void*)&W, (void*)&Wt, (void*)&flags, (void*)&p,
                  (void*)&nt};
  e = cudaLaunchCooperativeKernel((const void*)chol_dataflow_kernel, dim3(ctas), dim3(kCholThreads), args, kCholSmem, st);
  if (launches) ++*launches;
  return e;
}

cudaError_t beta_solve_launch(const double* W, const double* Wt, const double* g, double* tv, double* beta, int p,
                              unsigned long long seed, Ctl* ctl, cudaStream_t st, long long* launches) {
  const int P = chol_ld(p);
  const int grid = (p + kGemvWarps - 1) / kGemvWarps;
  beta_gemv1_kernel<<<grid, kGemvWarps * 32, 0, st>>>(W, g, tv, p, P, seed, ctl);
  beta_gemv2_kernel<<<grid, kGemvWarps * 32, 0, st>>>(Wt, tv, beta, p, P, ctl);
  if (launches) *launches += 2;
  return cudaGetLastError();
}

}  // namespace hsp
