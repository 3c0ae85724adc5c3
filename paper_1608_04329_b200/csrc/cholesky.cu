// cholesky.cu -- rows c, d1, d2 of the hot-path table:
//   c   Q = G + diag(tau^-2 lam_j^-2)
//   d1  Q = L L^T, tiled fp64 Cholesky
//   d2  beta = Q^-1 g + L^-T e,  e_j = Phi^-1(u_j)           PAPER.md:180, 198-202, 239 (reading R5)
//
// One persistent cooperative kernel (`chol_task_kernel`) does c and d1 and, in the same task graph, the
// inverse factor W = L^-1 (and its transpose Wt = L^-T): d2 then needs no substitution on the critical path
// after X^T z arrives -- it is two triangular matrix-vector products, t = W g + e and beta = Wt t,
// i.e. L t = g + L e and L^T beta = t, exactly the two solves of PAPER.md:199-201.
//
// Task graph on 64x64 tiles (nt = ceil(p/64) tile rows; matrices padded to P = 64 nt with the identity):
//   L(i,j), i >= j :  A = Q_ij - sum_{k<j} L_ik L_jk^T ;  i == j: L_jj = chol(A), W_jj = L_jj^-1 ;
//                                                         i >  j: L_ij = A W_jj^T
//   B(i,j), i <  j :  A = - sum_{k=i}^{j-1} L_jk Wt_ik^T ; W_ji = W_jj A  (stored in W and, transposed, in Wt)
// The critical path of the factorisation is  potrf(j) -> L(j+1,j) = A W_jj^T -> A(j+1,j+1) -= L(j+1,j) L(j+1,j)^T ->
// potrf(j+1): with two or more CTAs it is run by ONE dedicated CTA (the first list) as three chain tasks per column
// whose operands stay in its shared memory (types 2, 3, 4 below) -- no flag round trips through global memory between
// them; all other CTAs feed it partial accumulators (prefix tasks) and take the bulk of the products.  With a single
// CTA the host (chol_schedule.cu) instead splits the tiles on the critical path into prefix + finish tasks.  All
// tasks are dealt to the CTAs as static ordered lists; a CTA runs its list in order and waits on per-tile "done" flags
// inside the k-loop.  All CTAs are co-resident (cooperative launch) and every list is a subsequence of one
// global order in which producers precede consumers, so the spin-waits cannot deadlock.  Every tile is
// accumulated in ascending k by a fixed sequence of tasks: the result does not depend on the number of CTAs.
//
// Tile products run on the FP64 tensor pipe (mma.sync m8n8k4 f64 -> SASS DMMA; tcgen05 has no f64 kind):
// 8 warps x (32 rows x 16 columns) of the 64x64 accumulator.  CTA = 8 compute warps + a PRODUCER warp + a PUBLISHER warp.
// The producer streams the operands of the k-loops in 32-column chunks as 2-D TMA boxes (cp.async.bulk.tensor, 16 columns
// x 64 rows with the 128-byte swizzle, which makes the fragment loads conflict-free without padding; 4-stage ring, full /
// empty mbarriers), does all the flag polling for the k-loops and runs ahead of the compute warps across tasks, so the
// next task's operands arrive during this task's epilogue.  In the chain CTA the producer fetches the parked accumulators
// and the publisher warp writes the chain's results to global memory and sets their flags.
//
// Storage: row-major, leading dimension P; L lower, W lower, Wt upper.
#include <cuda.h>
#include <cuda_runtime.h>
#include <cstdint>
#include <cstdlib>
#include <vector>
#include "hsp_device.cuh"
#include "hsp_internal.h"

namespace hsp {

constexpr int CT = 64;                 // tile edge
constexpr int KC = 32;                 // k-columns per pipeline chunk
constexpr int KB = 16;                 // k-columns per TMA box: 128 bytes, the span of the 128-byte swizzle
constexpr int kBoxBytes = CT * KB * 8; // one box: 64 tile rows x 16 k-columns of doubles = 8 KB (1024-byte aligned in shared memory)
constexpr int TLD = CT + 4;            // full-tile row stride in shared memory (544 B)
constexpr int NST = 4;                 // stages of the operand ring (bulk copies, full / empty mbarriers)
constexpr int kCholThreads = 256;      // COMPUTE threads: 8 warps (16 warps with 16 x 16 warp tiles measured no faster)
constexpr int kCholWarps = kCholThreads / 32;
constexpr int kCholBlock = kCholThreads + 64;   // + the producer warp + the publisher warp (chain CTA)
constexpr int kChainStages = 2;        // ring stages the chain CTA uses for its parked accumulators; the rest of the ring holds its third tile buffer
constexpr int kMB = CT * CT / (kCholWarps * 16) / 8;   // 8-row blocks of a warp's accumulator: (8 kMB rows) x 16 columns per warp
constexpr int kStageBytes = 2 * (KC / KB) * kBoxBytes;            // A chunk + B chunk: 32 KB
constexpr int kPoolDoubles = NST * kStageBytes / 8;
constexpr uint32_t kStageTxBytes = (uint32_t)kStageBytes;   // bytes a full stage receives (A chunk + B chunk)
// 1 KB of slack (the ring is aligned to 1024 bytes by hand) + ring + S + X + rdiag + mbarriers
constexpr size_t kCholSmem = 1024 + (size_t)(kPoolDoubles + 2 * CT * TLD + CT) * sizeof(double) + (2 * NST + 4) * sizeof(unsigned long long);

int chol_tiles(int p) { return (p + CT - 1) / CT; }
int chol_ld(int p) { return chol_tiles(p) * CT; }

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
__device__ __forceinline__ unsigned long long globaltimer_ns() {
  unsigned long long t;
  asm volatile("mov.u64 %0, %globaltimer;" : "=l"(t));
  return t;
}
// The 8 compute warps synchronise among themselves (named barrier 1); the producer warp never joins.
__device__ __forceinline__ void cta_sync() { asm volatile("bar.sync 1, %0;" ::"n"(kCholThreads) : "memory"); }
// Flag protocol (the pattern of a CTA-wide semaphore): the producer CTA finishes its global stores, __syncthreads(), and
// ONE thread publishes with st.release.gpu; the consumer polls with ld.acquire.gpu from ONE thread (or the lanes of the
// producer warp, for many flags at once) and then synchronises the CTA (barrier / mbarrier).  An acquire load costs an L1 invalidation (SASS CCTL.IVALL);
// polled by every warp before every k-tile it was 20 % of the kernel's stall samples at p = 4000.
__device__ __forceinline__ void wait_flag_cta(const int* f, int tid) {
  if (tid == 0)
    while (ld_acquire(f) == 0) __nanosleep(20);
  cta_sync();
}
__device__ __forceinline__ void cmbar_init(uint32_t bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void cmbar_arrive(uint32_t bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void cmbar_expect_tx(uint32_t bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void cmbar_wait(uint32_t bar, uint32_t parity) {
  asm volatile(
      "{\n\t"
      ".reg .pred P1;\n\t"
      "CWAIT_LOOP:\n\t"
      "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n\t"
      "@P1 bra CDONE;\n\t"
      "bra CWAIT_LOOP;\n\t"
      "CDONE:\n\t"
      "}" ::"r"(bar),
      "r"(parity)
      : "memory");
}
// One box of a row-major P x P matrix of doubles (tensor map: 16 columns x 64 rows, 128-byte swizzle) -> shared memory.
__device__ __forceinline__ void tma_box(uint32_t dst_smem, const CUtensorMap* tm, int col, int row, uint32_t bar) {
  asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];" ::"r"(dst_smem),
               "l"(reinterpret_cast<uint64_t>(tm)), "r"(col), "r"(row), "r"(bar)
               : "memory");
}
__device__ __forceinline__ void bulk_g2s(uint32_t dst_smem, const void* src, uint32_t bytes, uint32_t bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst_smem),
               "l"(src), "r"(bytes), "r"(bar)
               : "memory");
}
__device__ __forceinline__ double2 lds_f64x2(uint32_t a) {
  double2 v;
  asm volatile("ld.shared.v2.f64 {%0,%1}, [%2];" : "=d"(v.x), "=d"(v.y) : "r"(a));
  return v;
}
__device__ __forceinline__ double lds_f64(uint32_t a) {
  double v;
  asm volatile("ld.shared.f64 %0, [%1];" : "=d"(v) : "r"(a));
  return v;
}
__device__ __forceinline__ void cp_async16_s(uint32_t dst_smem, const void* src) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst_smem), "l"(src) : "memory");
}

// D(8x8) += A(8x4) B(4x8) on the FP64 tensor pipe.  Fragments (PTX ISA, m8n8k4 .f64): with g = lane / 4,
// t = lane % 4:  a = A[g][t],  b = B[t][g],  c0,c1 = C[g][2t], C[g][2t+1].
__device__ __forceinline__ void dmma(double (&c)[2], double a, double b) {
  asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};" : "+d"(c[0]), "+d"(c[1]) : "d"(a), "d"(b));
}

// Accumulator layout of one thread: warp w covers rows wm*32..+32 (wm = w & 1) and columns wn*16..+16
// (wn = w >> 1); acc[mb][nb][e] is element (wm*32 + mb*8 + g, wn*16 + nb*8 + 2t + e).
struct Frag {
  int row0, col0, g, t;
  __device__ __forceinline__ explicit Frag(int tid) {
    const int w = tid >> 5, lane = tid & 31;
    constexpr int WR = CT / (8 * kMB);   // warps along the rows
    row0 = (w % WR) * 8 * kMB; col0 = (w / WR) * 16; g = lane >> 2; t = lane & 3;
  }
};

// acc[m][n] += sgn * sum_k A[m][k] B[n][k],  k in [0, K): A and B are row-major [row][k] in shared memory.
// PERM: a DMMA multiplies the k-columns {2m, 2m+1, 8+2m, 9+2m} of each group of 16 (the grouping of the k-loops,
// tile_mma_s) instead of four consecutive ones -- used where a chain task replaces a k-loop step (SYRK), so that the
// rounding, and with it every bit of L, does not depend on the number of CTAs.
template <int LDA, int LDB, int K, bool NEG, bool PERM = false>
__device__ __forceinline__ void tile_mma(const double* __restrict__ A, const double* __restrict__ B, const Frag& f,
                                         double (&acc)[kMB][2][2]) {
  const int tk = PERM ? (f.t >> 1) * 8 + (f.t & 1) : f.t;
  const double* ap = A + (f.row0 + f.g) * LDA + tk;
  const double* bp = B + (f.col0 + f.g) * LDB + tk;
#pragma unroll
  for (int kk = 0; kk < K; kk += 4) {
    const int ko = PERM ? (kk / 16) * 16 + ((kk % 16) / 4) * 2 : kk;
    double a[kMB], b[2];
#pragma unroll
    for (int mb = 0; mb < kMB; ++mb) { a[mb] = ap[mb * 8 * LDA + ko]; if (NEG) a[mb] = -a[mb]; }
#pragma unroll
    for (int nb = 0; nb < 2; ++nb) b[nb] = bp[nb * 8 * LDB + ko];
#pragma unroll
    for (int mb = 0; mb < kMB; ++mb)
#pragma unroll
      for (int nb = 0; nb < 2; ++nb) dmma(acc[mb][nb], a[mb], b[nb]);
  }
}

// out[m][n] += sum_{k <= n} A[m][k] Wm[n][k] for a LOWER-TRIANGULAR Wm (the product A W_jj^T that finishes an off-diagonal
// tile): the 8-column block cb needs only k < 8 (cb + 1).  A warp takes the column blocks {wc, 7 - wc} (wc = warp / 2) of
// its 32 rows, i.e. 72 of the 128 k-steps of the full product whatever wc -- balanced.  acc[mb][nb] is the block
// (row0 / 8 + mb, nb == 0 ? wc : 7 - wc); the skipped terms are exact zeros.
struct TriFrag {
  int row0, g, t, cb[2];
  __device__ __forceinline__ explicit TriFrag(int tid) {
    const int w = tid >> 5, lane = tid & 31;
    row0 = (w & 1) * 32; g = lane >> 2; t = lane & 3; cb[0] = w >> 1; cb[1] = 7 - (w >> 1);
  }
  __device__ __forceinline__ int col(int nb) const { return cb[nb] * 8 + 2 * t; }   // first of the two columns of acc[.][nb]
};
template <int LDA, int LDB>
__device__ __forceinline__ void tile_mma_tri(const double* __restrict__ A, const double* __restrict__ Wm, const TriFrag& z,
                                             double (&acc)[kMB][2][2]) {
  static_assert(kMB == 4, "the triangular product assumes 32 x 16 warp tiles");
  const double* ap = A + (z.row0 + z.g) * LDA + z.t;
  const double* b0 = Wm + (z.cb[0] * 8 + z.g) * LDB + z.t;
  const double* b1 = Wm + (z.cb[1] * 8 + z.g) * LDB + z.t;
  const int lim0 = 8 * (z.cb[0] + 1), lim1 = 8 * (z.cb[1] + 1);      // lim0 <= 32 < lim1, warp-uniform
#pragma unroll
  for (int kk = 0; kk < CT; kk += 4) {
    if (kk < lim1) {
      double a[kMB];
#pragma unroll
      for (int mb = 0; mb < kMB; ++mb) a[mb] = ap[mb * 8 * LDA + kk];
      const double bb1 = b1[kk];
#pragma unroll
      for (int mb = 0; mb < kMB; ++mb) dmma(acc[mb][1], a[mb], bb1);
      if (kk < lim0) {
        const double bb0 = b0[kk];
#pragma unroll
        for (int mb = 0; mb < kMB; ++mb) dmma(acc[mb][0], a[mb], bb0);
      }
    }
  }
}

// The k-loop version: operands are TMA boxes in shared memory (32-bit shared-window addresses A, B: KC / 16 boxes each, a
// box = 64 rows x 128 bytes with the 128-byte swizzle: the 16-byte unit u of row r sits at unit u ^ (r & 7)).  A lane
// reads row (row0 + 8 mb + g), whose r & 7 = g whatever mb, so its swizzled offsets inside a box are per-lane constants.
// Which four k-columns a DMMA multiplies is free (the same choice for A and B): step m = 0..3 of a box takes
// k = {2m, 2m+1, 8+2m, 9+2m} for t = 0..3, i.e. unit ((t >> 1) * 4 + m) ^ g, half t & 1.  The 16 lanes of a half-warp
// (g = 0..3 or 4..7) then touch 16 different (unit, half) pairs = all 32 banks once: two wavefronts per LDS.64, the
// minimum.  (Consecutive k = 4m + t put rows g and g ^ 1 on the same unit: a 2-way conflict, measured as 2x the ideal
// wavefronts on every fragment load.)
struct SwzFrag {
  uint32_t a0, b0, sw[4];
  __device__ __forceinline__ explicit SwzFrag(const Frag& f) {
    a0 = (uint32_t)((f.row0 + f.g) * 128);
    b0 = (uint32_t)((f.col0 + f.g) * 128);
#pragma unroll
    for (int q = 0; q < 4; ++q) sw[q] = (uint32_t)(((((f.t >> 1) * 4 + q) ^ f.g) * 16) + (f.t & 1) * 8);
  }
};
template <bool NEG>
__device__ __forceinline__ void tile_mma_s(uint32_t A, uint32_t B, const SwzFrag& z, double (&acc)[kMB][2][2]) {
#pragma unroll
  for (int kk = 0; kk < KC; kk += 4) {
    const uint32_t o = (uint32_t)((kk / KB) * kBoxBytes) + z.sw[(kk % KB) / 4];
    double a[kMB], b[2];
#pragma unroll
    for (int mb = 0; mb < kMB; ++mb) { a[mb] = lds_f64(A + z.a0 + (uint32_t)(mb * 8 * 128) + o); if (NEG) a[mb] = -a[mb]; }
#pragma unroll
    for (int nb = 0; nb < 2; ++nb) b[nb] = lds_f64(B + z.b0 + (uint32_t)(nb * 8 * 128) + o);
#pragma unroll
    for (int mb = 0; mb < kMB; ++mb)
#pragma unroll
      for (int nb = 0; nb < 2; ++nb) dmma(acc[mb][nb], a[mb], b[nb]);
  }
}

// 1/d for a positive normal d: MUFU seed (rcp.approx.ftz.f64, relative error e ~ 2^-20) and one cubic
// correction r (1 + e + e^2), three dependent FMAs; the result is within ~1 ulp.
__device__ __forceinline__ double fast_rcp(double d) {
  double r;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(d));
  const double e = fma(-d, r, 1.0);
  const double t = fma(e, e, e);
  return fma(r, t, r);
}

// In-place Cholesky of the 64x64 tile S (stride TLD, lower triangle used), every thread of the CTA; on return the
// lower triangle of S holds L (diagonal included) and rdiag[r] = 1 / L_rr.  Blocked by 16 columns: the
// 16-column panel below and including the diagonal block is factored in registers, 32 rows per warp (lanes
// 0-15 hold the diagonal block -- redundantly in every warp --, lanes 16-31 sixteen panel rows).  A pivot
// step broadcasts the UNSCALED column by shuffles and updates with a_rj a_cj / d_j, so the dependent chain
// per pivot is shuffle -> reciprocal -> two FMAs and needs no block barrier; columns are scaled by
// 1/sqrt(d_j) after the 16 pivots.  The trailing rows are then updated on the FP64 tensor pipe.
// Returns false if a pivot is not positive (it is then replaced by 1).
__device__ __forceinline__ bool tile_potrf(double* __restrict__ S, double* __restrict__ rdiag, int tid) {
  const int warp = tid >> 5, lane = tid & 31;
  bool ok = true;
#pragma unroll 1
  for (int b = 0; b < CT / 16; ++b) {
    const int o = b * 16;
    const int npanel = CT - o - 16;                        // rows below the diagonal block
    const int nwarps = npanel > 0 ? npanel / 16 : 1;
    if (warp < nwarps) {
      const bool isdiag = lane < 16;
      const int row = isdiag ? o + lane : o + 16 * (warp + 1) + (lane - 16);
      const bool live = isdiag || npanel > 0;
      double a[16], myd = 1.0;
      const double* src = S + (live ? row : o) * TLD + o;
#pragma unroll
      for (int c = 0; c < 16; c += 2) {
        const double2 v = *reinterpret_cast<const double2*>(src + c);
        a[c] = v.x; a[c + 1] = v.y;
      }
#pragma unroll
      for (int j = 0; j < 16; ++j) {
        const double d = __shfl_sync(0xffffffffu, a[j], j);
        double ac[16];
#pragma unroll
        for (int c = j + 1; c < 16; ++c) ac[c] = __shfl_sync(0xffffffffu, a[j], c);
        // the positivity test stays off the dependent chain: a bad pivot poisons the tile, which is
        // reported as HSP_ENOTPD by the caller
        if (!(d > 0.0)) ok = false;
        if (lane == j) myd = d;
        const double r = fast_rcp(d);
        if (j + 1 < 16) a[j + 1] = fma(-(a[j] * ac[j + 1]), r, a[j + 1]);   // next pivot first: one FMA after r
        const double sc = a[j] * r;
#pragma unroll
        for (int c = j + 2; c < 16; ++c) a[c] = fma(-sc, ac[c], a[c]);
      }
      if (!(myd > 0.0)) myd = 1.0;
      const double myrinv = rsqrt(myd);                    // lane j < 16: 1 / sqrt(d_j)
      if (warp == 0 && isdiag) rdiag[o + lane] = myrinv;
#pragma unroll
      for (int j = 0; j < 16; ++j) a[j] *= __shfl_sync(0xffffffffu, myrinv, j);   // lane j: d_j / sqrt(d_j)
      if (live && (warp == 0 || !isdiag)) {
        double* dst = S + row * TLD + o;
#pragma unroll
        for (int c = 0; c < 16; c += 2) {
          double2 v;
          v.x = (isdiag && c > lane) ? 0.0 : a[c];
          v.y = (isdiag && c + 1 > lane) ? 0.0 : a[c + 1];
          *reinterpret_cast<double2*>(dst + c) = v;
        }
      }
    }
    cta_sync();
    if (npanel > 0) {
      // trailing update: S[r][c] -= sum_{m<16} S[r][o+m] S[c][o+m] for o+16 <= c <= r < 64, 8x8 blocks
      const int o2 = o + 16, nb8 = npanel / 8, g = lane >> 2, t = lane & 3;
      const int nblocks = nb8 * (nb8 + 1) / 2;
      for (int q0 = warp; q0 < nblocks; q0 += 3 * (kCholThreads / 32)) {
        double c[3][2];
        double* cp[3];
        const double *ap[3], *bp[3];
        bool on[3];
#pragma unroll
        for (int u = 0; u < 3; ++u) {
          const int q = q0 + u * (kCholThreads / 32);
          on[u] = q < nblocks;
          int rb = 0, rem = on[u] ? q : 0;
          while (rem >= rb + 1) { rem -= rb + 1; ++rb; }
          const int cb = rem;
          cp[u] = S + (o2 + rb * 8 + g) * TLD + o2 + cb * 8 + 2 * t;
          ap[u] = S + (o2 + rb * 8 + g) * TLD + o + t;
          bp[u] = S + (o2 + cb * 8 + g) * TLD + o + t;
          const double2 c0 = *reinterpret_cast<const double2*>(cp[u]);
          c[u][0] = c0.x; c[u][1] = c0.y;
        }
#pragma unroll
        for (int kk = 0; kk < 16; kk += 4)
#pragma unroll
          for (int u = 0; u < 3; ++u) dmma(c[u], -ap[u][kk], bp[u][kk]);
#pragma unroll
        for (int u = 0; u < 3; ++u)
          if (on[u]) *reinterpret_cast<double2*>(cp[u]) = make_double2(c[u][0], c[u][1]);
      }
      cta_sync();
    }
  }
  return ok;
}

// C (H x H, stride TLD) = sgn * A B with A, B row-major H x H blocks (stride TLD) in shared memory, on the
// FP64 tensor pipe; the H/8 x H/8 output blocks are dealt to `nw` warps, this warp being number `w`.
template <int H>
__device__ __forceinline__ void sub_mma(const double* __restrict__ A, const double* __restrict__ B, double* __restrict__ C,
                                        bool neg, int w, int nw, int lane) {
  const int g = lane >> 2, t = lane & 3;
  constexpr int NB = H / 8;
  for (int q = w; q < NB * NB; q += nw) {
    const int mb = q / NB, nb = q % NB;
    double c[2] = {0.0, 0.0};
    const double* ap = A + (mb * 8 + g) * TLD + t;
    const double* bp = B + t * TLD + nb * 8 + g;
#pragma unroll
    for (int kk = 0; kk < H; kk += 4) dmma(c, ap[kk], bp[kk * TLD]);
    *reinterpret_cast<double2*>(C + (mb * 8 + g) * TLD + nb * 8 + 2 * t) = neg ? make_double2(-c[0], -c[1]) : make_double2(c[0], c[1]);
  }
}

// X = S^-1 for the lower-triangular 64x64 tile S (stride TLD); X (stride TLD) gets the full tile
// (zeros above the diagonal).  16x16 diagonal blocks by column-oriented substitution (one thread per
// column, registers), then two merge levels  [A 0; B C]^-1 = [A^-1 0; -C^-1 (B A^-1)  C^-1]  whose small
// products run on the FP64 tensor pipe.  rdiag[r] = 1 / S[r][r].
__device__ __forceinline__ void tile_trinv(const double* __restrict__ S, const double* __restrict__ rdiag,
                                           double* __restrict__ X, int tid) {
  const int warp = tid >> 5, lane = tid & 31;
  for (int e = tid; e < CT * TLD / 2; e += kCholThreads) reinterpret_cast<double2*>(X)[e] = make_double2(0.0, 0.0);
  cta_sync();
  if (tid < CT) {
    const int b0 = (tid >> 4) * 16, c = tid & 15;
    double x[16];
#pragma unroll
    for (int r = 0; r < 16; ++r) x[r] = (r == c) ? 1.0 : 0.0;
#pragma unroll
    for (int m = 0; m < 16; ++m) {
      const double xm = x[m] * rdiag[b0 + m];
      x[m] = xm;
#pragma unroll
      for (int r = m + 1; r < 16; ++r) x[r] = fma(-S[(b0 + r) * TLD + b0 + m], xm, x[r]);
    }
#pragma unroll
    for (int r = 0; r < 16; ++r) X[(b0 + r) * TLD + b0 + c] = x[r];
  }
  cta_sync();
  {
    // h = 16: the two 32x32 diagonal blocks, half of the warps each
    const int off = (warp / (kCholWarps / 2)) * 32, w = warp % (kCholWarps / 2);
    sub_mma<16>(S + (off + 16) * TLD + off, X + off * TLD + off, X + off * TLD + off + 16, false, w, kCholWarps / 2, lane);      // T = B A^-1
    cta_sync();
    sub_mma<16>(X + (off + 16) * TLD + off + 16, X + off * TLD + off + 16, X + (off + 16) * TLD + off, true, w, kCholWarps / 2, lane);   // -C^-1 T
    cta_sync();
    for (int e = tid; e < 2 * 16 * 16; e += kCholThreads) {
      const int blk = e >> 8, r = (e >> 4) & 15, c = e & 15;
      X[(blk * 32 + r) * TLD + blk * 32 + 16 + c] = 0.0;
    }
    cta_sync();
  }
  {
    // h = 32
    sub_mma<32>(S + 32 * TLD, X, X + 32, false, warp, kCholWarps, lane);
    cta_sync();
    sub_mma<32>(X + 32 * TLD + 32, X + 32, X + 32 * TLD, true, warp, kCholWarps, lane);
    cta_sync();
    for (int e = tid; e < 32 * 32; e += kCholThreads) X[(e >> 5) * TLD + 32 + (e & 31)] = 0.0;
    cta_sync();
  }
}

__global__ void __launch_bounds__(kCholBlock, 1)
chol_task_kernel(const double* __restrict__ G, const double* __restrict__ lam_inv2, Ctl* __restrict__ ctl,
                 double* __restrict__ L, double* __restrict__ W, double* __restrict__ Wt, double* __restrict__ ws,
                 int* __restrict__ flags, const CholTask* __restrict__ tasks, const int* __restrict__ list_off, int p,
                 int nt, unsigned long long* __restrict__ trace, double* __restrict__ Lt,
                 const __grid_constant__ CUtensorMap tmL, const __grid_constant__ CUtensorMap tmWt) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  // the operand ring must be 1024-byte aligned (128-byte swizzle atom = 8 rows x 128 bytes)
  double* pool = reinterpret_cast<double*>(smem_raw + ((1024u - ((uint32_t)__cvta_generic_to_shared(smem_raw) & 1023u)) & 1023u));
  double* S = pool + kPoolDoubles;                   // 64 x TLD
  double* X = S + CT * TLD;                          // 64 x TLD
  double* rdiag = X + CT * TLD;                      // 64
  const int P = nt * CT;
  const int tid = threadIdx.x;
  const uint32_t pool_s = (uint32_t)__cvta_generic_to_shared(pool);
  const uint32_t x_s = pool_s + (uint32_t)((kPoolDoubles + CT * TLD) * sizeof(double));
  const uint32_t bar_s = pool_s + (uint32_t)((kPoolDoubles + 2 * CT * TLD + CT) * sizeof(double));   // full[NST], empty[NST]
  // chain CTA: compute warps -> publisher warp: R_inv (L_jj and W_jj are in shared memory), R_trsm (the stores of L(j+1,j)
  // are issued); publisher -> compute warps: F_x (X has been read: the next inverse may overwrite it), F_d (the diagonal
  // buffer has been read: the next TRSM may overwrite it)
  const uint32_t rel_s = bar_s + 8u * (2 * NST);
  const uint32_t R_inv = rel_s, R_trsm = rel_s + 8u, F_x = rel_s + 16u, F_d = rel_s + 24u;
  double* T2 = pool + kChainStages * kStageBytes / 8;   // chain CTA: third 64 x TLD tile buffer, in the unused half of the ring
  int* fL = flags;
  int* fB = flags + (size_t)nt * nt;
  int* fP = fB + (size_t)nt * nt;
  if (tid == 0) {
    for (int q = 0; q < NST; ++q) {
      cmbar_init(bar_s + 8u * q, 1);                       // full: the producer's arrive.expect_tx (+ the bytes)
      cmbar_init(bar_s + 8u * (NST + q), kCholWarps);      // empty: one arrival per compute warp
    }
    cmbar_init(R_inv, kCholWarps); cmbar_init(R_trsm, kCholWarps); cmbar_init(F_x, 1); cmbar_init(F_d, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();                                         // the only CTA-wide barrier: the producer warp leaves here
  const int t_beg = list_off[blockIdx.x], t_end = list_off[blockIdx.x + 1];

  if (tid >= kCholThreads) {
    // ---- producer warp (and, in the chain CTA, the publisher warp).  Producer: for every k-loop of this CTA's list, in order: wait for the operands' flags (the lanes look at
    // up to 32 k-tiles at once), wait for a free stage, and stream the two 64 x 32 operand chunks into it: four 2-D TMA
    // boxes (cp.async.bulk.tensor, 128-byte swizzle), issued by one lane.
    const int lane = tid & 31;
    uint32_t st = 0, ph = 0;
    const bool chain_cta = t_beg < t_end && tasks[t_beg].type >= 2;   // its list then holds chain tasks only
    if (tid >= kCholThreads + 32) {
      // ---- publisher warp (chain CTA only): writes the chain's results to global memory and publishes them, so that the
      // compute warps go straight from the inverse to TRSM.  Per column j: W_jj (from X) -> flag fL[j][j] (the column's tiles
      // wait for it: it goes first), Wt_jj -> flag fB[j][j], L_jj (and Lt_jj) from the diagonal buffer; then the flag of
      // L(j+1,j), whose stores the compute warps issue themselves (the st.release fence waits for them here, not there).
      if (!chain_cta) return;
      const double* D = S;
      const double* O = T2;
      uint32_t p_inv = 0, p_trsm = 0;
      for (int ti = t_beg; ti < t_end; ++ti) {
        const CholTask tk = tasks[ti];
        const int j_ = tk.j;
        if (tk.type == 2) {
          cmbar_wait(R_inv, p_inv); p_inv ^= 1u;
          const size_t g0 = (size_t)(j_ * CT) * P + j_ * CT;
#pragma unroll 8
          for (int r = 0; r < CT; ++r)
            *reinterpret_cast<double2*>(W + g0 + (size_t)r * P + 2 * lane) = *reinterpret_cast<const double2*>(X + r * TLD + 2 * lane);
          __syncwarp();
          if (lane == 0) st_release(&fL[(size_t)j_ * nt + j_], 1);
          // transposes: 8 rows x 4 columns per step in the pattern of a DMMA fragment (conflict-free with the padded
          // stride), 8 lanes store 64 contiguous bytes of a transposed row
          const int g = lane >> 2, t = lane & 3;
#pragma unroll 8
          for (int b = 0; b < (CT / 8) * (CT / 4); ++b) {
            const int r = (b / (CT / 4)) * 8 + g, c = (b % (CT / 4)) * 4 + t;
            Wt[g0 + (size_t)c * P + r] = X[r * TLD + c];
          }
          __syncwarp();
          if (lane == 0) { st_release(&fB[(size_t)j_ * nt + j_], 1); cmbar_arrive(F_x); }
#pragma unroll 8
          for (int r = 0; r < CT; ++r) {
            const int c = 2 * lane;
            double2 l = *reinterpret_cast<const double2*>(D + r * TLD + c);
            if (c > r) l.x = 0.0;
            if (c + 1 > r) l.y = 0.0;
            *reinterpret_cast<double2*>(L + g0 + (size_t)r * P + c) = l;
          }
          if (Lt != nullptr) {   // L^T, used by the block back-substitution when only a block-diagonal inverse is built
#pragma unroll 8
            for (int b = 0; b < (CT / 8) * (CT / 4); ++b) {
              const int r = (b / (CT / 4)) * 8 + g, c = (b % (CT / 4)) * 4 + t;
              Lt[g0 + (size_t)c * P + r] = c <= r ? D[r * TLD + c] : 0.0;
            }
          }
          __syncwarp();
          if (j_ + 1 < nt) {                                   // the flag of L(j+1,j): its stores were issued by TRSM(j)
            cmbar_wait(R_trsm, p_trsm); p_trsm ^= 1u;
            if (lane == 0) st_release(&fL[(size_t)(j_ + 1) * nt + j_], 1);
          }
          // F_d last: a phase of any of these barriers completes only after the other side has consumed the previous one
          // (parity waits cannot tell phases two apart)
          if (lane == 0) cmbar_arrive(F_d);
          { const double* q = D; D = O; O = q; }               // the buffers swap roles every column
        }
      }
      return;
    }
    if (chain_cta) {
      // ---- producer warp of the chain CTA: lane 0 fetches the parked accumulators of TRSM / SYRK (32 KB, contiguous) into
      // ring stages as soon as their prefix tasks have stored them -- normally while POTRF is still running
      if (lane == 0) {
        for (int ti = t_beg; ti < t_end; ++ti) {
          const CholTask tk = tasks[ti];
          if (tk.type < 3 || tk.slot_in < 0) continue;
          const uint32_t full = bar_s + 8u * st, empty = bar_s + 8u * (NST + st);
          while (ld_acquire(&fP[tk.slot_in]) == 0) __nanosleep(20);
          asm volatile("fence.proxy.async.global;" ::: "memory");
          cmbar_wait(empty, ph ^ 1u);
          cmbar_expect_tx(full, (uint32_t)(CT * CT * sizeof(double)));
          bulk_g2s(pool_s + st * (uint32_t)kStageBytes, ws + (size_t)tk.slot_in * CT * CT, (uint32_t)(CT * CT * sizeof(double)), full);
          if (++st == kChainStages) { st = 0; ph ^= 1u; }
        }
      }
      return;
    }
    for (int ti = t_beg; ti < t_end; ++ti) {
      const CholTask tk = tasks[ti];
      if (tk.type >= 2 || tk.kend <= tk.kbeg) continue;
      const bool isL = tk.type == 0;
      const int ra = isL ? tk.i : tk.j, rb = isL ? tk.j : tk.i;
      int k_known = tk.kbeg;                               // k-tiles below this are known to be ready
      for (int k = tk.kbeg; k < tk.kend; ++k) {
        if (k >= k_known) {
          // operand flags of k-tile kq: L(ra,kq) and L(rb,kq) (L tasks), L(ra,kq) and Wt(rb,kq) (inverse tiles)
          const int kq = k + lane;
          int n;
          for (;;) {
            bool ok = false;
            if (kq < tk.kend) {
              ok = ld_acquire(&fL[(size_t)ra * nt + kq]) != 0;
              if (isL) { if (rb != ra) ok = (ld_acquire(&fL[(size_t)rb * nt + kq]) != 0) && ok; }
              else ok = (ld_acquire(&fB[(size_t)rb * nt + kq]) != 0) && ok;   // kq == rb: the diagonal tile Wt_ii
            }
            const unsigned m = __ballot_sync(0xffffffffu, ok);
            n = __ffs(~m) - 1;
            if (n < 0) n = 32;
            if (n > 0) break;
            __nanosleep(20);
          }
          k_known = k + n;
          // the tiles were written through the generic proxy by other CTAs; the bulk copies read through the async proxy
          asm volatile("fence.proxy.async.global;" ::: "memory");
        }
#pragma unroll 1
        for (int kc = 0; kc < CT / KC; ++kc) {
          const uint32_t full = bar_s + 8u * st, empty = bar_s + 8u * (NST + st);
          cmbar_wait(empty, ph ^ 1u);
          if (lane == 0) cmbar_expect_tx(full, kStageTxBytes);
          if (lane == 0) {
            const uint32_t sa = pool_s + st * (uint32_t)kStageBytes;
            const uint32_t sb = sa + (uint32_t)((KC / KB) * kBoxBytes);
#pragma unroll
            for (int q = 0; q < KC / KB; ++q) {
              tma_box(sa + (uint32_t)(q * kBoxBytes), &tmL, k * CT + kc * KC + q * KB, ra * CT, full);
              tma_box(sb + (uint32_t)(q * kBoxBytes), isL ? &tmL : &tmWt, k * CT + kc * KC + q * KB, rb * CT, full);
            }
          }
          if (++st == NST) { st = 0; ph ^= 1u; }
        }
      }
    }
    return;
  }

  const Frag f(tid);
  const SwzFrag zf(f);
  const TriFrag zt(tid);
  uint32_t c_st = 0, c_ph = 0;                             // the compute warps' position in the ring
  const double tau_inv2 = ctl->tau_inv2;

  // c: the Q tile (ti, tj) in the accumulator layout, padded with the identity
  auto load_q_tile = [&](int ti_, int tj_, double (&a)[kMB][2][2]) {
#pragma unroll
    for (int mb = 0; mb < kMB; ++mb)
#pragma unroll
      for (int nb = 0; nb < 2; ++nb)
#pragma unroll
        for (int e = 0; e < 2; ++e) {
          double v = 0.0;
          const int gr = ti_ * CT + f.row0 + mb * 8 + f.g, gc = tj_ * CT + f.col0 + nb * 8 + 2 * f.t + e;
          if (gr < p && gc < p) {
            v = G[(size_t)gr * p + gc];
            if (gr == gc) v = fma(tau_inv2, lam_inv2[gr], v);
          } else if (gr == gc) v = 1.0;
          a[mb][nb][e] = v;
        }
  };
  auto load_slot = [&](int slot, double (&a)[kMB][2][2]) {
    wait_flag_cta(&fP[slot], tid);
    const double2* src = reinterpret_cast<const double2*>(ws + (size_t)slot * CT * CT);
#pragma unroll
    for (int q = 0; q < 2 * kMB; ++q) {
      const double2 v = __ldcg(src + q * kCholThreads + tid);
      a[q >> 1][q & 1][0] = v.x; a[q >> 1][q & 1][1] = v.y;
    }
  };
  // the same accumulator, prefetched into the next ring stage by the producer warp (chain tasks)
  auto load_slot_ring = [&](double (&a)[kMB][2][2]) {
    cmbar_wait(bar_s + 8u * c_st, c_ph);
    const uint32_t src = pool_s + c_st * (uint32_t)kStageBytes + (uint32_t)(tid * sizeof(double2));
#pragma unroll
    for (int q = 0; q < 2 * kMB; ++q) {
      const double2 v = lds_f64x2(src + (uint32_t)(q * kCholThreads * sizeof(double2)));
      a[q >> 1][q & 1][0] = v.x; a[q >> 1][q & 1][1] = v.y;
    }
    __syncwarp();
    if ((tid & 31) == 0) cmbar_arrive(bar_s + 8u * (NST + c_st));
    if (++c_st == kChainStages) { c_st = 0; c_ph ^= 1u; }
  };
  auto acc_to_smem = [&](const double (&a)[kMB][2][2], double* T) {
#pragma unroll
    for (int mb = 0; mb < kMB; ++mb)
#pragma unroll
      for (int nb = 0; nb < 2; ++nb)
        *reinterpret_cast<double2*>(T + (f.row0 + mb * 8 + f.g) * TLD + f.col0 + nb * 8 + 2 * f.t) = make_double2(a[mb][nb][0], a[mb][nb][1]);
  };
  // diagonal tile outside the chain CTA (single-CTA schedules): L_jj = chol(S), W_jj = L_jj^-1 (X), both written out (with Wt
  // and, if asked for, Lt).  W_jj is published by flag fL[j][j] (the off-diagonal tiles of the column wait for it), Wt_jj by
  // fB[j][j] (inverse tiles).
  auto diag_finish = [&](int j_) {
    const bool ok = tile_potrf(S, rdiag, tid);
    if (!ok && tid == 0) atomicCAS(&ctl->status, 0, -4);
    tile_trinv(S, rdiag, X, tid);
    for (int e = tid; e < CT * CT / 2; e += kCholThreads) {
      const int r = e / (CT / 2), c = (e % (CT / 2)) * 2;
      const size_t g = (size_t)(j_ * CT + r) * P + j_ * CT + c;
      *reinterpret_cast<double2*>(W + g) = *reinterpret_cast<const double2*>(X + r * TLD + c);
      double2 l = *reinterpret_cast<const double2*>(S + r * TLD + c);
      if (c > r) l.x = 0.0;
      if (c + 1 > r) l.y = 0.0;
      *reinterpret_cast<double2*>(L + g) = l;
    }
    {
      const int g = (tid >> 2) & 7, t = tid & 3, w = tid >> 5;
#pragma unroll 4
      for (int b = w; b < (CT / 8) * (CT / 4); b += kCholWarps) {
        const int r = (b / (CT / 4)) * 8 + g, c = (b % (CT / 4)) * 4 + t;
        const size_t gt = (size_t)(j_ * CT + c) * P + j_ * CT + r;
        Wt[gt] = X[r * TLD + c];
        if (Lt != nullptr) Lt[gt] = c <= r ? S[r * TLD + c] : 0.0;
      }
    }
    cta_sync();
    if (tid == 0) { st_release(&fL[(size_t)j_ * nt + j_], 1); st_release(&fB[(size_t)j_ * nt + j_], 1); }
  };
  double* Dbuf = S;                                        // chain CTA: the diagonal tile being factored ...
  double* Obuf = T2;                                       // ... and the sub-diagonal tile; they swap every column

  for (int ti = t_beg; ti < t_end; ++ti) {
    const CholTask tk = tasks[ti];
    if (trace != nullptr && tid == 0) trace[4 * (size_t)ti] = globaltimer_ns();
    if (tk.type >= 2) {
      // ---- chain tasks (dedicated CTA; S, X persist in shared memory from one chain task to the next)
      const int j = tk.j;
      double acc[kMB][2][2];
      if (tk.type == 2) {
        // POTRF(j): Dbuf holds A_jj (left there by SYRK(j-1); column 0: the Q tile).  The publisher warp writes the results out.
        if (j == 0) { load_q_tile(0, 0, acc); acc_to_smem(acc, Dbuf); }
        cta_sync();
        const bool ok = tile_potrf(Dbuf, rdiag, tid);
        if (!ok && tid == 0) atomicCAS(&ctl->status, 0, -4);
        if (trace != nullptr && tid == 0) trace[4 * (size_t)ti + 1] = globaltimer_ns();
        if (j > 0) {   // the publisher is done with column j-1: X may be overwritten, and so may the old diagonal buffer (TRSM(j))
          cmbar_wait(F_x, (uint32_t)((j - 1) & 1));
          cmbar_wait(F_d, (uint32_t)((j - 1) & 1));
        }
        tile_trinv(Dbuf, rdiag, X, tid);                        // ends with a barrier of the compute warps
        if ((tid & 31) == 0) cmbar_arrive(R_inv);
        if (trace != nullptr && tid == 0) trace[4 * (size_t)ti + 2] = globaltimer_ns();
      } else if (tk.type == 3) {
        // TRSM(j): L(j+1,j) = A W_jj^T, A = parked accumulator of (j+1,j) with every k < j applied (column 0: Q tile);
        // W_jj is still in X.  The product goes to global memory and stays in Obuf as the operand of SYRK(j).
        if (tk.slot_in >= 0) load_slot_ring(acc); else load_q_tile(j + 1, j, acc);
        // (Obuf was the diagonal buffer of column j-1: POTRF(j) has waited for the publisher to be done with it)
        acc_to_smem(acc, Obuf);
        cta_sync();
        double out[kMB][2][2];
#pragma unroll
        for (int mb = 0; mb < kMB; ++mb)
#pragma unroll
          for (int nb = 0; nb < 2; ++nb) out[mb][nb][0] = out[mb][nb][1] = 0.0;
        tile_mma_tri<TLD, TLD>(Obuf, X, zt, out);
#pragma unroll
        for (int mb = 0; mb < kMB; ++mb)
#pragma unroll
          for (int nb = 0; nb < 2; ++nb) {
            const int r = (j + 1) * CT + zt.row0 + mb * 8 + zt.g, c = j * CT + zt.col(nb);
            *reinterpret_cast<double2*>(L + (size_t)r * P + c) = make_double2(out[mb][nb][0], out[mb][nb][1]);
          }
        __syncwarp();
        if ((tid & 31) == 0) cmbar_arrive(R_trsm);       // L(j+1,j) is on its way: the publisher warp sets its flag
        if (Lt != nullptr) {
#pragma unroll
          for (int mb = 0; mb < kMB; ++mb)
#pragma unroll
            for (int nb = 0; nb < 2; ++nb) {
              const int r = (j + 1) * CT + zt.row0 + mb * 8 + zt.g, c = j * CT + zt.col(nb);
              Lt[(size_t)c * P + r] = out[mb][nb][0]; Lt[(size_t)(c + 1) * P + r] = out[mb][nb][1];
            }
        }
        cta_sync();                              // the product has been read from Obuf by every warp
#pragma unroll
        for (int mb = 0; mb < kMB; ++mb)
#pragma unroll
          for (int nb = 0; nb < 2; ++nb)
            *reinterpret_cast<double2*>(Obuf + (zt.row0 + mb * 8 + zt.g) * TLD + zt.col(nb)) = make_double2(out[mb][nb][0], out[mb][nb][1]);
        cta_sync();
      } else {
        // SYRK(j): A(j+1,j+1) = parked accumulator (every k < j applied; column 1: Q tile) - L(j+1,j) L(j+1,j)^T -> Obuf,
        // which becomes the diagonal buffer of column j+1
        if (tk.slot_in >= 0) load_slot_ring(acc); else load_q_tile(j + 1, j + 1, acc);
        tile_mma<TLD, TLD, CT, true, true>(Obuf, Obuf, f, acc);
        cta_sync();
        acc_to_smem(acc, Obuf);
        { double* q = Dbuf; Dbuf = Obuf; Obuf = q; }
      }
      if (trace != nullptr && tid == 0) {
        const unsigned long long tn = globaltimer_ns();
        if (tk.type != 2) { trace[4 * (size_t)ti + 1] = tn; trace[4 * (size_t)ti + 2] = tn; }
        trace[4 * (size_t)ti + 3] = tn;                    // chain tasks (always CTA 0): the end time goes to the last word
      }
      continue;
    }
    const bool isL = tk.type == 0;
    const int i = tk.i, j = tk.j;
    // the k loop: acc -= MA(ra,k) MB(rb,k)^T, operands streamed by the producer warp
    const int kbeg = tk.kbeg, kend = tk.kend;

    double acc[kMB][2][2];
    if (tk.slot_in >= 0) load_slot(tk.slot_in, acc);
    else if (isL) load_q_tile(i, j, acc);
    else {
#pragma unroll
      for (int mb = 0; mb < kMB; ++mb)
#pragma unroll
        for (int nb = 0; nb < 2; ++nb) acc[mb][nb][0] = acc[mb][nb][1] = 0.0;
    }

    const int nchunks = (kend - kbeg) * (CT / KC);
    cta_sync();                                      // S and X are free (previous task is over)
#pragma unroll 1
    for (int c = 0; c < nchunks; ++c) {
      cmbar_wait(bar_s + 8u * c_st, c_ph);
      const uint32_t sa = pool_s + c_st * (uint32_t)kStageBytes;
      tile_mma_s<true>(sa, sa + (uint32_t)((KC / KB) * kBoxBytes), zf, acc);
      __syncwarp();
      if ((tid & 31) == 0) cmbar_arrive(bar_s + 8u * (NST + c_st));
      if (++c_st == NST) { c_st = 0; c_ph ^= 1u; }
    }
    if (trace != nullptr && tid == 0) trace[4 * (size_t)ti + 1] = globaltimer_ns();

    if (tk.slot_out >= 0) {
      // ---- prefix task: park the partial accumulator
      double2* dst = reinterpret_cast<double2*>(ws + (size_t)tk.slot_out * CT * CT);
#pragma unroll
      for (int q = 0; q < 2 * kMB; ++q) __stcg(dst + q * kCholThreads + tid, make_double2(acc[q >> 1][q & 1][0], acc[q >> 1][q & 1][1]));
      cta_sync();
      if (tid == 0) st_release(&fP[tk.slot_out], 1);
    } else if (isL && i == j) {
      // ---- diagonal: L_jj = chol(acc), W_jj = L_jj^-1
      acc_to_smem(acc, S);
      cta_sync();
      diag_finish(j);
    } else {
      // ---- off-diagonal: multiply by W_jj (from global; written by the diagonal task of column j)
      wait_flag_cta(&fL[(size_t)j * nt + j], tid);
      const double* wjj = W + (size_t)j * CT * P + (size_t)j * CT;
#pragma unroll
      for (int it = 0; it < CT / kCholWarps; ++it) {
        const int row = (tid >> 5) + it * kCholWarps, pc = (tid & 31) * 2;
        cp_async16_s(x_s + (uint32_t)((row * TLD + pc) * sizeof(double)), wjj + (size_t)row * P + pc);
      }
      cp_async_commit();
      double out[kMB][2][2];
#pragma unroll
      for (int mb = 0; mb < kMB; ++mb)
#pragma unroll
        for (int nb = 0; nb < 2; ++nb) out[mb][nb][0] = out[mb][nb][1] = 0.0;
      if (isL) {
#pragma unroll
        for (int mb = 0; mb < kMB; ++mb)
#pragma unroll
          for (int nb = 0; nb < 2; ++nb)
            *reinterpret_cast<double2*>(S + (f.row0 + mb * 8 + f.g) * TLD + f.col0 + nb * 8 + 2 * f.t) =
                make_double2(acc[mb][nb][0], acc[mb][nb][1]);
        cp_async_wait<0>();
        cta_sync();
        tile_mma_tri<TLD, TLD>(S, X, zt, out);                     // L_ij = A W_jj^T
#pragma unroll
        for (int mb = 0; mb < kMB; ++mb)
#pragma unroll
          for (int nb = 0; nb < 2; ++nb)
          {
            const int r = i * CT + zt.row0 + mb * 8 + zt.g, c = j * CT + zt.col(nb);
            *reinterpret_cast<double2*>(L + (size_t)r * P + c) = make_double2(out[mb][nb][0], out[mb][nb][1]);
            if (Lt != nullptr) { Lt[(size_t)c * P + r] = out[mb][nb][0]; Lt[(size_t)(c + 1) * P + r] = out[mb][nb][1]; }
          }
        cta_sync();
        if (tid == 0) st_release(&fL[(size_t)i * nt + j], 1);
      } else {
#pragma unroll
        for (int mb = 0; mb < kMB; ++mb)
#pragma unroll
          for (int nb = 0; nb < 2; ++nb)
#pragma unroll
            for (int e = 0; e < 2; ++e)
              S[(f.col0 + nb * 8 + 2 * f.t + e) * TLD + f.row0 + mb * 8 + f.g] = acc[mb][nb][e];   // transposed
        cp_async_wait<0>();
        cta_sync();
        tile_mma<TLD, TLD, CT, false>(X, S, f, out);               // W_ji = W_jj A
#pragma unroll
        for (int mb = 0; mb < kMB; ++mb)
#pragma unroll
          for (int nb = 0; nb < 2; ++nb) {
            const int r = j * CT + f.row0 + mb * 8 + f.g, c = i * CT + f.col0 + nb * 8 + 2 * f.t;
            *reinterpret_cast<double2*>(W + (size_t)r * P + c) = make_double2(out[mb][nb][0], out[mb][nb][1]);
            Wt[(size_t)c * P + r] = out[mb][nb][0];
            Wt[(size_t)(c + 1) * P + r] = out[mb][nb][1];
          }
        cta_sync();
        if (tid == 0) st_release(&fB[(size_t)i * nt + j], 1);
      }
    }
    if (trace != nullptr && tid == 0) { trace[4 * (size_t)ti + 2] = globaltimer_ns(); trace[4 * (size_t)ti + 3] = blockIdx.x; }
  }
}

// ---- d2: beta = Q^-1 g + L^-T e as two triangular matrix-vector products with the inverse factor,
//   t = W g + e  (L t = g + L e)   and   beta = Wt t  (L^T beta = t),   e_j = Phi^-1(U_A(j, k, E)).
// One warp per row; a lane keeps up to 16 double2 of its row in flight (one pass covers 1024 columns).
// Both kernels are launched with programmatic stream serialisation: the first pass over the row of W / Wt
// (ready since the Cholesky branch joined) and the normal variate are issued BEFORE griddepcontrol.wait,
// i.e. while the preceding kernel (reduce / first product) is still running.
constexpr double kPassSatSms = 112.0;              // SMs at which the fused pass saturates HBM (measured: 116 -> 7.1 TB/s)
constexpr int kGemvWarps = 4;
constexpr int kGemvPass = 1024;                      // columns per pass: 32 lanes x 16 double2

__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_trigger() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }

__device__ __forceinline__ void gemv_load(double2 (&w)[16], const double* __restrict__ row, int base, int lo, int hi, int lane) {
#pragma unroll
  for (int i = 0; i < 16; ++i) {
    const int c = base + 2 * (lane + 32 * i);
    w[i] = (c >= lo && c < hi) ? __ldcg(reinterpret_cast<const double2*>(row + c)) : make_double2(0.0, 0.0);
  }
}
// x is written by the preceding kernel and read after griddepcontrol.wait: it must NOT be a const __restrict__
// (invariant, ld.global.nc) load, which the compiler may hoist above the wait; __ldcg is an ordinary L2 load.
__device__ __forceinline__ void gemv_dot(const double2 (&w)[16], const double* x, int base, int lo, int hi, int lane,
                                         double& s0, double& s1) {
#pragma unroll
  for (int i = 0; i < 16; ++i) {
    const int c = base + 2 * (lane + 32 * i);
    if (c >= lo && c < hi) {
      const double2 b = __ldcg(reinterpret_cast<const double2*>(x + c));
      s0 = fma(w[i].x, b.x, s0);
      s1 = fma(w[i].y, b.y, s1);
    }
  }
}

__global__ void __launch_bounds__(kGemvWarps * 32)
beta_gemv1_kernel(const double* __restrict__ W, const double* g, double* __restrict__ tv, int p, int P,
                  unsigned long long seed, const Ctl* __restrict__ ctl) {
  pdl_trigger();
  const int row = blockIdx.x * kGemvWarps + (threadIdx.x >> 5), lane = threadIdx.x & 31;
  const bool live = row < p;
  const double* w = W + (size_t)(live ? row : 0) * P;
  const int hi = live ? (row / CT + 1) * CT : 0;     // W is zero right of the diagonal inside its tile
  double2 wr[16];
  gemv_load(wr, w, 0, 0, hi, lane);
  double e = 0.0;
  if (lane == 0 && live) {
    const uint32_t sweep = (uint32_t)(ctl->sweep + 1ull);   // written by the previous sweep's last kernel: complete
    e = norm_inv(uniform_a(seed, (unsigned long long)row, sweep, TAG_E));
  }
  pdl_wait();                                        // g (reduce_partials_kernel) is complete and visible
  double s0 = 0.0, s1 = 0.0;
  gemv_dot(wr, g, 0, 0, hi, lane, s0, s1);
  for (int base = kGemvPass; base < hi; base += kGemvPass) {
    gemv_load(wr, w, base, 0, hi, lane);
    gemv_dot(wr, g, base, 0, hi, lane, s0, s1);
  }
  double s = s0 + s1;
#pragma unroll
  for (int off = 16; off >= 1; off >>= 1) s += __shfl_xor_sync(0xffffffffu, s, off);
  if (lane == 0 && live) tv[row] = s + e;
}

// Second product; also appends beta to the device history (row g of the hot-path table) and,
// in the last CTA to finish, advances the sweep counter k <- k + 1.
__global__ void __launch_bounds__(kGemvWarps * 32)
beta_gemv2_kernel(const double* __restrict__ Wt, const double* tv, double* __restrict__ beta, int p, int P,
                  Ctl* __restrict__ ctl) {
  pdl_trigger();
  const int row = blockIdx.x * kGemvWarps + (threadIdx.x >> 5), lane = threadIdx.x & 31;
  const bool live = row < p;
  const double* w = Wt + (size_t)(live ? row : 0) * P;
  const int lo = (row / CT) * CT, hi = live ? P : 0; // Wt is zero left of the diagonal inside its tile
  const int base0 = (lo / kGemvPass) * kGemvPass;
  double2 wr[16];
  gemv_load(wr, w, base0, lo, hi, lane);
  const unsigned long long k = ctl->sweep + 1ull;
  double* __restrict__ h_beta = ctl->h_beta;
  const unsigned long long hrow = k - 1ull - ctl->hist_base;
  pdl_wait();                                        // tv (beta_gemv1_kernel) is complete and visible
  double s0 = 0.0, s1 = 0.0;
  gemv_dot(wr, tv, base0, lo, hi, lane, s0, s1);
  for (int base = base0 + kGemvPass; base < hi; base += kGemvPass) {
    gemv_load(wr, w, base, lo, hi, lane);
    gemv_dot(wr, tv, base, lo, hi, lane, s0, s1);
  }
  double s = s0 + s1;
#pragma unroll
  for (int off = 16; off >= 1; off >>= 1) s += __shfl_xor_sync(0xffffffffu, s, off);
  if (lane == 0 && live) {
    beta[row] = s;
    if (h_beta != nullptr) h_beta[hrow * (unsigned long long)p + row] = s;
    if (!isfinite(s)) atomicCAS(&ctl->status, 0, -5);
  }
  __syncthreads();
  if (threadIdx.x == 0) {
    __threadfence();
    if (atomicAdd(&ctl->done, 1) == (int)gridDim.x - 1) { ctl->done = 0; ctl->sweep = k; }
  }
}

// ---- d2 with a block-diagonal inverse (p > 1280): block forward / backward substitution over super-blocks of
// B = 64 sb rows,   r_I = g_I - sum_{J<I} L_IJ t'_J,  t'_I = W_II r_I;   s_I = t'_I + e_I - sum_{J>I} (L_JI)^T beta_J,
// beta_I = Wt_II s_I  (L^T is stored by the Cholesky kernel as Lt, so every product reads rows).  One generic
// row-range x column-range product, a warp per row, chained by programmatic dependent launch:
//   out[row] = (in ? in[row] : 0) + (add_e ? e_row : 0) -/+ sum_{c in [lo(row), hi(row))} M[row][c] x[c]
// tri = 0: columns [c0, c1);  1: [c0, end of the row's tile) (W);  2: [start of the row's tile, c1) (Wt).
__global__ void __launch_bounds__(kGemvWarps * 32)
blk_gemv_kernel(const double* __restrict__ M, int P, int row0, int nrows, int c0, int c1, int tri, const double* x,
                const double* in, double* out, int subtract, int add_e, int p, unsigned long long seed,
                const Ctl* __restrict__ ctl) {
  pdl_trigger();
  const int row = row0 + blockIdx.x * kGemvWarps + (threadIdx.x >> 5), lane = threadIdx.x & 31;
  const bool live = row < row0 + nrows;
  const double* w = M + (size_t)(live ? row : row0) * P;
  int lo = c0, hi = c1;
  if (tri == 1) hi = (row / CT + 1) * CT;
  if (tri == 2) lo = (row / CT) * CT;
  if (!live) hi = lo;
  const int base0 = (lo / kGemvPass) * kGemvPass;
  double2 wr[16];
  gemv_load(wr, w, base0, lo, hi, lane);
  double e = 0.0;
  if (add_e && lane == 0 && live && row < p) {
    const uint32_t sweep = (uint32_t)(ctl->sweep + 1ull);
    e = norm_inv(uniform_a(seed, (unsigned long long)row, sweep, TAG_E));
  }
  pdl_wait();
  double s0 = 0.0, s1 = 0.0;
  gemv_dot(wr, x, base0, lo, hi, lane, s0, s1);
  for (int base = base0 + kGemvPass; base < hi; base += kGemvPass) {
    gemv_load(wr, w, base, lo, hi, lane);
    gemv_dot(wr, x, base, lo, hi, lane, s0, s1);
  }
  double s = s0 + s1;
#pragma unroll
  for (int off = 16; off >= 1; off >>= 1) s += __shfl_xor_sync(0xffffffffu, s, off);
  if (lane == 0 && live) {
    const double a = (in != nullptr ? __ldcg(in + row) : 0.0) + e;
    out[row] = subtract ? a - s : a + s;
  }
}

// finish of the block solve: status check, history append, k <- k + 1 (one CTA; after the last beta block)
__global__ void __launch_bounds__(256)
beta_finish_kernel(const double* beta, int p, Ctl* __restrict__ ctl) {
  pdl_wait();
  const unsigned long long k = ctl->sweep + 1ull;
  double* __restrict__ h_beta = ctl->h_beta;
  const unsigned long long hrow = k - 1ull - ctl->hist_base;
  bool bad = false;
  for (int j = threadIdx.x; j < p; j += blockDim.x) {
    const double b = __ldcg(beta + j);
    bad |= !isfinite(b);
    if (h_beta != nullptr) h_beta[hrow * (unsigned long long)p + j] = b;
  }
  if (bad) atomicCAS(&ctl->status, 0, -5);
  __syncthreads();
  if (threadIdx.x == 0) ctl->sweep = k;
}

// FREEZE_BETA (tests): beta stays; append it to the history and advance the sweep counter.
__global__ void __launch_bounds__(256)
beta_keep_kernel(const double* __restrict__ beta, int p, Ctl* __restrict__ ctl) {
  const unsigned long long k = ctl->sweep + 1ull;
  double* __restrict__ h_beta = ctl->h_beta;
  const unsigned long long hrow = k - 1ull - ctl->hist_base;
  if (h_beta != nullptr)
    for (int j = threadIdx.x; j < p; j += blockDim.x) h_beta[hrow * (unsigned long long)p + j] = beta[j];
  __syncthreads();
  if (threadIdx.x == 0) ctl->sweep = k;
}

// Build the static schedule and decide how many SMs the Cholesky branch gets.  When the cost model says the
// branch hides behind the fused pass on K SMs of its own (the pass keeps num_sms - K), the smallest such K
// is taken; otherwise the branch uses every SM and runs before/after the pass.
static cudaError_t make_tile_map(CUtensorMap* tm, const double* base, int P);

cudaError_t chol_plan_create(CholPlan* pl, int p, int num_sms, double fused_ms_estimate, const Options& opt) {
  pl->p = p; pl->nt = chol_tiles(p); pl->P = chol_ld(p);
  const int nt = pl->nt;
  // Inverse factor: the whole W = L^-1 for nt <= 20 (d2 is then two matrix-vector products); for larger p only the
  // diagonal super-blocks of sb x sb tiles (the full inverse would double the flops) and d2 is a block substitution.
  const int sb_env = opt_or(opt.chol_sb, 0);
  const int sb = sb_env > 0 ? std::min(sb_env, nt) : (nt <= 20 ? nt : 8);
  pl->sb = sb;
  const long long tile_tasks = (long long)nt * nt;
  CholSchedule best;
  int k_env = opt_or(opt.chol_ctas, 0);
  if (k_env > num_sms) k_env = num_sms;
  if (k_env > 0) {
    best = chol_build_schedule(nt, sb, (int)std::min<long long>(k_env, tile_tasks));
    pl->overlap = k_env < num_sms;
  } else {
    // the cost model is calibrated with the factor's working set in L2; when G, L, Lt (or W, Wt) do not fit beside
    // the X stream (p >= ~1500) the tile loads of the overlapped branch go to HBM: measured ~1.3x at p = 2000
    const double ws_mb = 3.0 * (double)pl->P * pl->P * 8.0 / 1e6;
    // 0.70: the branch is latency-bound and slows down with the SM clock, the HBM-bound pass does not -- under the
    // board's power cap (~1.5-1.7 GHz instead of 1.965) a branch sized to 85 % of the pass became the critical path
    // (C3, 1000 sweeps: 1699 sweeps/s with 16 SMs, 1731 with 20)
    const double budget_us = 0.70 * fused_ms_estimate * 1e3 / (ws_mb > 48.0 ? 1.3 : 1.0);
    const int cands[] = {2, 4, 6, 8, 10, 12, 16, 20, 24, 32, 40, 48};
    bool found = false;
    if (nt <= 40)
      for (int k : cands) {
        if (k > tile_tasks || k >= num_sms / 2) break;
        CholSchedule s = chol_build_schedule(nt, sb, k);
        if (s.makespan_us <= budget_us) { best = std::move(s); found = true; break; }
      }
    if (!found) {
      // nothing hides completely.  A small branch (small p: C1, C2) is still better run BESIDE the pass on a few SMs
      // than before it on all of them: compare  max(pass on the remaining SMs, 1.25 x branch on K)  with the serial sum.
      const int k_all = (int)std::min<long long>(num_sms, tile_tasks);
      CholSchedule serial = chol_build_schedule(nt, sb, k_all);
      const double fused_us = fused_ms_estimate * 1e3;
      double best_t = fused_us + serial.makespan_us;
      if (nt <= 8)
        for (int k : {1, 2, 4, 6, 8}) {
          if (k > tile_tasks || k >= num_sms / 2) break;
          CholSchedule s = chol_build_schedule(nt, sb, k);
          const double t = std::max(fused_us * num_sms / (num_sms - k), 1.25 * s.makespan_us);
          if (t < best_t) { best_t = t; best = std::move(s); found = true; }
        }
      // A large branch (p >= ~2000) that is longer than the pass: split the SMs so that both finish together.  The pass
      // streams X at full HBM bandwidth on ~kPassSatSms SMs and slows down in proportion below that; the branch is
      // bound by its work on few SMs and by the chain of diagonal tiles on many.  A split that does not beat running
      // the two one after the other on every SM by 5 % is not taken.
      if (!found && nt > 20) {
        double split_t = 0.95 * best_t;
        for (int k : {64, 72, 80, 88, 96, 104, 112, 120}) {
          if (k > tile_tasks || k > num_sms - 16) break;
          CholSchedule s = chol_build_schedule(nt, sb, k);
          const double pass_us = fused_us * std::max(1.0, kPassSatSms / (double)(num_sms - k - 2));   // two SMs stay spare (hsp_api.cu)
          const double t = std::max(pass_us, 1.05 * s.makespan_us);   // 1.05: tile loads compete with the X stream in L2
          if (t < split_t) { split_t = t; best = std::move(s); found = true; }
        }
      }
      if (!found) best = std::move(serial);
    }
    pl->overlap = found;
  }
  pl->K = best.K; pl->n_slots = best.n_slots; pl->n_tasks = (int)best.tasks.size(); pl->est_us = best.makespan_us;
  pl->n_flags = 2 * (size_t)nt * nt + (size_t)std::max(1, best.n_slots);
  cudaError_t e = cudaMalloc(&pl->d_tasks, best.tasks.size() * sizeof(CholTask));
  if (e == cudaSuccess) e = cudaMalloc(&pl->d_list_off, best.list_off.size() * sizeof(int));
  if (e == cudaSuccess) e = cudaMalloc(&pl->d_flags, pl->n_flags * sizeof(int));
  if (e == cudaSuccess) e = cudaMalloc(&pl->d_ws, (size_t)std::max(1, best.n_slots) * CT * CT * sizeof(double));
  if (e == cudaSuccess) e = cudaMemcpy(pl->d_tasks, best.tasks.data(), best.tasks.size() * sizeof(CholTask), cudaMemcpyHostToDevice);
  if (e == cudaSuccess) e = cudaMemcpy(pl->d_list_off, best.list_off.data(), best.list_off.size() * sizeof(int), cudaMemcpyHostToDevice);
  if (e == cudaSuccess && opt_or(opt.chol_trace, 0)) {
    e = cudaMalloc(&pl->d_trace, best.tasks.size() * 4 * sizeof(unsigned long long));
    if (e == cudaSuccess) e = cudaMemset(pl->d_trace, 0, best.tasks.size() * 4 * sizeof(unsigned long long));
  }
  pl->h_tasks = best.tasks;
  if (e == cudaSuccess) e = cudaFuncSetAttribute(chol_task_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kCholSmem);
  if (e == cudaSuccess) {   // look the driver's tensor-map encoder up now, outside any stream capture
    CUtensorMap probe;
    e = make_tile_map(&probe, pl->d_ws, 64);
  }
  return e;
}

void chol_plan_destroy(CholPlan* pl) {
  if (pl->d_tasks) cudaFree(pl->d_tasks);
  if (pl->d_list_off) cudaFree(pl->d_list_off);
  if (pl->d_flags) cudaFree(pl->d_flags);
  if (pl->d_ws) cudaFree(pl->d_ws);
  if (pl->d_trace) cudaFree(pl->d_trace);
  *pl = CholPlan{};
}

// Tensor map of a row-major P x P matrix of doubles for boxes of 16 columns x 64 rows with the 128-byte swizzle.  The
// driver entry point is looked up through the runtime (libhsp.so links only cudart).
static cudaError_t make_tile_map(CUtensorMap* tm, const double* base, int P) {
  typedef CUresult (*EncodeFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                               const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                               CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
  static EncodeFn encode = nullptr;
  if (!encode) {
    void* fn = nullptr;
    cudaDriverEntryPointQueryResult qres;
    const cudaError_t e = cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres);
    if (e != cudaSuccess) return e;
    if (qres != cudaDriverEntryPointSuccess || !fn) return cudaErrorNotSupported;
    encode = reinterpret_cast<EncodeFn>(fn);
  }
  const cuuint64_t gdim[2] = {(cuuint64_t)P, (cuuint64_t)P};
  const cuuint64_t gstride[1] = {(cuuint64_t)P * sizeof(double)};
  const cuuint32_t box[2] = {(cuuint32_t)KB, (cuuint32_t)CT};
  const cuuint32_t estride[2] = {1, 1};
  const CUresult r = encode(tm, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 2, const_cast<double*>(base), gdim, gstride, box, estride,
                            CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                            CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  return r == CUDA_SUCCESS ? cudaSuccess : cudaErrorInvalidValue;
}

cudaError_t cholesky_launch(const CholPlan& pl, const double* G, const double* lam_inv2, Ctl* ctl, double* L, double* W,
                            double* Wt, double* Lt, cudaStream_t st, long long* launches) {
  cudaError_t e = cudaMemsetAsync(pl.d_flags, 0, pl.n_flags * sizeof(int), st);
  if (e != cudaSuccess) return e;
  int p = pl.p, nt = pl.nt;
  CUtensorMap tmL, tmWt;
  e = make_tile_map(&tmL, L, pl.P);
  if (e == cudaSuccess) e = make_tile_map(&tmWt, Wt, pl.P);
  if (e != cudaSuccess) return e;
  double* ws = pl.d_ws; int* flags = pl.d_flags; const CholTask* tasks = pl.d_tasks; const int* list_off = pl.d_list_off;
  unsigned long long* trace = pl.d_trace;
  void* args[] = {(void*)&G, (void*)&lam_inv2, (void*)&ctl, (void*)&L, (void*)&W, (void*)&Wt, (void*)&ws, (void*)&flags,
                  (void*)&tasks, (void*)&list_off, (void*)&p, (void*)&nt, (void*)&trace, (void*)&Lt, (void*)&tmL, (void*)&tmWt};
  e = cudaLaunchCooperativeKernel((const void*)chol_task_kernel, dim3(pl.K), dim3(kCholBlock), args, kCholSmem, st);
  if (launches) ++*launches;
  return e;
}

template <typename... KArgs, typename... Args>
static cudaError_t launch_pdl(void (*kern)(KArgs...), int grid, int block, cudaStream_t st, bool pdl, Args... args) {
  cudaLaunchConfig_t cfg{};
  cfg.gridDim = dim3(grid); cfg.blockDim = dim3(block); cfg.dynamicSmemBytes = 0; cfg.stream = st;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  at[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = at; cfg.numAttrs = pdl ? 1 : 0;
  return cudaLaunchKernelEx(&cfg, kern, args...);
}

cudaError_t beta_solve_launch(const double* W, const double* Wt, const double* g, double* tv, double* beta, int p,
                              unsigned long long seed, Ctl* ctl, cudaStream_t st, long long* launches, bool pdl) {
  const int P = chol_ld(p);
  const int grid = (p + kGemvWarps - 1) / kGemvWarps;
  cudaError_t e = launch_pdl(beta_gemv1_kernel, grid, kGemvWarps * 32, st, pdl, W, g, tv, p, P, seed, (const Ctl*)ctl);
  if (e != cudaSuccess) return e;
  e = launch_pdl(beta_gemv2_kernel, grid, kGemvWarps * 32, st, pdl, Wt, (const double*)tv, beta, p, P, ctl);
  if (launches) *launches += 2;
  return e;
}

cudaError_t beta_block_solve_launch(const double* L, const double* Lt, const double* W, const double* Wt, const double* g,
                                    double* tv, double* rv, double* beta, int p, int sb, unsigned long long seed, Ctl* ctl,
                                    cudaStream_t st, long long* launches, bool pdl) {
  const int P = chol_ld(p), B = sb * CT, nsb = (P + B - 1) / B;
  const Ctl* cc = ctl;
  cudaError_t e = cudaSuccess;
  auto launch = [&](const double* M, int row0, int nrows, int c0, int c1, int tri, const double* x, const double* in,
                    double* out, int subtract, int add_e) {
    if (e != cudaSuccess) return;
    e = launch_pdl(blk_gemv_kernel, (nrows + kGemvWarps - 1) / kGemvWarps, kGemvWarps * 32, st, pdl, M, P, row0, nrows, c0,
                   c1, tri, x, in, out, subtract, add_e, p, seed, cc);
    if (launches) ++*launches;
  };
  // forward: tv = L^-1 g
  for (int I = 0; I < nsb; ++I) {
    const int r0 = I * B, nr = std::min(B, P - r0);
    const double* rhs = g;
    if (I > 0) { launch(L, r0, nr, 0, r0, 0, tv, g, rv, 1, 0); rhs = rv; }       // r_I = g_I - L_{I,<I} t'_{<I}
    launch(W, r0, nr, r0, r0 + nr, 1, rhs, nullptr, tv, 0, 0);                    // t'_I = W_II r_I
  }
  // backward: beta = L^-T (tv + e)
  for (int I = nsb - 1; I >= 0; --I) {
    const int r0 = I * B, nr = std::min(B, P - r0);
    launch(Lt, r0, nr, r0 + nr, P, 0, beta, tv, rv, 1, 1);                        // s_I = t'_I + e_I - (L_{>I,I})^T beta_{>I}
    launch(Wt, r0, nr, r0, r0 + nr, 2, rv, nullptr, beta, 0, 0);                  // beta_I = Wt_II s_I
  }
  if (e != cudaSuccess) return e;
  e = launch_pdl(beta_finish_kernel, 1, 256, st, pdl, (const double*)beta, p, ctl);
  if (launches) ++*launches;
  return e;
}

cudaError_t beta_keep_launch(const double* beta, int p, Ctl* ctl, cudaStream_t st) {
  beta_keep_kernel<<<1, 256, 0, st>>>(beta, p, ctl);
  return cudaGetLastError();
}

}  // namespace hsp
