// gram_tc.cu -- row c0 on the 5th-generation tensor cores: G = X^T X for fp32 X
// (PAPER.md:195), the one dense contraction of the method.
//
// tcgen05 has no fp32/fp64 kind, so every fp32 element is split into three bf16 pieces, x = h + m + l (each
// piece rounded to nearest, the remainders are exact in fp32), and a product x y is taken as the six bf16
// products  h h' + (h m' + m h') + (h l' + l h' + m m')  -- the dropped terms are below 2^-25 |x y| -- accumulated
// in fp32 in TMEM by `tcgen05.mma.kind::f16` (SASS UTCHMMA) and flushed into fp64 register accumulators every
// kTcFlushStages x 32 rows, so an fp32 accumulator never sums more than 128 rows.  The TMEM accumulation
// truncates (measured: a relative bias of -2e-6 with one accumulator flushed every 256 rows), so the large h h'
// products and the five small products go to two separate accumulators: the bias is then ~1e-7.
//
// One CTA per (128 x 128 lower tile of G, row slot).  X is row-major, so for a K-step of 16 rows both operands are
// "MN-major" (the 128 columns of a row are contiguous): the sixteen warps convert a 32-row stage of the A and B
// column blocks straight from global memory into the canonical no-swizzle MN-major shared-memory layout
// (8 x 8 core matrices of 128 bytes: 8 columns contiguous, rows 16 bytes apart; core matrices 128 B apart along
// MN (SBO) and 2 KB apart along K (LBO)), two stages double-buffered; one thread issues the 12 MMAs of a stage and
// commits them to an mbarrier, which frees the stage for the conversion two stages later.  Epilogue: TMEM lane =
// tile row; warp w of 16 reads lanes 32 (w % 4) .. +32, columns 32 (w / 4) .. +32 with tcgen05.ld.32x32b.x32.
#include <cuda_runtime.h>
#include <cuda_bf16.h>
#include <cstdint>
#include "hsp_internal.h"

namespace hsp {

constexpr int kTcTile = 128;                    // G tile edge (UMMA M = N = 128)
constexpr int kTcStageRows = 32;                // rows of X per stage = 2 K-steps of 16
constexpr int kTcThreads = 512;
constexpr int kTcFlushStages = 4;               // fp32 accumulation over at most 128 rows
constexpr int kTcPlaneBytes = kTcStageRows * kTcTile * 2;          // 8 KB: one bf16 piece of one operand, one stage
constexpr int kTcStageBytes = 2 * 3 * kTcPlaneBytes;               // A and B, three pieces each: 48 KB
constexpr size_t kTcSmem = 2 * kTcStageBytes + 64;                 // two stages + barriers / TMEM address

__device__ __forceinline__ uint32_t tc_smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

// shared-memory matrix descriptor, no swizzle, MN-major: start address, LBO (K direction), SBO (MN direction),
// all in 16-byte units; bits [46,48) = 1 (sm_100 descriptor version); layout type 0.
__device__ __forceinline__ uint64_t tc_desc(uint32_t addr) {
  const uint64_t lbo = (uint64_t)((16 * 128) >> 4), sbo = (uint64_t)(128 >> 4);
  return (uint64_t)((addr & 0x3FFFFu) >> 4) | (lbo << 16) | (sbo << 32) | (1ull << 46);
}
// instruction descriptor: D fp32, A and B bf16, both MN-major, N = 128, M = 128
constexpr uint32_t kTcIdesc = (1u << 4) | (1u << 7) | (1u << 10) | (1u << 15) | (1u << 16) | ((128u >> 3) << 17) | ((128u >> 4) << 24);

__device__ __forceinline__ void tc_mma(uint32_t d_tmem, uint64_t da, uint64_t db, uint32_t accumulate) {
  asm volatile(
      "{\n\t"
      ".reg .pred p;\n\t"
      "setp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t"
      "}" ::"r"(d_tmem),
      "l"(da), "l"(db), "r"(kTcIdesc), "r"(accumulate)
      : "memory");
}
__device__ __forceinline__ void tc_commit(uint32_t bar) {
  asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void tc_bar_wait(uint32_t bar, uint32_t parity) {
  asm volatile(
      "{\n\t"
      ".reg .pred P1;\n\t"
      "TC_WAIT:\n\t"
      "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n\t"
      "@P1 bra TC_DONE;\n\t"
      "bra TC_WAIT;\n\t"
      "TC_DONE:\n\t"
      "}" ::"r"(bar),
      "r"(parity)
      : "memory");
}
__device__ __forceinline__ void tc_ld32(uint32_t taddr, uint32_t (&v)[32]) {
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x32.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16,%17,%18,%19,%20,%21,"
      "%22,%23,%24,%25,%26,%27,%28,%29,%30,%31}, [%32];"
      : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]), "=r"(v[8]), "=r"(v[9]),
        "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15]), "=r"(v[16]), "=r"(v[17]), "=r"(v[18]),
        "=r"(v[19]), "=r"(v[20]), "=r"(v[21]), "=r"(v[22]), "=r"(v[23]), "=r"(v[24]), "=r"(v[25]), "=r"(v[26]), "=r"(v[27]),
        "=r"(v[28]), "=r"(v[29]), "=r"(v[30]), "=r"(v[31])
      : "r"(taddr)
      : "memory");
  asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
}

__device__ __forceinline__ void tc_ld16(uint32_t taddr, uint32_t (&v)[16]) {
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
      : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]), "=r"(v[8]), "=r"(v[9]),
        "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15])
      : "r"(taddr)
      : "memory");
  asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
}

// x = h + m + l in bf16 pieces; 8 consecutive columns -> one 16-byte unit per piece.  Two elements at a time:
// cvt.rn.bf16x2.f32 packs (hi <- first operand, lo <- second); a bf16 widened to fp32 is its 16 bits << 16.
__device__ __forceinline__ uint32_t tc_cvt2(float lo, float hi) {
  uint32_t d;
  asm("cvt.rn.bf16x2.f32 %0, %1, %2;" : "=r"(d) : "f"(hi), "f"(lo));
  return d;
}
__device__ __forceinline__ void tc_split8(const float (&x)[8], uint4& h, uint4& m, uint4& l) {
  uint32_t hp[4], mp[4], lp[4];
#pragma unroll
  for (int q = 0; q < 4; ++q) {
    const float a = x[2 * q], b = x[2 * q + 1];
    const uint32_t hw = tc_cvt2(a, b);
    const float ra = a - __uint_as_float(hw << 16), rb = b - __uint_as_float(hw & 0xffff0000u);     // exact
    const uint32_t mw = tc_cvt2(ra, rb);
    const float sa = ra - __uint_as_float(mw << 16), sb = rb - __uint_as_float(mw & 0xffff0000u);   // exact
    hp[q] = hw; mp[q] = mw; lp[q] = tc_cvt2(sa, sb);
  }
  h = make_uint4(hp[0], hp[1], hp[2], hp[3]);
  m = make_uint4(mp[0], mp[1], mp[2], mp[3]);
  l = make_uint4(lp[0], lp[1], lp[2], lp[3]);
}

__global__ void __launch_bounds__(kTcThreads, 1)
gram_tc_kernel(const float* __restrict__ X, long long N, int p, double* __restrict__ out, int slot0, long long rows_per_slot) {
  extern __shared__ __align__(128) unsigned char smem[];
  uint64_t* bars = reinterpret_cast<uint64_t*>(smem + 2 * kTcStageBytes);        // mma_done[2]
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(smem + 2 * kTcStageBytes + 16);
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  int t = blockIdx.x, ti = 0;
  while (t >= ti + 1) { t -= ti + 1; ++ti; }
  const int tj = t;
  const bool diag = ti == tj;
  const long long r_begin = (long long)(slot0 + blockIdx.y) * rows_per_slot;
  const long long r_end = (r_begin + rows_per_slot < N) ? r_begin + rows_per_slot : N;
  const int n_stages = r_end > r_begin ? (int)((r_end - r_begin + kTcStageRows - 1) / kTcStageRows) : 0;

  if (tid == 0) {
    for (int b = 0; b < 2; ++b)
      asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(tc_smem_u32(&bars[b])));
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (warp == 0) {   // two fp32 accumulators of 128 columns: [0,128) the h h' products, [128,256) the five small products
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 256;" ::"r"(tc_smem_u32(tmem_slot)) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  __syncthreads();
  asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
  const uint32_t tmem = *tmem_slot;

  double acc[32];                                    // tile row 32 (warp % 4) + lane, columns 32 (warp / 4) .. +32
#pragma unroll
  for (int c = 0; c < 32; ++c) acc[c] = 0.0;
  const uint32_t smem0 = tc_smem_u32(smem);
  const uint32_t bar0 = tc_smem_u32(&bars[0]);
  const bool vec_ok = ((p & 3) == 0) && ((reinterpret_cast<uintptr_t>(X) & 15) == 0);
  const int k_in = lane & 7, mbsub = lane >> 3;
  uint32_t ph0 = 0u, ph1 = 0u;
  bool pend0 = false, pend1 = false;
  int since_flush = 0;

  // conversion work of this thread: 2 of the 32 warp-units (operand, 8-row group, group of 4 column blocks)
  float xr[2][8];
  auto load_stage = [&](int s) {
    const long long row0 = r_begin + (long long)s * kTcStageRows;
#pragma unroll
    for (int q = 0; q < 2; ++q) {
      const int u = warp + 16 * q, o = u >> 4, kg = (u >> 2) & 3, mb = (u & 3) * 4 + mbsub;
      const long long row = row0 + kg * 8 + k_in;
      const int col0 = (o == 0 ? ti : tj) * kTcTile + mb * 8;
      if (o == 1 && diag) continue;
      if (s < n_stages && row < r_end && vec_ok && col0 + 8 <= p) {
        const float4 a = __ldg(reinterpret_cast<const float4*>(X + (size_t)row * p + col0));
        const float4 b = __ldg(reinterpret_cast<const float4*>(X + (size_t)row * p + col0 + 4));
        xr[q][0] = a.x; xr[q][1] = a.y; xr[q][2] = a.z; xr[q][3] = a.w; xr[q][4] = b.x; xr[q][5] = b.y; xr[q][6] = b.z; xr[q][7] = b.w;
      } else {
#pragma unroll
        for (int e = 0; e < 8; ++e) xr[q][e] = (s < n_stages && row < r_end && col0 + e < p) ? X[(size_t)row * p + col0 + e] : 0.f;
      }
    }
  };
  load_stage(0);

  for (int s = 0; s < n_stages; ++s) {
    const int buf = s & 1;
    // the MMAs of stage s-2 have consumed this buffer
    if (buf == 0 && pend0) { tc_bar_wait(bar0, ph0); ph0 ^= 1u; pend0 = false; }
    if (buf == 1 && pend1) { tc_bar_wait(bar0 + 8u, ph1); ph1 ^= 1u; pend1 = false; }
#pragma unroll
    for (int q = 0; q < 2; ++q) {
      const int u = warp + 16 * q, o = u >> 4, kg = (u >> 2) & 3, mb = (u & 3) * 4 + mbsub;
      if (o == 1 && diag) continue;
      uint4 h, m, l;
      tc_split8(xr[q], h, m, l);
      unsigned char* dst = smem + (size_t)buf * kTcStageBytes + (size_t)o * 3 * kTcPlaneBytes + ((kg * 16 + mb) * 8 + k_in) * 16;
      *reinterpret_cast<uint4*>(dst) = h;
      *reinterpret_cast<uint4*>(dst + kTcPlaneBytes) = m;
      *reinterpret_cast<uint4*>(dst + 2 * kTcPlaneBytes) = l;
    }
    load_stage(s + 1);                                               // in flight during the barrier and the next wait
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");     // generic-proxy writes -> visible to the MMA (async proxy)
    __syncthreads();
    if (tid == 0) {
      asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
      const uint32_t a0 = smem0 + (uint32_t)buf * kTcStageBytes;
      const uint32_t b0 = diag ? a0 : a0 + 3 * kTcPlaneBytes;
      const int pa[5] = {2, 0, 1, 1, 0}, pb[5] = {0, 2, 1, 0, 1};     // l h', h l', m m', m h', h m'
#pragma unroll
      for (int ks = 0; ks < 2; ++ks) {
        const uint32_t ko = ks * 2 * 2048;
        const uint32_t first = (since_flush > 0 || ks > 0) ? 1u : 0u;
        tc_mma(tmem, tc_desc(a0 + ko), tc_desc(b0 + ko), first);                                      // h h'
#pragma unroll
        for (int q = 0; q < 5; ++q)
          tc_mma(tmem + 128, tc_desc(a0 + pa[q] * kTcPlaneBytes + ko), tc_desc(b0 + pb[q] * kTcPlaneBytes + ko),
                 (first || q > 0) ? 1u : 0u);
      }
      tc_commit(bar0 + 8u * buf);
    }
    if (buf == 0) pend0 = true; else pend1 = true;
    ++since_flush;
    if (since_flush == kTcFlushStages || s == n_stages - 1) {
      // ---- flush: every MMA issued so far is complete once the commits of both buffers have arrived
      if (pend0) { tc_bar_wait(bar0, ph0); ph0 ^= 1u; pend0 = false; }
      if (pend1) { tc_bar_wait(bar0 + 8u, ph1); ph1 ^= 1u; pend1 = false; }
      asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
      const uint32_t taddr = tmem + ((uint32_t)(32 * (warp & 3)) << 16) + (uint32_t)(32 * (warp >> 2));
      {
        // big + small in fp32 (round to nearest: ~1e-5 absolute per flush, unbiased), then ONE conversion per entry:
        // F2F.F64.F32 runs at 16 per clock and SM and would otherwise dominate the flush
#pragma unroll
        for (int hh = 0; hh < 2; ++hh) {
          uint32_t v[16], w[16];
          tc_ld16(taddr + 16 * hh, v);
          tc_ld16(taddr + 128 + 16 * hh, w);
#pragma unroll
          for (int c = 0; c < 16; ++c) acc[16 * hh + c] += (double)(__uint_as_float(v[c]) + __uint_as_float(w[c]));
        }
      }
      asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
      __syncthreads();
      since_flush = 0;
    }
  }
  // ---- store the lower part of the tile into this slot
  {
    const int row = ti * kTcTile + 32 * (warp & 3) + lane;
    double* dst = out + (size_t)(slot0 + blockIdx.y) * p * p;
#pragma unroll
    for (int c = 0; c < 32; ++c) {
      const int col = tj * kTcTile + 32 * (warp >> 2) + c;
      if (row < p && col < p && col <= row) dst[(size_t)row * p + col] = acc[c];
    }
  }
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  __syncthreads();
  if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 256;" ::"r"(tmem) : "memory");
}

int gram_tc_tiles(int p) { const int ts = (p + kTcTile - 1) / kTcTile; return ts * (ts + 1) / 2; }

cudaError_t gram_tc_chunk_launch(const GramPlan& g, int chunk, const float* X, long long N, int p, double* scratch, cudaStream_t st) {
  if (chunk == 0) {   // per-device attribute: set for the current device at every create (chunk 0), not once per process
    cudaError_t e = cudaFuncSetAttribute(gram_tc_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kTcSmem);
    if (e != cudaSuccess) return e;
  }
  dim3 grid(gram_tc_tiles(p), g.slots_per_chunk);
  gram_tc_kernel<<<grid, kTcThreads, kTcSmem, st>>>(X, N, p, scratch, chunk * g.slots_per_chunk, g.rows_per_slot);
  return cudaGetLastError();
}

}  // namespace hsp
