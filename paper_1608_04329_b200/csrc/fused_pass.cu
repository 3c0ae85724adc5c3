// fused_pass.cu -- rows a1, a2, a3 and b of the hot path (include/hsp.h):
//   one streaming pass over X that computes eta_i = x_i.beta, draws
//   z_i ~ TN(eta_i,1) on the side fixed by y_i and accumulates X^T z
//    from the same on-chip tile, so X is read from HBM once per sweep; then a
//   fixed-order reduction of the per-CTA partials.
//
// Two kernels:
//   fused_pass_tma     persistent, warp-specialised: one producer thread streams row tiles with
//                      cp.async.bulk (TMA, 1-D: a tile of R rows is contiguous in row-major X) into
//                      an S-stage shared-memory ring guarded by mbarriers; 8 compute warps own
//                      fixed column stripes (eta partials -> shuffle reduce -> smem; later, x*z
//                      accumulation from the same stage); 4 sampler warps turn eta into z (Philox +
//                      inverse-CDF) D tiles behind the eta phase, so the sampler's latency is hidden
//                      behind the stream.  Static tile->CTA map: bit-reproducible run to run.
//   fused_pass_generic any p, any alignment (rows not a multiple of 16 bytes, or narrow p):
//                      thread-per-row eta + sampler, then thread-per-column accumulation that
//                      re-reads the 256-row tile from L1/L2.
#include <cuda_runtime.h>
#include <cstdint>
#include <cstdlib>
#include <cstdio>
#include <type_traits>
#include "hsp_device.cuh"
#include "hsp_internal.h"

namespace hsp {

// ------------------------------------------------------------------------------------------------
// PTX helpers (mbarrier + 1-D bulk copy)
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t* bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
  asm volatile(
      "{\n\t"
      ".reg .pred P1;\n\t"
      "WAIT_LOOP:\n\t"
      "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n\t"
      "@P1 bra DONE;\n\t"
      "bra WAIT_LOOP;\n\t"
      "DONE:\n\t"
      "}" ::"r"(smem_u32(bar)),
      "r"(parity)
      : "memory");
}
// X is streamed once per sweep: its lines are marked evict-first in L2 so that the stream does not push out
// the p x p working set of the concurrent Cholesky branch (L, W, Wt are re-read ~p/64 times per sweep).
__device__ __forceinline__ uint64_t l2_evict_first_policy() {
  uint64_t pol;
  asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
  return pol;
}
__device__ __forceinline__ void mbar_arrive_a(uint32_t bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_wait_a(uint32_t bar, uint32_t parity) {
  asm volatile(
      "{\n\t"
      ".reg .pred P1;\n\t"
      "WAIT_LOOP:\n\t"
      "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n\t"
      "@P1 bra DONE;\n\t"
      "bra WAIT_LOOP;\n\t"
      "DONE:\n\t"
      "}" ::"r"(bar),
      "r"(parity)
      : "memory");
}
__device__ __forceinline__ float4 ld_shared_f32x4(uint32_t a) {
  float4 v;
  asm volatile("ld.shared.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(a));
  return v;
}
__device__ __forceinline__ float2 ld_shared_f32x2(uint32_t a) {
  float2 v;
  asm volatile("ld.shared.v2.f32 {%0,%1}, [%2];" : "=f"(v.x), "=f"(v.y) : "r"(a));
  return v;
}
__device__ __forceinline__ float ld_shared_f32(uint32_t a) {
  float v;
  asm volatile("ld.shared.f32 %0, [%1];" : "=f"(v) : "r"(a));
  return v;
}
__device__ __forceinline__ double2 ld_shared_f64x2(uint32_t a) {
  double2 v;
  asm volatile("ld.shared.v2.f64 {%0,%1}, [%2];" : "=d"(v.x), "=d"(v.y) : "r"(a));
  return v;
}
__device__ __forceinline__ double ld_shared_f64(uint32_t a) {
  double v;
  asm volatile("ld.shared.f64 %0, [%1];" : "=d"(v) : "r"(a));
  return v;
}
__device__ __forceinline__ void st_shared_f64(uint32_t a, double v) {
  asm volatile("st.shared.f64 [%0], %1;" ::"r"(a), "d"(v) : "memory");
}
__device__ __forceinline__ void bulk_g2s(void* dst_smem, const void* src_gmem, uint32_t bytes, uint64_t* bar, uint64_t pol) {
  asm volatile(
      "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;" ::"r"(
          smem_u32(dst_smem)),
      "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar)), "l"(pol)
      : "memory");
}

// ------------------------------------------------------------------------------------------------
// Column-stripe arithmetic for one 16-byte vector of X
// ------------------------------------------------------------------------------------------------
template <typename XT> struct Vec;
template <> struct Vec<float> {
  static constexpr int V = 4;
  using Acc = float;
  float4 v;
  __device__ __forceinline__ void load(uint32_t smem_addr) { v = ld_shared_f32x4(smem_addr); }
  __device__ __forceinline__ double dot(const double* b) const {
    double s = (double)v.x * b[0];
    s = fma((double)v.y, b[1], s);
    s = fma((double)v.z, b[2], s);
    s = fma((double)v.w, b[3], s);
    return s;
  }
  // fp32 chain of 4 (eta modes 1, 2): at most 4 roundings of 2^-24 relative to the running partial
  __device__ __forceinline__ float dotf(const float* b) const {
    float s = v.x * b[0];
    s = fmaf(v.y, b[1], s);
    s = fmaf(v.z, b[2], s);
    s = fmaf(v.w, b[3], s);
    return s;
  }
  __device__ __forceinline__ void axpy(float z, float* acc) const {
    acc[0] = fmaf(v.x, z, acc[0]);
    acc[1] = fmaf(v.y, z, acc[1]);
    acc[2] = fmaf(v.z, z, acc[2]);
    acc[3] = fmaf(v.w, z, acc[3]);
  }
};
template <> struct Vec<double> {
  static constexpr int V = 2;
  using Acc = double;
  double2 v;
  __device__ __forceinline__ void load(uint32_t smem_addr) { v = ld_shared_f64x2(smem_addr); }
  __device__ __forceinline__ double dot(const double* b) const { return fma(v.y, b[1], v.x * b[0]); }
  __device__ __forceinline__ float dotf(const float*) const { return 0.f; }   // never used: fp64 X is always eta mode 0
  __device__ __forceinline__ void axpy(double z, double* acc) const {
    acc[0] = fma(v.x, z, acc[0]);
    acc[1] = fma(v.y, z, acc[1]);
  }
};

// Reduce RT per-lane values over the 32 lanes of a warp with a fixed butterfly; on return v[0] of
// lane l is the warp total of row rows_of_lane<RT>(l).  (RT + 4..5 shuffles instead of 5 RT.)
template <typename T, int RT>
__device__ __forceinline__ T warp_reduce_rows(T (&v)[RT], int lane) {
  int off = 16;
#pragma unroll
  for (int n = RT; n > 1; n >>= 1, off >>= 1) {
    const bool upper = (lane & off) != 0;
#pragma unroll
    for (int i = 0; i < n / 2; ++i) {
      const T send = upper ? v[i] : v[i + n / 2];
      const T keep = upper ? v[i + n / 2] : v[i];
      v[i] = keep + __shfl_xor_sync(0xffffffffu, send, off);
    }
  }
  for (; off >= 1; off >>= 1) v[0] += __shfl_xor_sync(0xffffffffu, v[0], off);
  return v[0];
}
template <int RT>
__device__ __forceinline__ int row_of_lane(int lane) {
  int row = 0, off = 16;
#pragma unroll
  for (int n = RT; n > 1; n >>= 1, off >>= 1) row += (lane & off) ? n / 2 : 0;
  return row;
}

constexpr int kComputeWarpsAll = 16;             // compute warps per CTA
constexpr int kComputeThreadsAll = kComputeWarpsAll * 32;
constexpr int kSamplerWarps = 4;
constexpr int kTmaThreads = (kComputeWarpsAll + kSamplerWarps + 1) * 32;   // 672
constexpr int kFlushRows = 16;   // fp32 x*z chains are flushed into the fp64 accumulators every >= 16 rows

struct TmaSmemLayout {
  size_t tiles, eta_part, z64, z32, bars, total;
  // WPR: warps that share one row (they cover its columns); R: rows per tile
  __host__ __device__ TmaSmemLayout(int S, int R, int WPR, size_t stage_bytes) {
    tiles = 0;
    eta_part = tiles + (size_t)S * stage_bytes;
    z64 = eta_part + (size_t)S * WPR * R * sizeof(double);
    z32 = z64 + (size_t)S * R * sizeof(double);
    bars = (z32 + (size_t)S * R * sizeof(float) + 15) & ~(size_t)15;
    total = bars + (size_t)4 * S * sizeof(uint64_t);
  }
};

// The 512 compute threads form 512/W row groups of W threads (W = 256 or 512).  Thread t of a group owns the
// 16-byte column stripes (c*W + t)*V, c < C, of the rows [grp RT/G, (grp+1) RT/G) of every tile, keeps the
// X^T z accumulators of those columns in registers for the whole kernel and writes its group's partial row.
// Narrow rows (p <= 256 V) use two groups of 8 warps; wide rows one group of 16 warps, which halves the
// per-thread column state (accumulators, beta) and keeps the kernel free of spills up to p = 8192 fp32.
//
// EM, the arithmetic of the eta phase for fp32 X (fp64 X is always mode 0):
//   0  every element converted exactly to fp64, DFMA chain, fp64 butterfly       (z matches the oracle to ~1e-13)
//   2  fp32 FMA chains of 4 elements, fp32 butterfly, converted once per warp and row (~3e-7)
// Both are far inside north_star's 1e-4 for fp32 X; mode 2 trades the 4 F2F.F64.F32 + 4 DFMA per 16-byte vector
// (the conversion runs at a quarter of the FP64 rate through the MIO queue and made the pass SM-bound) for 4 FFMA.
template <typename XT, int RT, int C, int W, int EM>
__global__ void __launch_bounds__(kTmaThreads, 1)
fused_pass_tma(const XT* __restrict__ X, const unsigned char* __restrict__ y, long long N, int p,
               unsigned long long seed, const double* __restrict__ beta, const Ctl* __restrict__ ctl,
               double* __restrict__ partial, double* __restrict__ z_out, int S, int D, long long n_tiles, long long row_off) {
  constexpr int V = Vec<XT>::V;
  using Acc = typename Vec<XT>::Acc;
  constexpr bool kF32 = sizeof(XT) == 4;
  constexpr int G = kComputeThreadsAll / W;        // row groups
  constexpr int WPR = W / 32;                      // warps per row
  constexpr int RG = RT / G;                       // rows of a tile per group
  static_assert(RT % G == 0 && RG >= 1, "rows per tile must split evenly over the groups");
  extern __shared__ __align__(128) unsigned char smem[];
  const size_t row_bytes = (size_t)p * sizeof(XT);
  const size_t stage_bytes = ((size_t)RT * row_bytes + 127) & ~(size_t)127;
  const TmaSmemLayout lay(S, RT, WPR, stage_bytes);
  unsigned char* tiles = smem + lay.tiles;
  double* eta_part = reinterpret_cast<double*>(smem + lay.eta_part);
  double* z64 = reinterpret_cast<double*>(smem + lay.z64);
  float* z32 = reinterpret_cast<float*>(smem + lay.z32);
  uint64_t* full = reinterpret_cast<uint64_t*>(smem + lay.bars);
  uint64_t* empty = full + S;
  uint64_t* eta_full = empty + S;
  uint64_t* z_full = eta_full + S;

  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const long long cta = blockIdx.x, grid = gridDim.x;
  const long long my_tiles = cta < n_tiles ? (n_tiles - cta + grid - 1) / grid : 0;
  const uint32_t sweep = (uint32_t)(ctl->sweep + 1ull);

  if (tid == 0) {
    for (int s = 0; s < S; ++s) {
      mbar_init(&full[s], 1);
      mbar_init(&empty[s], kComputeWarpsAll);
      mbar_init(&eta_full[s], kComputeWarpsAll);
      mbar_init(&z_full[s], 1);
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  // Zero the ring once: rows of a ragged last tile that TMA does not write are then finite
  // (stale or zero) and contribute x * 0 = 0 in the xz phase, so the inner loops need no row guards.
  {
    const uint4 zero = make_uint4(0u, 0u, 0u, 0u);
    for (size_t o = (size_t)tid * 16; o < (size_t)S * stage_bytes; o += (size_t)kTmaThreads * 16)
      *reinterpret_cast<uint4*>(tiles + o) = zero;
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // generic writes before TMA writes
  }
  __syncthreads();

  if (warp == kComputeWarpsAll + kSamplerWarps) {
    // ===================== producer: one thread streams the tiles =====================
    if (lane == 0) {
      int st = 0;
      uint32_t ph = 0;
      const uint64_t pol = l2_evict_first_policy();
      for (long long n = 0; n < my_tiles; ++n) {
        mbar_wait(&empty[st], ph ^ 1u);
        const long long row0 = (cta + n * grid) * RT;
        const long long rows = (N - row0) < RT ? (N - row0) : RT;
        const uint32_t bytes = (uint32_t)((size_t)rows * row_bytes);
        mbar_arrive_expect_tx(&full[st], bytes);
        bulk_g2s(tiles + (size_t)st * stage_bytes, reinterpret_cast<const unsigned char*>(X) + (size_t)row0 * row_bytes,
                 bytes, &full[st], pol);
        if (++st == S) { st = 0; ph ^= 1u; }
      }
    }
  } else if (warp >= kComputeWarpsAll) {
    // ===================== sampler warps: eta -> z, D tiles behind the eta phase =====================
    // Tile n goes to sampler warp n mod ns.  ns <= S keeps every mbarrier wait at most one phase
    // behind (a waiter two phases behind would alias on the parity bit).
    const int sw = warp - kComputeWarpsAll;
    const int ns = S < kSamplerWarps ? S : kSamplerWarps;
    if (sw < ns) {
      // y is prefetched three tiles ahead: under a saturated HBM a lone 1-byte load takes microseconds
      auto load_y = [&](long long n) -> int {
        const long long i = (cta + n * grid) * RT + lane;
        return (n < my_tiles && lane < RT && i < N) ? (int)y[i] : 1;
      };
      int y0 = load_y(sw), y1 = load_y(sw + ns), y2 = load_y(sw + 2LL * ns);
      int st = sw;                  // sw < ns <= S
      uint32_t ph = 0;
      for (long long n = sw; n < my_tiles; n += ns) {
        const long long i = (cta + n * grid) * RT + lane;
        const bool valid = (lane < RT) && (i < N);
        const int y3 = load_y(n + 3LL * ns);
        // the Philox uniform does not depend on eta either: compute it before waiting
        const double u = uniform_a(seed, (unsigned long long)(row_off + (valid ? i : 0)), sweep, TAG_Z);
        const double ystar = 2.0 * (double)y0 - 1.0;
        mbar_wait(&eta_full[st], ph);
        double eta = 0.0;
        if (lane < RT) {
          const double* ep = eta_part + (size_t)st * WPR * RT + lane;
#pragma unroll
          for (int w = 0; w < WPR; ++w) eta += ep[w * RT];
        }
        const double wpos = tnpos(ystar * eta, u);
        const double z = valid ? ystar * wpos : 0.0;
        if (lane < RT) {
          z64[st * RT + lane] = z;
          z32[st * RT + lane] = (float)z;
        }
        if (valid && z_out != nullptr) z_out[i] = z;
        __syncwarp();
        if (lane == 0) mbar_arrive(&z_full[st]);
        y0 = y1; y1 = y2; y2 = y3;
        st += ns;
        if (st >= S) { st -= S; ph ^= 1u; }
      }
    }
  } else {
    // ===================== compute warps: eta partials, then x*z from the same stage =====================
    // Stripes past p read column 0 with beta = 0 and are never written back, so the loops below are
    // straight-line code.  All shared-memory addresses are 32-bit and advance incrementally with the ring.
    const int grp = tid / W, wg = (tid % W) >> 5, gt = tid % W;
    double breg[EM == 0 ? C : 1][V];
    float bregf[EM == 0 ? 1 : C][V];
    double acc64[C][V];
    Acc acc[C][V];
    uint32_t coff[C];
#pragma unroll
    for (int c = 0; c < C; ++c) {
      const int col = (c * W + gt) * V;
      coff[c] = (col < p) ? (uint32_t)(col * sizeof(XT)) : 0u;
#pragma unroll
      for (int v = 0; v < V; ++v) {
        const double bv = (col + v < p) ? beta[col + v] : 0.0;
        if constexpr (EM == 0) breg[c][v] = bv; else bregf[c][v] = (float)bv;
        acc64[c][v] = 0.0;
        acc[c][v] = (Acc)0;
      }
    }
    const int my_row = grp * RG + row_of_lane<RG>(lane);
    const bool writer = (lane & (32 / RG - 1)) == 0;
    const uint32_t rb = (uint32_t)row_bytes, sb = (uint32_t)stage_bytes;
    const uint32_t tiles0 = smem_u32(tiles) + (uint32_t)(grp * RG) * rb;      // this group's first row, stage 0
    const uint32_t tiles_end = tiles0 + (uint32_t)S * sb;
    const uint32_t full0 = smem_u32(full), empty0 = smem_u32(empty), etaf0 = smem_u32(eta_full), zf0 = smem_u32(z_full);
    const uint32_t epart0 = smem_u32(eta_part) + (uint32_t)((wg * RT + my_row) * sizeof(double));
    const uint32_t zsrc0 = kF32 ? smem_u32(z32) + (uint32_t)(grp * RG * sizeof(float))
                                : smem_u32(z64) + (uint32_t)(grp * RG * sizeof(double));
    constexpr uint32_t kEpStride = WPR * RT * sizeof(double), kZStride = RT * (kF32 ? sizeof(float) : sizeof(double));
    int rows_since_flush = 0;
    // eta phase on the tile in stage st (phase parity ph); x*z phase on the tile in stage st.  Called with literal
    // stage numbers from the unrolled steady-state body below, every address below folds into an immediate.
    auto eta_phase = [&](uint32_t st, uint32_t ph) {
      mbar_wait_a(full0 + 8u * st, ph);
      const uint32_t tile = tiles0 + st * sb;
        double tot;
        if constexpr (EM == 0) {
          double part[RG];
#pragma unroll
          for (int r = 0; r < RG; ++r) part[r] = 0.0;
#pragma unroll
          for (int c = 0; c < C; ++c) {
            Vec<XT> x[RG];
#pragma unroll
            for (int r = 0; r < RG; ++r) x[r].load(tile + r * rb + coff[c]);
#pragma unroll
            for (int r = 0; r < RG; ++r) part[r] += x[r].dot(breg[c]);
          }
          tot = warp_reduce_rows<double, RG>(part, lane);
        } else {
          float part[RG];
#pragma unroll
          for (int r = 0; r < RG; ++r) part[r] = 0.f;
#pragma unroll
          for (int c = 0; c < C; ++c) {
            Vec<XT> x[RG];
#pragma unroll
            for (int r = 0; r < RG; ++r) x[r].load(tile + r * rb + coff[c]);
#pragma unroll
            for (int r = 0; r < RG; ++r) part[r] += x[r].dotf(bregf[c]);
          }
          tot = (double)warp_reduce_rows<float, RG>(part, lane);
        }
      if (writer) st_shared_f64(epart0 + st * kEpStride, tot);
      __syncwarp();
      if (lane == 0) mbar_arrive_a(etaf0 + 8u * st);
    };
    auto xz_phase = [&](uint32_t st, uint32_t ph) {
      mbar_wait_a(zf0 + 8u * st, ph);
      const uint32_t tile = tiles0 + st * sb;
        Acc zr[RG];
        const uint32_t zp = zsrc0 + st * kZStride;
        if constexpr (kF32) {
          if constexpr (RG % 4 == 0) {
#pragma unroll
            for (int q = 0; q < RG / 4; ++q) {
              const float4 t = ld_shared_f32x4(zp + 16 * q);
              zr[4 * q] = t.x; zr[4 * q + 1] = t.y; zr[4 * q + 2] = t.z; zr[4 * q + 3] = t.w;
            }
          } else if constexpr (RG == 2) {
            const float2 t = ld_shared_f32x2(zp);
            zr[0] = t.x; zr[1] = t.y;
          } else {
            zr[0] = ld_shared_f32(zp);
          }
        } else {
          if constexpr (RG % 2 == 0) {
#pragma unroll
            for (int q = 0; q < RG / 2; ++q) {
              const double2 t = ld_shared_f64x2(zp + 16 * q);
              zr[2 * q] = t.x; zr[2 * q + 1] = t.y;
            }
          } else {
            zr[0] = ld_shared_f64(zp);
          }
        }
#pragma unroll
        for (int c = 0; c < C; ++c) {
          Vec<XT> x[RG];
#pragma unroll
          for (int r = 0; r < RG; ++r) x[r].load(tile + r * rb + coff[c]);
#pragma unroll
          for (int r = 0; r < RG; ++r) x[r].axpy(zr[r], acc[c]);
        }
      __syncwarp();
      if (lane == 0) mbar_arrive_a(empty0 + 8u * st);
      if constexpr (kF32) {
        rows_since_flush += RG;
        if (rows_since_flush >= kFlushRows) {
          rows_since_flush = 0;
#pragma unroll
          for (int c = 0; c < C; ++c)
#pragma unroll
            for (int v = 0; v < V; ++v) { acc64[c][v] += (double)acc[c][v]; acc[c][v] = (Acc)0; }
        }
      }
    };
    uint32_t st_e = 0, st_g = 0, ph_e = 0, ph_g = 0;
    const int n_my = (int)my_tiles, total_it = n_my + D;
    int it = 0;
    auto generic_iter = [&]() {
      if (it < n_my) {
        eta_phase(st_e, ph_e);
        if (++st_e == (uint32_t)S) { st_e = 0; ph_e ^= 1u; }
      }
      if (it >= D) {
        xz_phase(st_g, ph_g);
        if (++st_g == (uint32_t)S) { st_g = 0; ph_g ^= 1u; }
      }
      ++it;
    };
    constexpr bool kUnrollRing = (C == 1);   // wider per-thread state spills when the body is unrolled 7 times
    if (kUnrollRing && S == 7 && D == 3 && n_my >= 14) {
      // steady state unrolled over the ring (the shape of C3, C4, C5: 7 stages of 32 KB, lag 3): iteration 7k + s runs
      // the eta phase on stage s and the x*z phase on stage (s + 4) mod 7 -- no wrap logic, no loop conditions.
      for (int q = 0; q < 7; ++q) generic_iter();                 // it = 7: st_e = 0, st_g = 4
      uint32_t phb = ph_e;                                        // parity of k = it / 7
      for (; it + 7 <= n_my; it += 7) {
#pragma unroll
        for (int u = 0; u < 7; ++u) {
          eta_phase((uint32_t)u, phb);
          xz_phase((uint32_t)((u + 4) % 7), u >= 3 ? phb : phb ^ 1u);
        }
        phb ^= 1u;
      }
      ph_e = phb; ph_g = phb ^ 1u; st_e = 0; st_g = 4;            // state of the generic loop at it = 7k
    }
    while (it < total_it) generic_iter();
    (void)tiles_end;
#pragma unroll
    for (int c = 0; c < C; ++c) {
      const int col = (c * W + gt) * V;
#pragma unroll
      for (int v = 0; v < V; ++v)
        if (col + v < p) partial[((size_t)cta * G + grp) * p + col + v] = acc64[c][v] + (double)acc[c][v];
    }
  }
}

// ------------------------------------------------------------------------------------------------
// Narrow rows (fewer than 128 16-byte vectors per row, any p: the rows need not be a multiple of 16 bytes --
// config C2, and the shape of the paper's real-data run, N = 1.3e6, p = 141).
// Same pipeline as fused_pass_tma (producer / 16 compute warps / sampler warps, S-stage ring, lag D), but a tile
// holds RT = 32..256 whole rows (RT a multiple of 32, so a tile starts 16-byte aligned and is a whole number of
// 16-byte units) and the thread mappings differ:
//   eta phase   L = 2^k lanes share a row (E = ceil(p / L) <= EMAX elements per lane, beta in registers); the
//               512 compute threads cover 512/L rows per pass; shuffle reduction over the L lanes.
//   xz phase    thread t owns column t mod p for the rows r = t div p (mod NG), NG = floor(512 / p) row groups;
//               the NG accumulators of a column are combined through shared memory at the end (fixed order).
//   sampler     a sampler warp takes a whole tile: lane = row, RT/32 batches.
// The ragged last tile may not be a multiple of 16 bytes: the producer copies the 16-byte units by TMA and the
// last < 16 bytes with plain loads.
// ------------------------------------------------------------------------------------------------
constexpr int kNarrowSamplers = 8;
constexpr int kNarrowThreads = (kComputeWarpsAll + kNarrowSamplers + 1) * 32;   // 800

struct NarrowSmemLayout {
  size_t tiles, eta, z64, z32, red, bars, total;
  __host__ __device__ NarrowSmemLayout(int S, int RT, int p, size_t stage_bytes) {
    tiles = 0;
    eta = tiles + (size_t)S * stage_bytes;
    z64 = eta + (size_t)S * RT * sizeof(double);
    z32 = z64 + (size_t)S * RT * sizeof(double);
    red = (z32 + (size_t)S * RT * sizeof(float) + 15) & ~(size_t)15;
    bars = red + (size_t)kComputeThreadsAll * sizeof(double);
    total = bars + (size_t)4 * S * sizeof(uint64_t);
    (void)p;
  }
};

// A stage is RT rows plus 1 KB that TMA never writes and that stays zero: the eta phase reads up to EMAX L - p
// elements past the end of a row (times beta = 0), which for the last row of a tile lands in this pad.
__host__ __device__ constexpr size_t narrow_stage_bytes(int RT, size_t row_bytes) {
  return (((size_t)RT * row_bytes + 127) & ~(size_t)127) + 1024;
}

template <typename XT> __device__ __forceinline__ XT ld_shared_x(uint32_t a);
template <> __device__ __forceinline__ float ld_shared_x<float>(uint32_t a) { return ld_shared_f32(a); }
template <> __device__ __forceinline__ double ld_shared_x<double>(uint32_t a) { return ld_shared_f64(a); }

template <typename XT, int EMAX, int EM>
__global__ void __launch_bounds__(kNarrowThreads, 1)
fused_pass_narrow(const XT* __restrict__ X, const unsigned char* __restrict__ y, long long N, int p,
                  unsigned long long seed, const double* __restrict__ beta, const Ctl* __restrict__ ctl,
                  double* __restrict__ partial, double* __restrict__ z_out, int S, int D, int RT, int L,
                  long long n_tiles, long long row_off) {
  constexpr bool kF32 = sizeof(XT) == 4;
  using Acc = typename std::conditional<kF32, float, double>::type;
  extern __shared__ __align__(128) unsigned char smem[];
  const size_t row_bytes = (size_t)p * sizeof(XT);
  const size_t stage_bytes = narrow_stage_bytes(RT, row_bytes);
  const NarrowSmemLayout lay(S, RT, p, stage_bytes);
  unsigned char* tiles = smem + lay.tiles;
  double* eta_s = reinterpret_cast<double*>(smem + lay.eta);
  double* z64 = reinterpret_cast<double*>(smem + lay.z64);
  float* z32 = reinterpret_cast<float*>(smem + lay.z32);
  double* red = reinterpret_cast<double*>(smem + lay.red);
  uint64_t* full = reinterpret_cast<uint64_t*>(smem + lay.bars);
  uint64_t* empty = full + S;
  uint64_t* eta_full = empty + S;
  uint64_t* z_full = eta_full + S;

  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const long long cta = blockIdx.x, grid = gridDim.x;
  const long long my_tiles = cta < n_tiles ? (n_tiles - cta + grid - 1) / grid : 0;
  const uint32_t sweep = (uint32_t)(ctl->sweep + 1ull);

  if (tid == 0) {
    for (int s = 0; s < S; ++s) {
      mbar_init(&full[s], 1);
      mbar_init(&empty[s], kComputeWarpsAll);
      mbar_init(&eta_full[s], kComputeWarpsAll);
      mbar_init(&z_full[s], RT / 32);
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  {
    const uint4 zero = make_uint4(0u, 0u, 0u, 0u);
    for (size_t o = (size_t)tid * 16; o < (size_t)S * stage_bytes; o += (size_t)kNarrowThreads * 16)
      *reinterpret_cast<uint4*>(tiles + o) = zero;
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  }
  __syncthreads();

  if (warp == kComputeWarpsAll + kNarrowSamplers) {
    // ===================== producer =====================
    if (lane == 0) {
      int st = 0;
      uint32_t ph = 0;
      const uint64_t pol = l2_evict_first_policy();
      for (long long n = 0; n < my_tiles; ++n) {
        mbar_wait(&empty[st], ph ^ 1u);
        const long long row0 = (cta + n * grid) * RT;
        const long long rows = (N - row0) < RT ? (N - row0) : RT;
        const size_t bytes = (size_t)rows * row_bytes;
        const uint32_t bulk = (uint32_t)(bytes & ~(size_t)15);
        const unsigned char* src = reinterpret_cast<const unsigned char*>(X) + (size_t)row0 * row_bytes;
        unsigned char* dst = tiles + (size_t)st * stage_bytes;
        for (size_t b = bulk; b < bytes; ++b) dst[b] = src[b];       // ragged last tile only: < 16 bytes
        if (bulk) {
          mbar_arrive_expect_tx(&full[st], bulk);
          bulk_g2s(dst, src, bulk, &full[st], pol);
        } else {
          mbar_arrive(&full[st]);
        }
        if (++st == S) { st = 0; ph ^= 1u; }
      }
    }
  } else if (warp >= kComputeWarpsAll) {
    // ===================== sampler warps: batches of 32 rows (lane = row), dealt round-robin =====================
    // Batch gb = tile * BPT + b goes to sampler warp gb mod ns, so the BPT = RT/32 batches of a tile are sampled in
    // parallel by different warps; z_full[stage] counts BPT arrivals.  ns <= S * BPT: a warp then never waits on a
    // stage whose previous use has not completed its eta phase (a parity wait two phases early would pass at once).
    const int sw = warp - kComputeWarpsAll;
    const int BPT = RT / 32;
    const int ns = S * BPT < kNarrowSamplers ? S * BPT : kNarrowSamplers;
    const long long n_batches = my_tiles * BPT;
    if (sw < ns) {
      for (long long gb = sw; gb < n_batches; gb += ns) {
        const long long n = gb / BPT;
        const int b = (int)(gb - n * BPT) * 32;
        const int st = (int)(n % S);
        const uint32_t ph = (uint32_t)((n / S) & 1);
        const long long i = (cta + n * grid) * RT + b + lane;
        const bool valid = i < N;
        const int yi = valid ? (int)y[i] : 1;
        const double u = uniform_a(seed, (unsigned long long)(row_off + (valid ? i : 0)), sweep, TAG_Z);
        const double ystar = 2.0 * (double)yi - 1.0;
        mbar_wait(&eta_full[st], ph);
        const double eta = eta_s[st * RT + b + lane];
        const double wpos = tnpos(ystar * eta, u);
        const double z = valid ? ystar * wpos : 0.0;
        z64[st * RT + b + lane] = z;
        z32[st * RT + b + lane] = (float)z;
        if (valid && z_out != nullptr) z_out[i] = z;
        __syncwarp();
        if (lane == 0) mbar_arrive(&z_full[st]);
      }
    }
  } else {
    // ===================== compute warps =====================
    // eta mapping: lane group of L lanes per row
    const int l = tid & (L - 1), rsub = tid / L, rows_per_pass = kComputeThreadsAll / L;
    double bd[kF32 && EM != 0 ? 1 : EMAX];
    float bf[kF32 && EM != 0 ? EMAX : 1];
#pragma unroll
    for (int e = 0; e < EMAX; ++e) {
      const int j = l + e * L;
      const double bv = (j < p) ? beta[j] : 0.0;
      if constexpr (kF32 && EM != 0) bf[e] = (float)bv; else bd[e] = bv;
    }
    // xz mapping: thread t -> column t mod p, row group t div p
    const int NG = kComputeThreadsAll / p > 0 ? kComputeThreadsAll / p : 1;   // p <= 512 here
    const int xg = tid / p, xj = tid - xg * p;
    const bool xz_on = xg < NG;
    const int RPG = ((RT + NG - 1) / NG + 3) / 4 * 4;                      // rows of a tile per row group, a multiple of 4
    const uint32_t z32a = smem_u32(z32), z64a = smem_u32(z64);
    double acc64 = 0.0;
    Acc acc = (Acc)0;
    const uint32_t rb = (uint32_t)row_bytes, sb = (uint32_t)stage_bytes;
    const uint32_t tiles0 = smem_u32(tiles);
    const uint32_t full0 = smem_u32(full), empty0 = smem_u32(empty), etaf0 = smem_u32(eta_full), zf0 = smem_u32(z_full);
    uint32_t st_e = 0, st_g = 0, ph_e = 0, ph_g = 0;
    int rows_since_flush = 0;
    const int n_my = (int)my_tiles, total_it = n_my + D;
    for (int it = 0; it < total_it; ++it) {
      if (it < n_my) {
        mbar_wait_a(full0 + 8u * st_e, ph_e);
        const uint32_t tile = tiles0 + st_e * sb;
        for (int r = rsub; r < RT; r += rows_per_pass) {
          const uint32_t xa = tile + (uint32_t)r * rb + (uint32_t)l * (uint32_t)sizeof(XT);
          double s;
          if constexpr (kF32 && EM != 0) {
            float c = 0.f;
#pragma unroll
            for (int e = 0; e < EMAX; ++e) c = fmaf(ld_shared_f32(xa + (uint32_t)(e * L) * 4u), bf[e], c);   // past p: beta = 0
#pragma unroll
            for (int off = 16; off >= 1; off >>= 1)
              if (off < L) c += __shfl_xor_sync(0xffffffffu, c, off);       // L is uniform: no divergence
            s = (double)c;
          } else {
            s = 0.0;
#pragma unroll
            for (int e = 0; e < EMAX; ++e) s = fma((double)ld_shared_x<XT>(xa + (uint32_t)(e * L) * (uint32_t)sizeof(XT)), bd[e], s);
#pragma unroll
            for (int off = 16; off >= 1; off >>= 1)
              if (off < L) s += __shfl_xor_sync(0xffffffffu, s, off);
          }
          if (l == 0) eta_s[st_e * RT + r] = s;
        }
        __syncwarp();
        if (lane == 0) mbar_arrive_a(etaf0 + 8u * st_e);
        if (++st_e == (uint32_t)S) { st_e = 0; ph_e ^= 1u; }
      }
      if (it >= D) {
        mbar_wait_a(zf0 + 8u * st_g, ph_g);
        if (xz_on) {
          // rows [xg RPG, (xg+1) RPG) of the tile, four at a time (z as one 16-byte / two 16-byte loads)
          const uint32_t xa = tiles0 + st_g * sb + (uint32_t)xj * (uint32_t)sizeof(XT);
          const int r_hi = (xg + 1) * RPG < RT ? (xg + 1) * RPG : RT;
          if constexpr (kF32) {
            const uint32_t za = z32a + (uint32_t)(st_g * RT) * 4u;
            for (int r = xg * RPG; r < r_hi; r += 4) {
              const float4 z4 = ld_shared_f32x4(za + (uint32_t)r * 4u);
              const uint32_t x0 = xa + (uint32_t)r * rb;
              const float a0 = ld_shared_f32(x0), a1 = ld_shared_f32(x0 + rb), a2 = ld_shared_f32(x0 + 2u * rb), a3 = ld_shared_f32(x0 + 3u * rb);
              acc = fmaf(a0, z4.x, acc); acc = fmaf(a1, z4.y, acc); acc = fmaf(a2, z4.z, acc); acc = fmaf(a3, z4.w, acc);
            }
          } else {
            const uint32_t za = z64a + (uint32_t)(st_g * RT) * 8u;
            for (int r = xg * RPG; r < r_hi; r += 4) {
              const double2 za01 = ld_shared_f64x2(za + (uint32_t)r * 8u), za23 = ld_shared_f64x2(za + (uint32_t)r * 8u + 16u);
              const uint32_t x0 = xa + (uint32_t)r * rb;
              const double a0 = ld_shared_f64(x0), a1 = ld_shared_f64(x0 + rb), a2 = ld_shared_f64(x0 + 2u * rb), a3 = ld_shared_f64(x0 + 3u * rb);
              acc = fma(a0, za01.x, acc); acc = fma(a1, za01.y, acc); acc = fma(a2, za23.x, acc); acc = fma(a3, za23.y, acc);
            }
          }
        }
        __syncwarp();
        if (lane == 0) mbar_arrive_a(empty0 + 8u * st_g);
        if (++st_g == (uint32_t)S) { st_g = 0; ph_g ^= 1u; }
        if constexpr (kF32) {
          rows_since_flush += RPG;
          if (rows_since_flush >= kFlushRows) { rows_since_flush = 0; acc64 += (double)acc; acc = 0.f; }
        }
      }
    }
    // combine the NG row groups of every column in fixed order (named barrier over the 16 compute warps)
    red[tid] = acc64 + (double)acc;
    asm volatile("bar.sync 1, %0;" ::"n"(kComputeThreadsAll) : "memory");
    if (tid < p) {
      double s = 0.0;
      for (int g = 0; g < NG; ++g) s += red[g * p + tid];
      partial[(size_t)cta * p + tid] = s;
    }
  }
}

// ------------------------------------------------------------------------------------------------
// Generic kernel: any p / alignment.  256-row tiles; phase 1 thread-per-row, phase 2 thread-per-column.
// ------------------------------------------------------------------------------------------------
constexpr int kGenThreads = 256;
constexpr int kGenMaxC = 16;

template <typename XT>
__global__ void __launch_bounds__(kGenThreads)
fused_pass_generic(const XT* __restrict__ X, const unsigned char* __restrict__ y, long long N, int p,
                   unsigned long long seed, const double* __restrict__ beta, const Ctl* __restrict__ ctl,
                   double* __restrict__ partial, double* __restrict__ z_out, int csg /*pow2 column slots*/, long long row_off) {
  __shared__ double z_s[kGenThreads];
  __shared__ double red[kGenThreads];
  const int tid = threadIdx.x;
  const uint32_t sweep = (uint32_t)(ctl->sweep + 1ull);
  const int rg_count = kGenThreads / csg, rg = tid / csg, cs = tid % csg;
  const int C = (p + csg - 1) / csg;                 // column chunks per thread (1 when csg < 256)
  const bool in_regs = C <= kGenMaxC;
  double acc[kGenMaxC];
#pragma unroll
  for (int c = 0; c < kGenMaxC; ++c) acc[c] = 0.0;
  double* my_partial = partial + (size_t)blockIdx.x * p;
  if (!in_regs)
    for (int j = tid; j < p; j += kGenThreads) my_partial[j] = 0.0;
  const long long n_tiles = (N + kGenThreads - 1) / kGenThreads;
  for (long long t = blockIdx.x; t < n_tiles; t += gridDim.x) {
    const long long row0 = t * kGenThreads;
    const long long i = row0 + tid;
    double z = 0.0;
    if (i < N) {
      const XT* xr = X + (size_t)i * p;
      double eta = 0.0;
      for (int j = 0; j < p; ++j) eta = fma((double)xr[j], beta[j], eta);
      const double ystar = 2.0 * (double)y[i] - 1.0;
      const double u = uniform_a(seed, (unsigned long long)(row_off + i), sweep, TAG_Z);
      z = ystar * tnpos(ystar * eta, u);
      if (z_out != nullptr) z_out[i] = z;
    }
    __syncthreads();     // previous tile's phase 2 is done with z_s
    z_s[tid] = z;
    __syncthreads();
    const int nrows = (N - row0) < kGenThreads ? (int)(N - row0) : kGenThreads;
    if (in_regs) {
#pragma unroll
      for (int c = 0; c < kGenMaxC; ++c) {
        const int j = c * csg + cs;
        if (c < C && j < p) {
          double a = 0.0;
          for (int r = rg; r < nrows; r += rg_count) a = fma((double)X[(size_t)(row0 + r) * p + j], z_s[r], a);
          acc[c] += a;
        }
      }
    } else {
      for (int j = tid; j < p; j += kGenThreads) {
        double a = 0.0;
        for (int r = 0; r < nrows; ++r) a = fma((double)X[(size_t)(row0 + r) * p + j], z_s[r], a);
        my_partial[j] += a;
      }
    }
  }
  if (in_regs) {
    if (rg_count == 1) {
#pragma unroll
      for (int c = 0; c < kGenMaxC; ++c) {
        const int j = c * csg + cs;
        if (c < C && j < p) my_partial[j] = acc[c];
      }
    } else {   // C == 1: combine the row groups in fixed order
      __syncthreads();
      red[tid] = acc[0];
      __syncthreads();
      if (rg == 0 && cs < p) {
        double s = 0.0;
        for (int q = 0; q < rg_count; ++q) s += red[q * csg + cs];
        my_partial[cs] = s;
      }
    }
  }
}

// b: g_j = sum_c partial[c][j] in a fixed order (no float atomics): 32 columns per CTA; thread (x, y)
// adds rows y, y+32, ... of column x, then row 0 adds the 32 sub-sums in ascending y.
__global__ void __launch_bounds__(1024)
reduce_partials_kernel(const double* __restrict__ partial, int n_part, int p, double* __restrict__ g) {
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");   // the first product of d2 may start its prologue
  __shared__ double red[32][33];
  const int x = threadIdx.x, y = threadIdx.y;
  const int j = blockIdx.x * 32 + x;
  double s = 0.0;
  if (j < p)
    for (int c = y; c < n_part; c += 32) s += partial[(size_t)c * p + j];
  red[y][x] = s;
  __syncthreads();
  if (y == 0 && j < p) {
    double t = 0.0;
#pragma unroll
    for (int q = 0; q < 32; ++q) t += red[q][x];
    g[j] = t;
  }
}

// ------------------------------------------------------------------------------------------------
// Host side: variant selection and launch
// ------------------------------------------------------------------------------------------------

// Tile shapes of the TMA kernel: W threads across a row, C 16-byte chunks per thread, RT rows per tile
// (a stage is ~32 KB).  vec = 16-byte vectors per row.
struct TmaShape { int RT, C, W; };
static bool tma_shape(int vec, int prefer_w, TmaShape* out) {
  const TmaShape shapes[] = {{8, 1, 256}, {4, 2, 256}, {4, 1, 512}, {2, 2, 512}, {1, 4, 512}, {1, 8, 512}};
  for (const TmaShape& sh : shapes) {
    if (vec > sh.C * sh.W) continue;
    if (sh.W != (prefer_w ? prefer_w : 512) && vec <= 512 && vec > 256) continue;   // p in (256 V, 512 V]: two candidates, 16 warps across the row by default
    *out = sh;
    return true;
  }
  return false;
}

static bool narrow_plan(int dtype, long long N, int p, int num_sms, const void* X, const Options& opt, FusedPlan* pl) {
  const size_t elem = dtype == kF32 ? 4 : 8;
  const size_t row_bytes = (size_t)p * elem;
  // tiny problems (C1) are launch-bound: the generic kernel has no 224 KB ring to set up
  if ((reinterpret_cast<uintptr_t>(X) & 15) != 0 || p > kComputeThreadsAll - 1 || (size_t)N * row_bytes < ((size_t)2 << 20)) return false;
  int L = 1;
  while (L < 32 && (p + L - 1) / L > 4) L <<= 1;
  const int E = (p + L - 1) / L;
  if (E > 16) return false;
  int RT = (int)(56000 / row_bytes) / 32 * 32;      // ~50 KB stages (4 fit): the per-tile overhead is what limits narrow rows
  RT = RT < 32 ? 32 : RT > 256 ? 256 : RT;
  if (opt.narrow_rt > 0) RT = opt.narrow_rt / 32 * 32;
  const size_t stage_bytes = narrow_stage_bytes(RT, row_bytes);
  const size_t budget = 227 * 1024;
  int S = opt_or(opt.fused_stages, 0);
  if (S <= 0) {
    S = 8;
    while (S > 2 && NarrowSmemLayout(S, RT, p, stage_bytes).total > budget) --S;
  }
  if (S < 3 || NarrowSmemLayout(S, RT, p, stage_bytes).total > budget) return false;
  int D = opt_or(opt.fused_lag, 0);
  if (D <= 0) D = (S - 1) / 2 > 2 ? (S - 1) / 2 : 2;
  if (D > S - 2) D = S - 2;
  if (D < 1) D = 1;
  pl->variant = 2;
  pl->rows_per_tile = RT; pl->chunks = E <= 4 ? 4 : E <= 6 ? 6 : E <= 8 ? 8 : E <= 12 ? 12 : 16; pl->width = L; pl->stages = S; pl->lag = D;
  pl->groups = 1;
  int em = dtype == kF32 ? opt_or(opt.fused_eta, 2) : 0;
  pl->eta_mode = (em == 0) ? 0 : 2;
  pl->n_tiles = (N + RT - 1) / RT;
  int grid = opt.fused_grid > 0 ? opt.fused_grid : num_sms;
  if ((long long)grid > pl->n_tiles) grid = (int)pl->n_tiles;
  pl->grid = grid; pl->block = kNarrowThreads;
  pl->smem = NarrowSmemLayout(S, RT, p, stage_bytes).total;
  return true;
}

template <typename XT, int EMAX, int EM>
static cudaError_t launch_narrow(const FusedPlan& pl, const void* X, const unsigned char* y, long long N, int p,
                                 unsigned long long seed, const double* beta, const Ctl* ctl, double* partial,
                                 double* z_out, cudaStream_t st) {
  auto kern = fused_pass_narrow<XT, EMAX, EM>;
  // prepare-only call (hsp_create, once per chain, outside stream capture): the attribute is per DEVICE, so it is
  // set for the current device every time a chain is created, not once per process
  if (N < 0) return cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024);
  kern<<<pl.grid, pl.block, pl.smem, st>>>(static_cast<const XT*>(X), y, N, p, seed, beta, ctl, partial, z_out,
                                          pl.stages, pl.lag, pl.rows_per_tile, pl.width, pl.n_tiles, pl.row_offset);
  return cudaGetLastError();
}

template <typename XT>
static cudaError_t dispatch_narrow(const FusedPlan& pl, const void* X, const unsigned char* y, long long N, int p,
                                   unsigned long long seed, const double* beta, const Ctl* ctl, double* partial,
                                   double* z_out, cudaStream_t st) {
#define HSP_NARROW_ARGS pl, X, y, N, p, seed, beta, ctl, partial, z_out, st
#define HSP_NARROW_CASE(E_)                                                                   \
  if (pl.chunks == E_) {                                                                      \
    if constexpr (sizeof(XT) == 4) {                                                          \
      if (pl.eta_mode == 2) return launch_narrow<XT, E_, 2>(HSP_NARROW_ARGS);                 \
    }                                                                                         \
    return launch_narrow<XT, E_, 0>(HSP_NARROW_ARGS);                                         \
  }
  HSP_NARROW_CASE(4)
  HSP_NARROW_CASE(6)
  HSP_NARROW_CASE(8)
  HSP_NARROW_CASE(12)
  HSP_NARROW_CASE(16)
#undef HSP_NARROW_CASE
#undef HSP_NARROW_ARGS
  return cudaErrorInvalidValue;
}

FusedPlan fused_plan(int dtype, long long N, int p, int num_sms, const void* X, const Options& opt) {
  FusedPlan pl{};
  const size_t elem = dtype == kF32 ? 4 : 8;
  const size_t row_bytes = (size_t)p * elem;
  const bool aligned = (row_bytes % 16 == 0) && ((reinterpret_cast<uintptr_t>(X) & 15) == 0);
  const int vec = (int)(row_bytes / 16);
  const bool wide = vec >= 128;
  const int force = opt.fused_variant;
  TmaShape sh{};
  if (aligned && (wide || force == 1) && force != 0 && tma_shape(vec, opt_or(opt.fused_w, 0), &sh)) {
    const int RT = sh.RT, WPR = sh.W / 32;
    const size_t stage_bytes = ((size_t)RT * row_bytes + 127) & ~(size_t)127;
    const size_t budget = 227 * 1024;
    int S = opt_or(opt.fused_stages, 0);
    if (S <= 0) {
      S = 12;
      while (S > 2 && TmaSmemLayout(S, RT, WPR, stage_bytes).total > budget) --S;
    }
    if (S >= 3 && TmaSmemLayout(S, RT, WPR, stage_bytes).total <= budget) {
      int D = opt_or(opt.fused_lag, 0);
      if (D <= 0) D = (S - 1) / 2;
      if (D > S - 2) D = S - 2;
      if (D < 1) D = 1;
      pl.variant = 1;
      pl.rows_per_tile = RT; pl.chunks = sh.C; pl.width = sh.W; pl.stages = S; pl.lag = D;
      pl.groups = kComputeThreadsAll / sh.W;
      int em = dtype == kF32 ? opt_or(opt.fused_eta, 2) : 0;
      pl.eta_mode = (em == 0) ? 0 : 2;
      pl.n_tiles = (N + RT - 1) / RT;
      int grid = opt.fused_grid > 0 ? opt.fused_grid : num_sms;
      if ((long long)grid > pl.n_tiles) grid = (int)pl.n_tiles;
      pl.grid = grid; pl.block = kTmaThreads;
      pl.smem = TmaSmemLayout(S, RT, WPR, stage_bytes).total;
      return pl;
    }
  }
  if (force != 0 && opt_or(opt.fused_narrow, 1) && narrow_plan(dtype, N, p, num_sms, X, opt, &pl)) return pl;
  pl = FusedPlan{};
  pl.variant = 0;
  pl.n_tiles = (N + kGenThreads - 1) / kGenThreads;
  long long grid = (long long)num_sms * 4;
  if (grid > pl.n_tiles) grid = pl.n_tiles;
  pl.grid = (int)grid; pl.block = kGenThreads; pl.smem = 0;
  pl.rows_per_tile = kGenThreads; pl.chunks = 0; pl.stages = 0; pl.lag = 0; pl.groups = 1;
  return pl;
}

template <typename XT, int RT, int C, int W, int EM>
static cudaError_t launch_tma(const FusedPlan& pl, const void* X, const unsigned char* y, long long N, int p,
                              unsigned long long seed, const double* beta, const Ctl* ctl, double* partial,
                              double* z_out, cudaStream_t st) {
  auto kern = fused_pass_tma<XT, RT, C, W, EM>;
  // prepare-only call (hsp_create, once per chain, outside stream capture): per-device attribute, see launch_narrow
  if (N < 0) return cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024);
  kern<<<pl.grid, pl.block, pl.smem, st>>>(static_cast<const XT*>(X), y, N, p, seed, beta, ctl, partial, z_out,
                                          pl.stages, pl.lag, pl.n_tiles, pl.row_offset);
  return cudaGetLastError();
}

template <typename XT>
static cudaError_t dispatch_tma(const FusedPlan& pl, const void* X, const unsigned char* y, long long N, int p,
                                unsigned long long seed, const double* beta, const Ctl* ctl, double* partial,
                                double* z_out, cudaStream_t st) {
#define HSP_TMA_ARGS pl, X, y, N, p, seed, beta, ctl, partial, z_out, st
#define HSP_TMA_CASE(RT_, C_, W_)                                                                  \
  if (pl.rows_per_tile == RT_ && pl.chunks == C_ && pl.width == W_) {                              \
    if constexpr (sizeof(XT) == 4) {                                                               \
      if (pl.eta_mode == 2) return launch_tma<XT, RT_, C_, W_, 2>(HSP_TMA_ARGS);                   \
    }                                                                                              \
    return launch_tma<XT, RT_, C_, W_, 0>(HSP_TMA_ARGS);                                           \
  }
  HSP_TMA_CASE(8, 1, 256)
  HSP_TMA_CASE(4, 2, 256)
  HSP_TMA_CASE(4, 1, 512)
  HSP_TMA_CASE(2, 2, 512)
  HSP_TMA_CASE(1, 4, 512)
  HSP_TMA_CASE(1, 8, 512)
#undef HSP_TMA_CASE
#undef HSP_TMA_ARGS
  return cudaErrorInvalidValue;
}

cudaError_t fused_pass_launch(const FusedPlan& pl, const void* X, int dtype, const unsigned char* y, long long N,
                              int p, unsigned long long seed, const double* beta, const Ctl* ctl, double* partial,
                              double* z_out, cudaStream_t st) {
  if (pl.variant == 0 && N < 0) return cudaSuccess;
  if (pl.variant == 2) {
    return dtype == kF32 ? dispatch_narrow<float>(pl, X, y, N, p, seed, beta, ctl, partial, z_out, st)
                         : dispatch_narrow<double>(pl, X, y, N, p, seed, beta, ctl, partial, z_out, st);
  }
  if (pl.variant == 1) {
    return dtype == kF32 ? dispatch_tma<float>(pl, X, y, N, p, seed, beta, ctl, partial, z_out, st)
                         : dispatch_tma<double>(pl, X, y, N, p, seed, beta, ctl, partial, z_out, st);
  }
  int csg = 1;
  while (csg < p && csg < kGenThreads) csg <<= 1;
  if (dtype == kF32)
    fused_pass_generic<float><<<pl.grid, pl.block, 0, st>>>(static_cast<const float*>(X), y, N, p, seed, beta, ctl,
                                                            partial, z_out, csg, pl.row_offset);
  else
    fused_pass_generic<double><<<pl.grid, pl.block, 0, st>>>(static_cast<const double*>(X), y, N, p, seed, beta, ctl,
                                                             partial, z_out, csg, pl.row_offset);
  return cudaGetLastError();
}

cudaError_t reduce_partials_launch(const double* partial, int n_part, int p, double* g, cudaStream_t st) {
  reduce_partials_kernel<<<(p + 31) / 32, dim3(32, 32), 0, st>>>(partial, n_part, p, g);
  return cudaGetLastError();
}

}  // namespace hsp
