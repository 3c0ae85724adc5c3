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
// Packed fp32 pairs (sm_100: fma.rn.f32x2 -> SASS FFMA2, two fp32 FMAs per issued instruction; each half is an
// ordinary IEEE fp32 FMA).  Halves the FMA instruction count of the fp32-X phases.
__device__ __forceinline__ unsigned long long f2_pack(float a, float b) {
  unsigned long long r;
  asm("mov.b64 %0, {%1,%2};" : "=l"(r) : "f"(a), "f"(b));
  return r;
}
__device__ __forceinline__ void f2_unpack(unsigned long long v, float& a, float& b) {
  asm("mov.b64 {%0,%1}, %2;" : "=f"(a), "=f"(b) : "l"(v));
}
__device__ __forceinline__ unsigned long long f2_fma(unsigned long long a, unsigned long long b, unsigned long long c) {
  unsigned long long d;
  asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c));
  return d;
}
__device__ __forceinline__ void ld_shared_b64x2(uint32_t a, unsigned long long& lo, unsigned long long& hi) {
  asm volatile("ld.shared.v2.b64 {%0,%1}, [%2];" : "=l"(lo), "=l"(hi) : "r"(a));
}

template <typename XT> struct Vec;
template <> struct Vec<float> {
  static constexpr int V = 4;
  using Acc = float;
  using Pair = unsigned long long;          // accumulators of a 16-byte vector: two packed fp32 pairs
  unsigned long long lo, hi;                // (x0, x1), (x2, x3)
  __device__ __forceinline__ void load(uint32_t smem_addr) { ld_shared_b64x2(smem_addr, lo, hi); }
  __device__ __forceinline__ double dot(const double* b) const {
    float x0, x1, x2, x3;
    f2_unpack(lo, x0, x1); f2_unpack(hi, x2, x3);
    double s = (double)x0 * b[0];
    s = fma((double)x1, b[1], s);
    s = fma((double)x2, b[2], s);
    s = fma((double)x3, b[3], s);
    return s;
  }
  // fp32 (eta mode 2): part += x .* b on packed pairs; the two halves are two chains of 2 FMAs per vector, added at
  // the end of the row's chunks -- at most ~2C+1 roundings of 2^-24 relative to the running partial
  __device__ __forceinline__ void dotf2(const Pair* b2, Pair& part) const {
    part = f2_fma(lo, b2[0], part);
    part = f2_fma(hi, b2[1], part);
  }
  __device__ __forceinline__ void axpy(float z, Pair* acc) const {
    const Pair z2 = f2_pack(z, z);
    acc[0] = f2_fma(lo, z2, acc[0]);
    acc[1] = f2_fma(hi, z2, acc[1]);
  }
  static __device__ __forceinline__ Pair zero() { return 0ull; }
  static __device__ __forceinline__ void flush(Pair* acc, double* acc64) {   // acc64[0..3] += acc; acc = 0
    float a, b;
    f2_unpack(acc[0], a, b); acc64[0] += (double)a; acc64[1] += (double)b;
    f2_unpack(acc[1], a, b); acc64[2] += (double)a; acc64[3] += (double)b;
    acc[0] = acc[1] = 0ull;
  }
};
template <> struct Vec<double> {
  static constexpr int V = 2;
  using Acc = double;
  using Pair = double;
  double2 v;
  __device__ __forceinline__ void load(uint32_t smem_addr) { v = ld_shared_f64x2(smem_addr); }
  __device__ __forceinline__ double dot(const double* b) const { return fma(v.y, b[1], v.x * b[0]); }
  __device__ __forceinline__ void dotf2(const Pair*, Pair&) const {}   // never used: fp64 X is always eta mode 0
  __device__ __forceinline__ void axpy(double z, Pair* acc) const {
    acc[0] = fma(v.x, z, acc[0]);
    acc[1] = fma(v.y, z, acc[1]);
  }
  static __device__ __forceinline__ Pair zero() { return 0.0; }
  static __device__ __forceinline__ void flush(Pair* acc, double* acc64) {
    acc64[0] += acc[0]; acc64[1] += acc[1];
    acc[0] = acc[1] = 0.0;
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
    using Pair = typename Vec<XT>::Pair;
    double breg[EM == 0 ? C : 1][V];
    Pair breg2[EM == 0 ? 1 : C][2];               // beta as packed fp32 pairs (eta mode 2)
    double acc64[C][V];
    Pair acc[C][2];
    uint32_t coff[C];
#pragma unroll
    for (int c = 0; c < C; ++c) {
      const int col = (c * W + gt) * V;
      coff[c] = (col < p) ? (uint32_t)(col * sizeof(XT)) : 0u;
      double bv[V];
#pragma unroll
      for (int v = 0; v < V; ++v) {
        bv[v] = (col + v < p) ? beta[col + v] : 0.0;
        acc64[c][v] = 0.0;
      }
      if constexpr (EM == 0) {
#pragma unroll
        for (int v = 0; v < V; ++v) breg[c][v] = bv[v];
      } else if constexpr (kF32) {
        breg2[c][0] = f2_pack((float)bv[0], (float)bv[1]);
        breg2[c][1] = f2_pack((float)bv[2], (float)bv[3]);
      }
      acc[c][0] = acc[c][1] = Vec<XT>::zero();
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
          if constexpr (kF32) {
            Pair part2[RG];
#pragma unroll
            for (int r = 0; r < RG; ++r) part2[r] = 0ull;
#pragma unroll
            for (int c = 0; c < C; ++c) {
              Vec<XT> x[RG];
#pragma unroll
              for (int r = 0; r < RG; ++r) x[r].load(tile + r * rb + coff[c]);
#pragma unroll
              for (int r = 0; r < RG; ++r) x[r].dotf2(breg2[c], part2[r]);
            }
#pragma unroll
            for (int r = 0; r < RG; ++r) {
              float a, b;
              f2_unpack(part2[r], a, b);
              part[r] = a + b;
            }
          } else {
#pragma unroll
            for (int r = 0; r < RG; ++r) part[r] = 0.f;
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
          for (int c = 0; c < C; ++c) Vec<XT>::flush(acc[c], acc64[c]);
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
      Vec<XT>::flush(acc[c], acc64[c]);
#pragma unroll
      for (int v = 0; v < V; ++v)
        if (col + v < p) partial[((size_t)cta * G + grp) * p + col + v] = acc64[c][v];
    }
  }
}

// ------------------------------------------------------------------------------------------------
// Narrow rows (fewer than 128 16-byte vectors per row, any p: the rows need not be a multiple of 16 bytes --
// config C2, and the shape of the paper's real-data run, N = 1.3e6, p = 141).
// A tile holds RT = 32..256 whole rows (RT a multiple of 32, so a tile starts 128-byte aligned and the batches of 32
// rows a z-warp takes never straddle a tile); one cp.async.bulk per tile, S-stage ring.  Warp roles:
//   producer   1 thread: streams the tiles (the < 16 trailing bytes of a ragged last tile by plain loads).
//   z-warps    8 warps, batches of 32 rows dealt round-robin (lane = row): eta_i = x_i . beta by a THREAD-PER-ROW dot
//              product straight from the tile in shared memory (beta staged once in shared memory, read as 16-byte
//              broadcasts), then the Philox uniform and TNpos -> z to shared memory.  No shuffles, no eta round trip.
//              Bank conflicts: lanes read the same column of 32 consecutive rows, i.e. addresses row_bytes apart.  With
//              U = the largest power of two <= 16 that divides row_bytes, the row is read in U-byte units; row_bytes / U
//              is odd for U < 16, which makes the 4-, 8-byte accesses of a warp conflict-free; for U = 16 and
//              q = row_bytes / 16 even, lane r of each quarter-warp starts (r >> shift) units later (and wraps), which
//              spreads the 8 lanes over the 8 16-byte banks again (shift = log2(8 / gcd(q, 8))).
//   x*z warps  16 warps: thread t owns column t mod p for the rows t div p (mod NG), NG = floor(512 / p); conflict-free
//              4-/8-byte loads along the row; the NG accumulators of a column are combined through shared memory at
//              the end (fixed order).  fp32 X: fp32 FMA chains, flushed into fp64 every >= 16 rows.
// Per element of X this is ~2.3 + ~2.6 issued thread-instructions (the previous lane-group/shuffle design: ~7), which is
// what takes the kernel from issue-bound to HBM-bound at p ~ 100-150.
// ------------------------------------------------------------------------------------------------
constexpr int kNarrowZWarps = 8;
constexpr int kNarrowThreads = (kComputeWarpsAll + kNarrowZWarps + 1) * 32;   // 800
constexpr int kNarrowMaxP = kComputeThreadsAll - 1;                          // 511: one x*z thread per column
constexpr size_t kNarrowBetaBytes = (size_t)(kComputeThreadsAll + 16) * sizeof(double);

struct NarrowSmemLayout {
  size_t tiles, beta, z64, z32, red, bars, total;
  __host__ __device__ NarrowSmemLayout(int S, int RT, size_t stage_bytes) {
    tiles = 0;
    beta = tiles + (size_t)S * stage_bytes;
    z64 = beta + kNarrowBetaBytes;
    z32 = z64 + (size_t)S * RT * sizeof(double);
    red = (z32 + (size_t)S * RT * sizeof(float) + 15) & ~(size_t)15;
    bars = red + (size_t)kComputeThreadsAll * sizeof(double);
    total = bars + (size_t)3 * S * sizeof(uint64_t);
  }
};

// A stage is RT rows plus 1 KB that TMA never writes and that stays zero: the last 16-byte step of a row's dot product
// may read up to 12 bytes past the end of the row (times beta = 0), which for the last row of a tile lands in this pad.
__host__ __device__ constexpr size_t narrow_stage_bytes(int RT, size_t row_bytes) {
  return (((size_t)RT * row_bytes + 127) & ~(size_t)127) + 1024;
}

template <typename XT> __device__ __forceinline__ XT ld_shared_x(uint32_t a);
template <> __device__ __forceinline__ float ld_shared_x<float>(uint32_t a) { return ld_shared_f32(a); }
template <> __device__ __forceinline__ double ld_shared_x<double>(uint32_t a) { return ld_shared_f64(a); }

// 16 bytes of a row, read in U-byte units (U = 4, 8, 16)
template <int U> __device__ __forceinline__ float4 ld_step_f32(uint32_t a) {
  if constexpr (U == 16) return ld_shared_f32x4(a);
  else if constexpr (U == 8) {
    const float2 lo = ld_shared_f32x2(a), hi = ld_shared_f32x2(a + 8);
    return make_float4(lo.x, lo.y, hi.x, hi.y);
  } else return make_float4(ld_shared_f32(a), ld_shared_f32(a + 4), ld_shared_f32(a + 8), ld_shared_f32(a + 12));
}
template <int U> __device__ __forceinline__ double2 ld_step_f64(uint32_t a) {
  if constexpr (U == 16) return ld_shared_f64x2(a);
  else return make_double2(ld_shared_f64(a), ld_shared_f64(a + 8));
}

// eta of one row: sum over n_steps 16-byte steps of the row at shared address xrow; beta0: beta in shared memory in
// the accumulation type (float for fp32 X with EM != 0, else double), zero beyond p.  delta: start offset (in steps) of
// this lane for U = 16 (see above), 0 otherwise.
template <typename XT, int U, int EM>
__device__ __forceinline__ double narrow_row_dot(uint32_t xrow, uint32_t beta0, int n_steps, int delta) {
  constexpr bool kF32 = sizeof(XT) == 4;
  auto rot = [&](int c) {
    if constexpr (U == 16) { c += delta; c = c >= n_steps ? c - n_steps : c; }
    return c;
  };
  if constexpr (kF32 && EM != 0) {
    // fp32 chains of <= 16 FMAs per accumulator (4 accumulators = the 4 elements of a step, as two packed pairs:
    // FFMA2), flushed into fp64
    double eta = 0.0;
    for (int c0 = 0; c0 < n_steps; c0 += 16) {
      const int c1 = c0 + 16 < n_steps ? c0 + 16 : n_steps;
      unsigned long long a01 = 0ull, a23 = 0ull;
#pragma unroll 4
      for (int c = c0; c < c1; ++c) {
        const uint32_t off = (uint32_t)rot(c) * 16u;
        unsigned long long b01, b23, x01, x23;
        ld_shared_b64x2(beta0 + off, b01, b23);
        if constexpr (U == 16) ld_shared_b64x2(xrow + off, x01, x23);
        else {
          const float4 x = ld_step_f32<U>(xrow + off);
          x01 = f2_pack(x.x, x.y); x23 = f2_pack(x.z, x.w);
        }
        a01 = f2_fma(x01, b01, a01); a23 = f2_fma(x23, b23, a23);
      }
      float a0, a1, a2, a3;
      f2_unpack(a01, a0, a1); f2_unpack(a23, a2, a3);
      eta += ((double)a0 + (double)a1) + ((double)a2 + (double)a3);
    }
    return eta;
  } else if constexpr (kF32) {
    // exact: every element converted to fp64 (beta: 4 doubles per step)
    double a0 = 0.0, a1 = 0.0, a2 = 0.0, a3 = 0.0;
#pragma unroll 2
    for (int c = 0; c < n_steps; ++c) {
      const uint32_t s = (uint32_t)rot(c);
      const double2 b01 = ld_shared_f64x2(beta0 + s * 32u), b23 = ld_shared_f64x2(beta0 + s * 32u + 16u);
      const float4 x = ld_step_f32<U>(xrow + s * 16u);
      a0 = fma((double)x.x, b01.x, a0); a1 = fma((double)x.y, b01.y, a1);
      a2 = fma((double)x.z, b23.x, a2); a3 = fma((double)x.w, b23.y, a3);
    }
    return (a0 + a1) + (a2 + a3);
  } else {
    // fp64 X: 2 elements per step, two steps per iteration -> 4 independent DFMA chains
    double a0 = 0.0, a1 = 0.0, a2 = 0.0, a3 = 0.0;
    int c = 0;
#pragma unroll 2
    for (; c + 1 < n_steps; c += 2) {
      const uint32_t s0 = (uint32_t)rot(c) * 16u, s1 = (uint32_t)rot(c + 1) * 16u;
      const double2 b0 = ld_shared_f64x2(beta0 + s0), b1 = ld_shared_f64x2(beta0 + s1);
      const double2 x0 = ld_step_f64<U>(xrow + s0), x1 = ld_step_f64<U>(xrow + s1);
      a0 = fma(x0.x, b0.x, a0); a1 = fma(x0.y, b0.y, a1); a2 = fma(x1.x, b1.x, a2); a3 = fma(x1.y, b1.y, a3);
    }
    if (c < n_steps) {
      const uint32_t s0 = (uint32_t)rot(c) * 16u;
      const double2 b0 = ld_shared_f64x2(beta0 + s0);
      const double2 x0 = ld_step_f64<U>(xrow + s0);
      a0 = fma(x0.x, b0.x, a0); a1 = fma(x0.y, b0.y, a1);
    }
    return (a0 + a1) + (a2 + a3);
  }
}

template <typename XT, int U, int EM>
__global__ void __launch_bounds__(kNarrowThreads, 1)
fused_pass_narrow(const XT* __restrict__ X, const unsigned char* __restrict__ y, long long N, int p,
                  unsigned long long seed, const double* __restrict__ beta, const Ctl* __restrict__ ctl,
                  double* __restrict__ partial, double* __restrict__ z_out, int S, int RT, int skew_shift,
                  long long n_tiles, long long row_off) {
  constexpr bool kF32 = sizeof(XT) == 4;
  constexpr bool kFloatAcc = kF32 && EM != 0;
  constexpr int SE = 16 / (int)sizeof(XT);                 // elements per 16-byte step
  extern __shared__ __align__(128) unsigned char smem[];
  const size_t row_bytes = (size_t)p * sizeof(XT);
  const size_t stage_bytes = narrow_stage_bytes(RT, row_bytes);
  const NarrowSmemLayout lay(S, RT, stage_bytes);
  unsigned char* tiles = smem + lay.tiles;
  double* z64 = reinterpret_cast<double*>(smem + lay.z64);
  float* z32 = reinterpret_cast<float*>(smem + lay.z32);
  double* red = reinterpret_cast<double*>(smem + lay.red);
  uint64_t* full = reinterpret_cast<uint64_t*>(smem + lay.bars);
  uint64_t* empty = full + S;
  uint64_t* z_full = empty + S;

  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const long long cta = blockIdx.x, grid = gridDim.x;
  const long long my_tiles = cta < n_tiles ? (n_tiles - cta + grid - 1) / grid : 0;
  const uint32_t sweep = (uint32_t)(ctl->sweep + 1ull);
  const int BPT = RT / 32;
  const int n_steps = (p + SE - 1) / SE;

  if (tid == 0) {
    for (int s = 0; s < S; ++s) {
      mbar_init(&full[s], 1);
      mbar_init(&empty[s], kComputeWarpsAll);
      mbar_init(&z_full[s], BPT);
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  {
    const uint4 zero = make_uint4(0u, 0u, 0u, 0u);
    for (size_t o = (size_t)tid * 16; o < (size_t)S * stage_bytes; o += (size_t)kNarrowThreads * 16)
      *reinterpret_cast<uint4*>(tiles + o) = zero;
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    // beta in the accumulation type of the eta phase, zero beyond p (the last step of a row reads up to SE - 1 past it)
    for (int e = tid; e < n_steps * SE; e += kNarrowThreads) {
      const double bv = e < p ? beta[e] : 0.0;
      if constexpr (kFloatAcc) reinterpret_cast<float*>(smem + lay.beta)[e] = (float)bv;
      else reinterpret_cast<double*>(smem + lay.beta)[e] = bv;
    }
  }
  __syncthreads();

  if (warp == kComputeWarpsAll + kNarrowZWarps) {
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
    // ===================== z-warps: eta (thread per row) -> z, batches of 32 rows dealt round-robin =====================
    // Batch gb = tile * BPT + b goes to z-warp gb mod ns.  ns <= S * BPT: a warp then never waits on a stage whose
    // previous use it has not finished itself (a parity wait two phases early would pass at once).
    const int zw = warp - kComputeWarpsAll;
    const int ns = S * BPT < kNarrowZWarps ? S * BPT : kNarrowZWarps;
    const long long n_batches = my_tiles * BPT;
    if (zw < ns) {
      const uint32_t beta0 = smem_u32(smem + lay.beta);
      const uint32_t tiles0 = smem_u32(tiles), rb = (uint32_t)row_bytes, sb = (uint32_t)stage_bytes;
      const int delta = (U == 16) ? ((lane & 7) >> skew_shift) : 0;
      auto load_y = [&](long long gb) -> int {
        const long long n = gb / BPT;
        const long long i = (cta + n * grid) * RT + (gb - n * BPT) * 32 + lane;
        return (gb < n_batches && i < N) ? (int)y[i] : 1;
      };
      int y_next = load_y(zw);                       // y is prefetched one batch ahead (a lone 1-byte load under a saturated HBM)
      for (long long gb = zw; gb < n_batches; gb += ns) {
        const long long n = gb / BPT;
        const int b = (int)(gb - n * BPT) * 32;
        const int st = (int)(n % S);
        const uint32_t ph = (uint32_t)((n / S) & 1);
        const long long i = (cta + n * grid) * RT + b + lane;
        const bool valid = i < N;
        const int yi = y_next;
        y_next = load_y(gb + ns);
        // the Philox uniform does not depend on eta: computed before waiting for the tile
        const double u = uniform_a(seed, (unsigned long long)(row_off + (valid ? i : 0)), sweep, TAG_Z);
        const double ystar = 2.0 * (double)yi - 1.0;
        mbar_wait(&full[st], ph);
        const double eta = narrow_row_dot<XT, U, EM>(tiles0 + (uint32_t)st * sb + (uint32_t)(b + lane) * rb, beta0, n_steps, delta);
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
    // ===================== x*z warps =====================
    // thread t -> column t mod p, row group t div p
    const int NG = kComputeThreadsAll / p > 0 ? kComputeThreadsAll / p : 1;   // p <= 511 here
    const int xg = tid / p, xj = tid - xg * p;
    const bool xz_on = xg < NG;
    const int RPG = ((RT + NG - 1) / NG + 3) / 4 * 4;                      // rows of a tile per row group, a multiple of 4
    const int r_lo = xg * RPG, r_hi = (xg + 1) * RPG < RT ? (xg + 1) * RPG : RT;
    const uint32_t z32a = smem_u32(z32), z64a = smem_u32(z64);
    double acc64 = 0.0;
    typename std::conditional<kF32, unsigned long long, double>::type acc = 0;   // fp32 X: a packed pair of fp32 chains
    auto acc_value = [&]() -> double {
      if constexpr (kF32) { float a, b; f2_unpack(acc, a, b); return (double)a + (double)b; }
      else return acc;
    };
    const uint32_t rb = (uint32_t)row_bytes, sb = (uint32_t)stage_bytes;
    const uint32_t xcol0 = smem_u32(tiles) + (uint32_t)xj * (uint32_t)sizeof(XT) + (uint32_t)r_lo * rb;
    const uint32_t full0 = smem_u32(full), empty0 = smem_u32(empty), zf0 = smem_u32(z_full);
    uint32_t st = 0, ph = 0;
    int rows_since_flush = 0;
    const int n_my = (int)my_tiles;
    for (int it = 0; it < n_my; ++it) {
      mbar_wait_a(zf0 + 8u * st, ph);
      mbar_wait_a(full0 + 8u * st, ph);          // complete long ago; orders this thread's reads after the bulk copy
      if (xz_on && r_lo < r_hi) {
        uint32_t x0 = xcol0 + st * sb;
        if constexpr (kF32) {
          uint32_t za = z32a + (uint32_t)(st * RT + r_lo) * 4u;
#pragma unroll 2
          for (int r = r_lo; r < r_hi; r += 4) {
            unsigned long long z01, z23;
            ld_shared_b64x2(za, z01, z23);
            const float a0 = ld_shared_f32(x0), a1 = ld_shared_f32(x0 + rb), a2 = ld_shared_f32(x0 + 2u * rb), a3 = ld_shared_f32(x0 + 3u * rb);
            acc = f2_fma(f2_pack(a0, a1), z01, acc);      // even rows in the low half, odd rows in the high half
            acc = f2_fma(f2_pack(a2, a3), z23, acc);
            za += 16u; x0 += 4u * rb;
          }
        } else {
          uint32_t za = z64a + (uint32_t)(st * RT + r_lo) * 8u;
#pragma unroll 2
          for (int r = r_lo; r < r_hi; r += 4) {
            const double2 za01 = ld_shared_f64x2(za), za23 = ld_shared_f64x2(za + 16u);
            const double a0 = ld_shared_f64(x0), a1 = ld_shared_f64(x0 + rb), a2 = ld_shared_f64(x0 + 2u * rb), a3 = ld_shared_f64(x0 + 3u * rb);
            acc = fma(a0, za01.x, acc); acc = fma(a1, za01.y, acc); acc = fma(a2, za23.x, acc); acc = fma(a3, za23.y, acc);
            za += 32u; x0 += 4u * rb;
          }
        }
      }
      __syncwarp();
      if (lane == 0) mbar_arrive_a(empty0 + 8u * st);
      if (++st == (uint32_t)S) { st = 0; ph ^= 1u; }
      if constexpr (kF32) {
        rows_since_flush += RPG;
        if (rows_since_flush >= kFlushRows) { rows_since_flush = 0; acc64 += acc_value(); acc = 0ull; }
      }
    }
    // combine the NG row groups of every column in fixed order (named barrier over the 16 x*z warps)
    red[tid] = acc64 + acc_value();
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
  if ((reinterpret_cast<uintptr_t>(X) & 15) != 0 || p > kNarrowMaxP || (size_t)N * row_bytes < ((size_t)2 << 20)) return false;
  // U: unit of the thread-per-row dot product; skew for rows that are an even number of 16-byte units (see the kernel)
  int U = 16;
  while (row_bytes % (size_t)U) U >>= 1;
  int shift = 3;
  if (U == 16) {
    const size_t q = row_bytes / 16;
    int g = 1;
    while (g < 8 && q % (size_t)(2 * g) == 0) g <<= 1;       // gcd(q, 8)
    shift = g == 1 ? 3 : g == 2 ? 2 : g == 4 ? 1 : 0;
  }
  // ~36 KB stages, five or six in the ring (measured at the R1 shape, 564-byte rows: 64 rows x 5 stages 6.0 TB/s; 32 x 12 and
  // 96 x 3 5.4-5.6 TB/s; 64 x 4 5.3 TB/s)
  int RT = ((int)(36000 / row_bytes) + 16) / 32 * 32;
  RT = RT < 32 ? 32 : RT > 256 ? 256 : RT;
  if (opt.narrow_rt > 0) RT = opt.narrow_rt / 32 * 32;
  if (RT < 32) RT = 32;
  const size_t stage_bytes = narrow_stage_bytes(RT, row_bytes);
  const size_t budget = 227 * 1024;
  int S = opt_or(opt.fused_stages, 0);
  if (S <= 0) {
    S = 12;
    while (S > 2 && NarrowSmemLayout(S, RT, stage_bytes).total > budget) --S;
  }
  if (S < 3 || NarrowSmemLayout(S, RT, stage_bytes).total > budget) return false;
  pl->variant = 2;
  pl->rows_per_tile = RT; pl->chunks = U; pl->width = shift; pl->stages = S; pl->lag = 0;
  pl->groups = 1;
  int em = dtype == kF32 ? opt_or(opt.fused_eta, 2) : 0;
  pl->eta_mode = (em == 0) ? 0 : 2;
  pl->n_tiles = (N + RT - 1) / RT;
  int grid = opt.fused_grid > 0 ? opt.fused_grid : num_sms;
  if ((long long)grid > pl->n_tiles) grid = (int)pl->n_tiles;
  pl->grid = grid; pl->block = kNarrowThreads;
  pl->smem = NarrowSmemLayout(S, RT, stage_bytes).total;
  return true;
}

template <typename XT, int U, int EM>
static cudaError_t launch_narrow(const FusedPlan& pl, const void* X, const unsigned char* y, long long N, int p,
                                 unsigned long long seed, const double* beta, const Ctl* ctl, double* partial,
                                 double* z_out, cudaStream_t st) {
  auto kern = fused_pass_narrow<XT, U, EM>;
  // prepare-only call (hsp_create, once per chain, outside stream capture): the attribute is per DEVICE, so it is
  // set for the current device every time a chain is created, not once per process
  if (N < 0) return cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024);
  kern<<<pl.grid, pl.block, pl.smem, st>>>(static_cast<const XT*>(X), y, N, p, seed, beta, ctl, partial, z_out,
                                          pl.stages, pl.rows_per_tile, pl.width, pl.n_tiles, pl.row_offset);
  return cudaGetLastError();
}

template <typename XT>
static cudaError_t dispatch_narrow(const FusedPlan& pl, const void* X, const unsigned char* y, long long N, int p,
                                   unsigned long long seed, const double* beta, const Ctl* ctl, double* partial,
                                   double* z_out, cudaStream_t st) {
#define HSP_NARROW_ARGS pl, X, y, N, p, seed, beta, ctl, partial, z_out, st
#define HSP_NARROW_CASE(U_)                                                                   \
  if (pl.chunks == U_) {                                                                      \
    if constexpr (sizeof(XT) == 4) {                                                          \
      if (pl.eta_mode == 2) return launch_narrow<XT, U_, 2>(HSP_NARROW_ARGS);                 \
    }                                                                                         \
    return launch_narrow<XT, U_, 0>(HSP_NARROW_ARGS);                                         \
  }
  if constexpr (sizeof(XT) == 4) { HSP_NARROW_CASE(4) }
  HSP_NARROW_CASE(8)
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
