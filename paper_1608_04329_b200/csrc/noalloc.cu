// noalloc.cu -- hsp_xtz_noalloc: rows a1-a3 + b of the hot path (eta = X beta, z ~ TN(eta, 1), g = X^T z; PAPER.md:200,
// 206-208) as ONE stateless entry point that allocates nothing, for callers that cannot call cudaMalloc (code under CUDA
// graph capture, tight serving loops, harnesses that forbid it).  The kernels are the ones of the chain (fused_pass.cu);
// what differs is where their scratch lives: the per-CTA partials of X^T z and the 72-byte control block go into a
// file-scope device array of fixed size instead of buffers allocated at hsp_create.
//
// The array costs kNoAllocBytes of device memory on every GPU that loads libhsp.so, until the process exits.  All calls
// share it: it keeps the last call's contents (everything a call reads is written by that call first: the control
// block and the used part of the partials are cleared by a set-up kernel), and two calls that overlap on the GPU
// (different streams, or different host threads) race on it -- serialise them.
#include <cuda_runtime.h>
#include <algorithm>
#include <cstdint>
#include <mutex>
#include <string>
#include "../../include/hsp.h"
#include "hsp_internal.h"

namespace hsp {

constexpr size_t kNoAllocHeadDoubles = 32;                         // 256 bytes: the control block (Ctl, 72 bytes)
constexpr size_t kNoAllocPartialDoubles = (size_t)1 << 20;         // 8 MiB of partials: (CTAs x row groups) x p doubles
constexpr size_t kNoAllocBytes = (kNoAllocHeadDoubles + kNoAllocPartialDoubles) * sizeof(double);
static_assert(sizeof(Ctl) <= kNoAllocHeadDoubles * sizeof(double), "the control block must fit the head of the scratch array");

// In HOST code this name is a host-side stand-in, not a device address: the address the kernels get comes from
// cudaGetSymbolAddress (scratch_for_current_device below).  Device code may name it directly (noalloc_setup_kernel does).
static __device__ __align__(256) double g_noalloc_scratch[kNoAllocHeadDoubles + kNoAllocPartialDoubles];

// Control block: sweep = k - 1 (the pass draws with counter word c2 = sweep + 1); the rest zero.  Partials: the part this
// call uses starts at zero.
__global__ void __launch_bounds__(256)
noalloc_setup_kernel(unsigned long long sweep_before, size_t n_partial) {
  const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i == 0) {
    Ctl c{};
    c.sweep = sweep_before; c.hist_base = 0; c.tau_inv2 = 1.0; c.xi_inv = 1.0; c.status = 0; c.done = 0;
    c.h_beta = c.h_lambda = c.h_tau = nullptr;
    *reinterpret_cast<Ctl*>(g_noalloc_scratch) = c;
  }
  for (size_t q = i; q < n_partial; q += (size_t)gridDim.x * blockDim.x) g_noalloc_scratch[kNoAllocHeadDoubles + q] = 0.0;
}

constexpr int kMaxDevices = 64;
static std::mutex g_noalloc_mutex;
static double* g_noalloc_ptr[kMaxDevices] = {};

// Device address of the array on the CURRENT device, looked up once per device with that device current.
static cudaError_t scratch_for_current_device(double** out) {
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if (dev < 0 || dev >= kMaxDevices) return cudaErrorInvalidDevice;
  std::lock_guard<std::mutex> lock(g_noalloc_mutex);
  if (g_noalloc_ptr[dev] == nullptr) {
    double* ptr = nullptr;
    e = cudaGetSymbolAddress(reinterpret_cast<void**>(&ptr), g_noalloc_scratch);
    if (e != cudaSuccess) return e;
    g_noalloc_ptr[dev] = ptr;
  }
  *out = g_noalloc_ptr[dev];
  return cudaSuccess;
}

}  // namespace hsp

using namespace hsp;

static thread_local std::string g_noalloc_err;
static int na_fail(int code, const std::string& msg) { g_noalloc_err = msg; return code; }

extern "C" {

const char* hsp_noalloc_last_error(void) { return g_noalloc_err.c_str(); }

long long hsp_noalloc_scratch_bytes(void) { return (long long)kNoAllocBytes; }

int hsp_xtz_noalloc(const void* X, int x_dtype, const unsigned char* y, long long N, int p, unsigned long long seed,
                    long long k, const double* beta, double* g_out, double* z_out, void* stream) {
  if (!X || !y || !beta || !g_out) return na_fail(HSP_EINVAL, "hsp_xtz_noalloc: X, y, beta or g_out is NULL");
  if (x_dtype != HSP_F32 && x_dtype != HSP_F64) return na_fail(HSP_EINVAL, "hsp_xtz_noalloc: x_dtype must be HSP_F32 or HSP_F64");
  if (N < 2 || p < 1) return na_fail(HSP_EINVAL, "hsp_xtz_noalloc: need N >= 2 and p >= 1");
  if (k < 1 || k > 0xffffffffLL) return na_fail(HSP_EINVAL, "hsp_xtz_noalloc: the sweep number k must be in [1, 2^32)");
  cudaStream_t st = (cudaStream_t)stream;
  int dev = 0, num_sms = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e == cudaSuccess) e = cudaDeviceGetAttribute(&num_sms, cudaDevAttrMultiProcessorCount, dev);
  if (e != cudaSuccess) return na_fail(HSP_ECUDA, std::string("hsp_xtz_noalloc: ") + cudaGetErrorString(e));
  const Options opt{};                                   // the automatic plan: this entry point takes no options
  const int dtype = x_dtype == HSP_F32 ? kF32 : kF64;
  const FusedPlan plan = fused_plan(dtype, N, p, num_sms, X, opt);
  const size_t n_part = (size_t)plan.grid * plan.groups;
  if (n_part * (size_t)p > kNoAllocPartialDoubles)
    return na_fail(HSP_EINVAL, "hsp_xtz_noalloc: problem too large for the static scratch: (CTAs x row groups) x p = " +
                                   std::to_string(n_part) + " x " + std::to_string(p) + " doubles > " +
                                   std::to_string(kNoAllocPartialDoubles) + " (8 MiB); use hsp_create / hsp_sweep");
  double* scratch = nullptr;
  e = scratch_for_current_device(&scratch);
  if (e != cudaSuccess) return na_fail(HSP_ECUDA, std::string("hsp_xtz_noalloc: cudaGetSymbolAddress: ") + cudaGetErrorString(e));
  const Ctl* ctl = reinterpret_cast<const Ctl*>(scratch);
  double* partial = scratch + kNoAllocHeadDoubles;
  // opt-in shared-memory attribute of the selected kernel (per device; no allocation), then: set-up, pass, reduce
  e = fused_pass_launch(plan, X, dtype, y, -1, p, 0, nullptr, nullptr, nullptr, nullptr, st);
  if (e == cudaSuccess) {
    const size_t n_clear = n_part * (size_t)p;
    const unsigned blocks = (unsigned)std::min<size_t>((n_clear + 255) / 256 + 1, 1184);
    noalloc_setup_kernel<<<blocks, 256, 0, st>>>((unsigned long long)(k - 1), n_clear);
    e = cudaGetLastError();
  }
  if (e == cudaSuccess) e = fused_pass_launch(plan, X, dtype, y, N, p, seed, beta, ctl, partial, z_out, st);
  if (e == cudaSuccess) e = reduce_partials_launch(partial, (int)n_part, p, g_out, st);
  if (e != cudaSuccess) return na_fail(HSP_ECUDA, std::string("hsp_xtz_noalloc: ") + cudaGetErrorString(e));
  return HSP_OK;
}

}  // extern "C"
