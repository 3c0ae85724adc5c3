// Test-only probe (NOT part of libhsp.so, never on the product path): the CUDA toolkit's own cuRAND DEVICE
// Philox4_32_10 generator, addressed the way DESIGN.md 3 maps the sweep's counters onto it:
//   curand_init(seed, subsequence = (tag << 32) | k, offset = 4 * idx)  ->  counter (idx_lo, idx_hi, k, tag), key = seed
// so that curand4() returns the Philox-4x32-10 block of one variate.  tests/test_gpu_curand_pin.py compares the
// words with the oracle's independent implementation: this pins counter words c2 and c3 (sweep and tag), which the
// cuRAND HOST generator of tests/test_oracle_rng.py cannot reach.
#include <cuda_runtime.h>
#include <curand_kernel.h>

__global__ void probe_kernel(unsigned long long seed, const unsigned long long* subseq, const unsigned long long* offset,
                             unsigned* out, int n) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  curandStatePhilox4_32_10_t st;
  curand_init(seed, subseq[i], offset[i], &st);
  const uint4 r = curand4(&st);
  out[4 * i] = r.x; out[4 * i + 1] = r.y; out[4 * i + 2] = r.z; out[4 * i + 3] = r.w;
}

// HOST pointers in and out; returns 0 or the cudaError_t.
extern "C" int curand_philox_probe(unsigned long long seed, const unsigned long long* subseq, const unsigned long long* offset,
                                   unsigned* out, int n) {
  unsigned long long *d_s = nullptr, *d_o = nullptr;
  unsigned* d_out = nullptr;
  cudaError_t e = cudaMalloc(&d_s, n * sizeof(unsigned long long));
  if (e == cudaSuccess) e = cudaMalloc(&d_o, n * sizeof(unsigned long long));
  if (e == cudaSuccess) e = cudaMalloc(&d_out, 4 * n * sizeof(unsigned));
  if (e == cudaSuccess) e = cudaMemcpy(d_s, subseq, n * sizeof(unsigned long long), cudaMemcpyHostToDevice);
  if (e == cudaSuccess) e = cudaMemcpy(d_o, offset, n * sizeof(unsigned long long), cudaMemcpyHostToDevice);
  if (e == cudaSuccess) {
    probe_kernel<<<(n + 127) / 128, 128>>>(seed, d_s, d_o, d_out, n);
    e = cudaGetLastError();
  }
  if (e == cudaSuccess) e = cudaMemcpy(out, d_out, 4 * n * sizeof(unsigned), cudaMemcpyDeviceToHost);
  cudaFree(d_s); cudaFree(d_o); cudaFree(d_out);
  return (int)e;
}
