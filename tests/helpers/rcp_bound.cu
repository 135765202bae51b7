// rcp_bound.cu -- evidence for the error bound the approximate-quotient filters of rt_bundle.cuh
// (scan_filtered) and rt_fast.cuh (q_key) rest on: rcp.approx.ftz.f64 (MUFU.RCP64H) is within
// 2^-19.5 relative of 1/x for every normal x in [2^-923, 2^924) (outside that range the kernels do
// not use it: filter_unsafe).  Compiled and run by tests/test_gpu_kernel_facts.py; standalone:
//   nvcc -O3 -gencode arch=compute_100a,code=sm_100a -o rcp_bound rcp_bound.cu && ./rcp_bound
// Sweep: every exponent of the range with (a) the mantissas all-zeros, all-ones, alternating bits,
// single low/high bits, (b) mantissas stepping through the 2^20 values of the high word (the only
// part MUFU.RCP64H reads) with random low words, (c) pseudo-random values -- > 2e9 inputs in all.
// Relative error is measured as |fma(y, x, -1)|, exact up to one rounding of a quantity ~2^-20.
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <cmath>
#include <cstdint>
#include <cuda_runtime.h>

typedef unsigned long long u64;

__device__ __forceinline__ double rcp_approx(double x) {
  double y;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
  return y;
}
__device__ __forceinline__ u64 mix(u64 z) {   // splitmix64
  z += 0x9E3779B97F4A7C15ull;
  z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
  z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
  return z ^ (z >> 31);
}
__device__ __forceinline__ void probe(double x, double &worst, double &worst_x) {
  const double e = fabs(fma(rcp_approx(x), x, -1.0));
  if (e > worst) { worst = e; worst_x = x; }
}

constexpr int kExpLo = 1023 - 923, kExpHi = 1023 + 924;   // biased exponents [lo, hi)

__global__ void sweep(u64 *out_err_bits, u64 *out_x_bits, u64 *out_count, int per_thread_random) {
  const u64 gid = (u64)blockIdx.x * blockDim.x + threadIdx.x;
  const u64 nthreads = (u64)gridDim.x * blockDim.x;
  double worst = 0.0, worst_x = 1.0;
  u64 count = 0;
  // (a) + (b): exponent-major, mantissa high words strided over the threads
  for (u64 idx = gid; idx < (u64)(kExpHi - kExpLo) * (1u << 20); idx += nthreads) {
    const u64 e = kExpLo + idx / (1u << 20), hi20 = idx % (1u << 20);
    const u64 lows[4] = {0ull, 0xffffffffull, 0xaaaaaaaaull, mix(idx) & 0xffffffffull};
#pragma unroll
    for (int v = 0; v < 4; ++v) {
      probe(__longlong_as_double((long long)((e << 52) | (hi20 << 32) | lows[v])), worst, worst_x);
      count += 1;
    }
  }
  // (c) pseudo-random normal values of the range, both signs of nothing: a_k > 0 always
  u64 s = mix(gid * 0x100000001B3ull + 12345);
  for (int i = 0; i < per_thread_random; ++i) {
    s = mix(s);
    const u64 e = kExpLo + (s >> 52) % (u64)(kExpHi - kExpLo);
    probe(__longlong_as_double((long long)((e << 52) | (s & 0xfffffffffffffull))), worst, worst_x);
    count += 1;
  }
  atomicAdd(out_count, count);
  const u64 bits = (u64)__double_as_longlong(worst);          // non-negative doubles order like integers
  if (atomicMax(out_err_bits, bits) < bits) *out_x_bits = (u64)__double_as_longlong(worst_x);
}

int main() {
  u64 *d;
  if (cudaMalloc(&d, 3 * sizeof(u64)) != cudaSuccess) { printf("cudaMalloc failed\n"); return 2; }
  cudaMemset(d, 0, 3 * sizeof(u64));
  sweep<<<148 * 8, 256>>>(d, d + 1, d + 2, 4096);
  if (cudaDeviceSynchronize() != cudaSuccess) { printf("kernel failed: %s\n", cudaGetErrorString(cudaGetLastError())); return 2; }
  u64 h[3];
  cudaMemcpy(h, d, sizeof(h), cudaMemcpyDeviceToHost);
  double err, x;
  memcpy(&err, &h[0], 8);
  memcpy(&x, &h[1], 8);
  printf("inputs=%llu max_rel_err=%a (%.6g = 2^%.3f) near x=%a\n", h[2], err, err, log2(err), x);
  return 0;
}
