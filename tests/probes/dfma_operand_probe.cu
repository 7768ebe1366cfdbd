// dfma_operand_probe.cu — test-only micro-architecture probe (NOT part of liblr.so).
//
// Measures the DFMA issue rate of this device for instruction streams whose sources come from different places;
// tests/test_gpu_fp64_probe.py compiles this file with nvcc on the GPU box, loads it with ctypes and checks the
// ordering DESIGN.md §6 relies on (shared operands issue faster than fresh ones).
#include <cuda_runtime.h>
#include <stdint.h>

namespace {
// The DFMA streams behind DESIGN.md §6's issue rules: 7 accumulators per thread, each instruction
// acc[i] = fma(x, y, acc[i]) with (x, y) =
//   mode 0: (c[j], w[j])      both sources shared with the neighbouring instructions
//   mode 1: (c[i], w[j])      one source shared
//   mode 2: (c[i], w[i])      none shared: three registers the previous instruction did not read
//   mode 3: mode 1 plus one shared-memory load (LDS.64, immediate offset) per 7 DFMA, as in a filter loop
template <int MODE>
__global__ void __launch_bounds__(128) dfma_operand_kernel(const double* __restrict__ in, int iters, double* out) {
  __shared__ double ks[64];
  if (threadIdx.x < 64) ks[threadIdx.x] = in[threadIdx.x];
  __syncthreads();
  double acc[7], c[7], w[7];
#pragma unroll
  for (int i = 0; i < 7; ++i) { acc[i] = in[i]; c[i] = in[7 + i + threadIdx.x % 3]; w[i] = in[14 + i + threadIdx.x % 5]; }
  for (int it = 0; it < iters; ++it) {
    const double* kp = ks + (it & 31);
#pragma unroll
    for (int j = 0; j < 7; ++j) {
      const double wj = MODE == 3 ? kp[j] : w[j];
#pragma unroll
      for (int i = 0; i < 7; ++i) {
        if (MODE == 0) acc[i] = fma(c[j], w[j], acc[i]);
        if (MODE == 1 || MODE == 3) acc[i] = fma(c[i], wj, acc[i]);
        if (MODE == 2) acc[i] = fma(c[i], w[i], acc[i]);
      }
    }
  }
  double s = 0.0;
#pragma unroll
  for (int i = 0; i < 7; ++i) s += acc[i];
  out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

template <int MODE>
static int run_operand_probe(int sms, int iters, double* rate) {
  const int blocks = sms * 4, threads = 128;
  double *in = nullptr, *out = nullptr;
  if (cudaMalloc(&in, 64 * sizeof(double)) != cudaSuccess) return -3;
  if (cudaMalloc(&out, (size_t)blocks * threads * sizeof(double)) != cudaSuccess) { cudaFree(in); return -3; }
  cudaMemset(in, 0, 64 * sizeof(double));
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0);
  cudaEventCreate(&e1);
  dfma_operand_kernel<MODE><<<blocks, threads>>>(in, 16, out);
  cudaEventRecord(e0);
  dfma_operand_kernel<MODE><<<blocks, threads>>>(in, iters, out);
  cudaEventRecord(e1);
  int rc = 0;
  if (cudaEventSynchronize(e1) != cudaSuccess || cudaGetLastError() != cudaSuccess) rc = -3;
  float ms = 0;
  cudaEventElapsedTime(&ms, e0, e1);
  *rate = (double)blocks * threads * 49.0 * (double)iters / (ms * 1e-3);
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  cudaFree(in);
  cudaFree(out);
  return rc;
}
}  // namespace

extern "C" int probe_fp64_operands(int mode, double* inst_per_s) {
  if (!inst_per_s || mode < 0 || mode > 3) return -1;
  int dev = 0, sms = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) return -3;
  if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return -3;
  const int iters = 4000;
  switch (mode) {
    case 0: return run_operand_probe<0>(sms, iters, inst_per_s);
    case 1: return run_operand_probe<1>(sms, iters, inst_per_s);
    case 2: return run_operand_probe<2>(sms, iters, inst_per_s);
    default: return run_operand_probe<3>(sms, iters, inst_per_s);
  }
}

