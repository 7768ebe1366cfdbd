// lr_peak.cu — FP64 issue-rate microbenchmark (lr_measure_fp64_peak).
//
// MEASURED_PEAKS.json records no FP64 peak, and the response path is bound by the FP64 pipe,
// so bench.py measures the roofline denominator on the device it runs on: every thread runs 8 independent
// DFMA chains, 1024 threads per SM-slot, all SMs, for about the requested time.
#include <cuda_runtime.h>
#include <stdint.h>

#include <atomic>

#include "../../include/lr.h"

namespace lr {
extern std::atomic<int64_t> g_launches;

constexpr int kChains = 8;
constexpr int kInner = 64;  // DFMA per chain per outer iteration

__global__ void __launch_bounds__(256) dfma_kernel(double a, double b, int64_t outer, double* sink) {
  double acc[kChains];
#pragma unroll
  for (int c = 0; c < kChains; ++c) acc[c] = (double)(threadIdx.x + c) * 1e-9;
  for (int64_t it = 0; it < outer; ++it) {
#pragma unroll
    for (int i = 0; i < kInner; ++i) {
#pragma unroll
      for (int c = 0; c < kChains; ++c) acc[c] = fma(acc[c], a, b);
    }
  }
  double s = 0.0;
#pragma unroll
  for (int c = 0; c < kChains; ++c) s += acc[c];
  if (s == 123.456) sink[0] = s;  // never true for the arguments used; keeps the chains alive
}
}  // namespace lr

extern "C" int lr_measure_fp64_peak(double seconds, double* inst_per_s) {
  if (!inst_per_s || !(seconds > 0) || seconds > 30) return LR_EINVAL;
  int dev = 0, sms = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) return LR_ECUDA;
  if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return LR_ECUDA;
  double* sink = nullptr;
  if (cudaMalloc(&sink, sizeof(double)) != cudaSuccess) return LR_ECUDA;
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0);
  cudaEventCreate(&e1);
  const int threads = 256, blocks = sms * 8;
  int rc = LR_OK;
  int64_t outer = 256;
  double best = 0.0;
  // calibrate, then one long run
  for (int pass = 0; pass < 3; ++pass) {
    cudaEventRecord(e0);
    lr::dfma_kernel<<<blocks, threads>>>(0.999999, 1e-7, outer, sink);
    lr::g_launches.fetch_add(1);
    cudaEventRecord(e1);
    if (cudaEventSynchronize(e1) != cudaSuccess || cudaGetLastError() != cudaSuccess) { rc = LR_ECUDA; break; }
    float ms = 0;
    cudaEventElapsedTime(&ms, e0, e1);
    const double inst = (double)blocks * threads * lr::kChains * lr::kInner * (double)outer;
    const double rate = inst / (ms * 1e-3);
    if (pass == 2 || rate > best) best = rate;
    if (pass == 2) break;
    const double target = (pass == 0 ? 0.05 : seconds);
    outer = (int64_t)(outer * (target / (ms * 1e-3))) + 1;
  }
  *inst_per_s = best;
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  cudaFree(sink);
  return rc;
}
