// lr_peak.cu — FP64 issue-rate microbenchmark (lr_measure_fp64_peak).
//
// MEASURED_PEAKS.json records no FP64 peak, and the response path is bound by the FP64 pipe,
// so bench.py measures the roofline denominator on the device it runs on: every thread runs 8 independent
// DFMA chains acc = fma(acc, x, y), x a register shared by the chains and y a kernel parameter (ptxas keeps it in
// a uniform register: `DFMA R2, R2, R26.reuse, UR6`), 2,048 threads per SM, all SMs, for about the requested time.
// The operand form matters on sm_100 (measured on B200 at 1.965 GHz, 16-64 warps per SM, 8 or 16 chains):
//   acc * reg + uniform register            63.0-63.6 DFMA per SM and clock  (the pipe has 64: this kernel)
//   acc * reg + reg (both shared, .reuse)   58.1-58.7  (the round's first version of this kernel: 1.71e13 /s)
//   two fresh register operands per DFMA    48-54, depending on the registers ptxas picks
// The first line is the rate of the pipe itself and the one a kernel is held against.
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
  const double x = a - (double)threadIdx.x * 1e-12;   // a register; b stays a kernel parameter (uniform register)
  for (int64_t it = 0; it < outer; ++it) {
#pragma unroll
    for (int i = 0; i < kInner; ++i) {
#pragma unroll
      for (int c = 0; c < kChains; ++c) acc[c] = fma(acc[c], x, b);
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
