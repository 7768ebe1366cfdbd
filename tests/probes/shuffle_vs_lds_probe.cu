// shuffle_vs_lds_probe.cu — test-only probe (NOT part of liblr.so): what does it cost a warp to hand every lane the
// 16-byte stencil element (h+, hx difference) of its neighbour, from shared memory (one LDS.128 per lane) or from the
// neighbour's registers (four SHFL.32 per lane)?  north_star names warp shuffles for the stencil reductions; DESIGN.md
// §6 argues that they go through the same pipe as the loads at four times the issue slots.  This measures it.
// probe_exchange(mode, &elements_per_s): mode 0 = LDS.128, mode 1 = 4 x SHFL.32; 16-byte elements delivered per second
// over the whole device (16 warps per SM, a dependent-free stream of exchanges, a few milliseconds).
#include <cuda_runtime.h>
#include <stdint.h>

namespace {
constexpr int kThreads = 128, kUnroll = 16;

template <int MODE>
__global__ void __launch_bounds__(kThreads) exchange_kernel(const double2* __restrict__ in, int iters, double* out) {
  __shared__ double2 win[kThreads + kUnroll + 1];
  for (int i = threadIdx.x; i < kThreads + kUnroll + 1; i += kThreads) win[i] = in[i];
  __syncthreads();
  double ax = 0.0, ay = 0.0;
  double2 mine[4];   // four independent values: the shuffles of one do not wait for each other
#pragma unroll
  for (int i = 0; i < 4; ++i) mine[i] = win[threadIdx.x + i];
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int u = 0; u < kUnroll; ++u) {
      double2 v;
      if (MODE == 0) {
        v = win[threadIdx.x + u + (it & 1)];                       // LDS.128, lanes 16 bytes apart: conflict-free
      } else {
        // the same element from the neighbour's registers: two 64-bit shuffles = four SHFL.32
        v.x = __shfl_down_sync(0xffffffffu, mine[u & 3].x, 1);
        v.y = __shfl_down_sync(0xffffffffu, mine[u & 3].y, 1);
        mine[u & 3].x = v.y;                                        // (keeps every shuffle in the loop)
        mine[u & 3].y = v.x;
      }
      ax += v.x;
      ay += v.y;
    }
  }
  out[blockIdx.x * kThreads + threadIdx.x] = ax + ay;
}

template <int MODE>
int run(int sms, int iters, double* rate) {
  const int blocks = sms * 4;
  double2* in = nullptr;
  double* out = nullptr;
  if (cudaMalloc(&in, (kThreads + kUnroll + 1) * sizeof(double2)) != cudaSuccess) return -3;
  if (cudaMalloc(&out, (size_t)blocks * kThreads * sizeof(double)) != cudaSuccess) { cudaFree(in); return -3; }
  cudaMemset(in, 0, (kThreads + kUnroll + 1) * sizeof(double2));
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0);
  cudaEventCreate(&e1);
  exchange_kernel<MODE><<<blocks, kThreads>>>(in, 16, out);
  cudaEventRecord(e0);
  exchange_kernel<MODE><<<blocks, kThreads>>>(in, iters, out);
  cudaEventRecord(e1);
  int rc = 0;
  if (cudaEventSynchronize(e1) != cudaSuccess || cudaGetLastError() != cudaSuccess) rc = -3;
  float ms = 0;
  cudaEventElapsedTime(&ms, e0, e1);
  *rate = (double)blocks * kThreads * kUnroll * (double)iters / (ms * 1e-3);
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  cudaFree(in);
  cudaFree(out);
  return rc;
}
}  // namespace

extern "C" int probe_exchange(int mode, double* elements_per_s) {
  if (!elements_per_s || mode < 0 || mode > 1) return -1;
  int dev = 0, sms = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) return -3;
  if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return -3;
  return mode == 0 ? run<0>(sms, 20000, elements_per_s) : run<1>(sms, 20000, elements_per_s);
}
