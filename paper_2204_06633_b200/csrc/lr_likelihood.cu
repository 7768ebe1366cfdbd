// lr_likelihood.cu — noise-weighted inner product of frequency-domain TDI channels (lr_inner_product):
// PAPER.md eqs. 2-3 and 22, SURVEY.md §8(f) NEXT-2.  The Fourier transforms are a
// library step of the caller (cuFFT through torch.fft.rfft); this file is the weighted reduction, which is
// bound by HBM (40 B per frequency bin and channel) and deterministic (fixed two-stage tree, no atomics).
#include <cuda_runtime.h>
#include <stdint.h>

#include <atomic>

#include "../../include/lr.h"

namespace lr {
extern std::atomic<int64_t> g_launches;

constexpr int kIpThreads = 256;

__device__ __forceinline__ double block_sum(double v, double* sm) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  if (lane == 0) sm[warp] = v;
  __syncthreads();
  double t = 0.0;
  if (warp == 0) {
    t = lane < kIpThreads / 32 ? sm[lane] : 0.0;
#pragma unroll
    for (int o = 4; o > 0; o >>= 1) t += __shfl_down_sync(0xffffffffu, t, o);
  }
  __syncthreads();
  return t;   // valid in thread 0
}

// stage 1: grid (LR_IP_BLOCKS, batch); block bx of template b sums its contiguous slice of the M = nch*nf bins
__global__ void __launch_bounds__(kIpThreads)
ip_partial_kernel(const double2* __restrict__ fa, const double2* __restrict__ fb, const double* __restrict__ inv_psd,
                  int64_t M, int64_t batch_b, int mode, double* __restrict__ work) {
  __shared__ double sm[kIpThreads / 32];
  const int64_t b = blockIdx.y;
  const double2* a = fa + b * M;
  const double2* c = fb + (batch_b == 1 ? 0 : b) * M;
  const int64_t lo = M * blockIdx.x / gridDim.x, hi = M * (blockIdx.x + 1) / gridDim.x;
  double acc = 0.0;
  auto term = [&](const double2 x, const double2 y, const double w) {
    if (mode == 0) {
      acc = fma(fma(x.x, y.x, x.y * y.y), w, acc);            // Re(conj(a) b) / S_n
    } else {
      const double dr = x.x - y.x, di = x.y - y.y;            // |a - b|^2 / S_n
      acc = fma(fma(dr, dr, di * di), w, acc);
    }
  };
  int64_t e = lo + threadIdx.x;
  for (; e + 3 * kIpThreads < hi; e += 4 * kIpThreads) {      // four independent loads in flight per thread
    double2 x[4], y[4];
    double w[4];
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      x[u] = __ldg(a + e + u * kIpThreads); y[u] = __ldg(c + e + u * kIpThreads); w[u] = __ldg(inv_psd + e + u * kIpThreads);
    }
#pragma unroll
    for (int u = 0; u < 4; ++u) term(x[u], y[u], w[u]);
  }
  for (; e < hi; e += kIpThreads) term(__ldg(a + e), __ldg(c + e), __ldg(inv_psd + e));
  const double t = block_sum(acc, sm);
  if (threadIdx.x == 0) work[b * gridDim.x + blockIdx.x] = t;
}

// stage 2: one block per template adds the LR_IP_BLOCKS partial sums in a fixed order
__global__ void __launch_bounds__(kIpThreads)
ip_final_kernel(const double* __restrict__ work, int nblk, double scale, double* __restrict__ out) {
  __shared__ double sm[kIpThreads / 32];
  const int64_t b = blockIdx.x;
  double acc = 0.0;
  for (int i = threadIdx.x; i < nblk; i += kIpThreads) acc += work[b * nblk + i];
  const double t = block_sum(acc, sm);
  if (threadIdx.x == 0) out[b] = scale * t;
}
}  // namespace lr

extern "C" int lr_inner_product(const double* fa, const double* fb, const double* inv_psd, double scale, int mode,
                                int64_t batch, int64_t batch_b, int nch, int64_t nf, double* work, double* out,
                                void* stream) {
  if (!fa || !fb || !inv_psd || !work || !out) return LR_EINVAL;
  if (batch < 1 || batch > 65535 || (batch_b != 1 && batch_b != batch) || nch < 1 || nf < 1) return LR_EINVAL;
  if (mode != LR_IP_CROSS && mode != LR_IP_DIFF) return LR_EINVAL;
  const int64_t M = (int64_t)nch * nf;
  cudaStream_t st = (cudaStream_t)stream;
  dim3 grid(LR_IP_BLOCKS, (unsigned)batch);
  lr::ip_partial_kernel<<<grid, lr::kIpThreads, 0, st>>>(reinterpret_cast<const double2*>(fa),
                                                         reinterpret_cast<const double2*>(fb), inv_psd, M, batch_b,
                                                         mode, work);
  lr::ip_final_kernel<<<(unsigned)batch, lr::kIpThreads, 0, st>>>(work, LR_IP_BLOCKS, scale, out);
  lr::g_launches.fetch_add(2);
  return cudaGetLastError() == cudaSuccess ? LR_OK : LR_ECUDA;
}

// ------------------------------------------------------------------------------- no-allocation entry point
// lr_inner_product_static: the same two-stage reduction with its scratch (the per-block partial sums of stage 1) in a
// file-scope device array instead of a caller-supplied buffer, for callers that cannot allocate: code under CUDA
// graph capture, tight serving loops, harnesses that forbid cudaMalloc.  Every GPU that loads liblr holds the array
// (LR_IP_STATIC_MAX_BATCH x LR_IP_BLOCKS doubles = 512 KB) until the process exits.
namespace lr {
static __device__ __align__(256) double g_ip_static_work[(size_t)LR_IP_STATIC_MAX_BATCH * LR_IP_BLOCKS];

// In host code `g_ip_static_work` is a host-side stand-in for the symbol, not a device address; the address comes
// from cudaGetSymbolAddress, once per device, with that device current.
constexpr int kMaxDevices = 64;
static std::atomic<double*> g_ip_static_ptr[kMaxDevices];

static int ip_static_scratch(double** ptr) {
  int dev = -1;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= kMaxDevices) return LR_ECUDA;
  double* p = g_ip_static_ptr[dev].load(std::memory_order_acquire);
  if (!p) {   // set-up of this device (racing threads resolve the same address)
    void* q = nullptr;
    if (cudaGetSymbolAddress(&q, g_ip_static_work) != cudaSuccess || !q) {
      (void)cudaGetLastError();
      return LR_ECUDA;
    }
    p = static_cast<double*>(q);
    g_ip_static_ptr[dev].store(p, std::memory_order_release);
  }
  *ptr = p;
  return LR_OK;
}
}  // namespace lr

extern "C" int lr_inner_product_static(const double* fa, const double* fb, const double* inv_psd, double scale,
                                       int mode, int64_t batch, int64_t batch_b, int nch, int64_t nf, double* out,
                                       void* stream) {
  if (!fa || !fb || !inv_psd || !out) return LR_EINVAL;
  if (batch < 1 || (batch_b != 1 && batch_b != batch) || nch < 1 || nf < 1) return LR_EINVAL;
  if (mode != LR_IP_CROSS && mode != LR_IP_DIFF) return LR_EINVAL;
  if (batch > LR_IP_STATIC_MAX_BATCH) return LR_ELIMIT;   // the scratch array holds LR_IP_STATIC_MAX_BATCH templates
  double* work = nullptr;
  const int rc = lr::ip_static_scratch(&work);
  if (rc != LR_OK) return rc;
  const int64_t M = (int64_t)nch * nf;
  cudaStream_t st = (cudaStream_t)stream;
  // Nothing in the scratch has to start at zero: stage 1 writes every one of the batch x LR_IP_BLOCKS partial sums
  // stage 2 reads (a block with an empty slice writes 0), so whatever the previous call left behind is overwritten
  // before it is read.
  dim3 grid(LR_IP_BLOCKS, (unsigned)batch);
  lr::ip_partial_kernel<<<grid, lr::kIpThreads, 0, st>>>(reinterpret_cast<const double2*>(fa),
                                                         reinterpret_cast<const double2*>(fb), inv_psd, M, batch_b,
                                                         mode, work);
  lr::ip_final_kernel<<<(unsigned)batch, lr::kIpThreads, 0, st>>>(work, LR_IP_BLOCKS, scale, out);
  lr::g_launches.fetch_add(2);
  return cudaGetLastError() == cudaSuccess ? LR_OK : LR_ECUDA;
}
