// lr_kernels.cu — kernel instantiations and launchers (sm_100a).
//
// Orders in LR_FAST_ORDERS get a kernel with the pair count P fixed at compile time (fully unrolled
// weight recurrences, everything in registers); any other odd order up to LR_MAX_ORDER runs the same code
// with P read at run time.
#include <cuda_runtime.h>

#include <atomic>

#include "lr_kernels.cuh"

namespace lr {

std::atomic<int64_t> g_launches{0};

__global__ void eval_orbit_kernel(const Params prm, int ch, double t_start, const double* __restrict__ t,
                                  int64_t m, double* __restrict__ out) {
  const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (i < m) out[i] = spline_eval(prm, ch, t[i] - t_start);
}

template <class K>
static cudaError_t prepare(K kernel, size_t smem) {
  if (smem > 48 * 1024) return cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  return cudaSuccess;
}

template <int PT>
static int launch_project_t(const Params& prm, const double* hp, const double* hc, const double* basis, double* y,
                            int64_t batch, cudaStream_t st) {
  const size_t W = (size_t)kProjThreads + prm.halo_lo + prm.halo_hi;
  const size_t smem = 2 * W * sizeof(D2);
  cudaError_t e = prepare(project_kernel<PT>, smem);
  if (e != cudaSuccess) return (int)e;
  const int64_t grid = (int64_t)prm.ntiles * batch;
  project_kernel<PT><<<(unsigned)grid, kProjThreads, smem, st>>>(prm, hp, hc, basis, y);
  g_launches.fetch_add(1);
  return (int)cudaGetLastError();
}

int launch_project(const Params& prm, int order, const double* hp, const double* hc, const double* basis,
                   double* y, int64_t batch, void* stream) {
  cudaStream_t st = (cudaStream_t)stream;
  switch (order) {
#ifndef LR_DEV_ONLY_P13
    case 1: return launch_project_t<1>(prm, hp, hc, basis, y, batch, st);
    case 3: return launch_project_t<2>(prm, hp, hc, basis, y, batch, st);
    case 9: return launch_project_t<5>(prm, hp, hc, basis, y, batch, st);
    case 41: return launch_project_t<21>(prm, hp, hc, basis, y, batch, st);
#endif
    case 25: return launch_project_t<13>(prm, hp, hc, basis, y, batch, st);
    default: return launch_project_t<0>(prm, hp, hc, basis, y, batch, st);
  }
}

template <int PT, int GEN, int MODE>
static int launch_tdi_t(const Params& prm, int channels, const double* y, double* out, int64_t batch,
                        cudaStream_t st) {
  const size_t W = (size_t)kTdiThreads + prm.halo_lo + prm.halo_hi;
  const size_t smem = 12 * W * sizeof(double);
  cudaError_t e = prepare(tdi_kernel<PT, GEN, MODE>, smem);
  if (e != cudaSuccess) return (int)e;
  const int64_t grid = (int64_t)prm.ntiles * batch;
  tdi_kernel<PT, GEN, MODE><<<(unsigned)grid, kTdiThreads, smem, st>>>(prm, y, out, channels);
  g_launches.fetch_add(1);
  return (int)cudaGetLastError();
}

template <int PT>
static int launch_tdi_p(const Params& prm, int gen, int mode, int channels, const double* y, double* out,
                        int64_t batch, cudaStream_t st) {
  if (gen == 1) {
    return mode == 0 ? launch_tdi_t<PT, 1, 0>(prm, channels, y, out, batch, st)
                     : launch_tdi_t<PT, 1, 1>(prm, channels, y, out, batch, st);
  }
  return mode == 0 ? launch_tdi_t<PT, 2, 0>(prm, channels, y, out, batch, st)
                   : launch_tdi_t<PT, 2, 1>(prm, channels, y, out, batch, st);
}

int launch_tdi(const Params& prm, int order, int gen, int mode, int channels, const double* y, double* out,
               int64_t batch, void* stream) {
  cudaStream_t st = (cudaStream_t)stream;
  switch (order) {
#ifndef LR_DEV_ONLY_P13
    case 1: return launch_tdi_p<1>(prm, gen, mode, channels, y, out, batch, st);
    case 3: return launch_tdi_p<2>(prm, gen, mode, channels, y, out, batch, st);
    case 9: return launch_tdi_p<5>(prm, gen, mode, channels, y, out, batch, st);
    case 41: return launch_tdi_p<21>(prm, gen, mode, channels, y, out, batch, st);
#endif
    case 25: return launch_tdi_p<13>(prm, gen, mode, channels, y, out, batch, st);
    default: return launch_tdi_p<0>(prm, gen, mode, channels, y, out, batch, st);
  }
}

}  // namespace lr
