// lr_kernels.cu — dispatch on the Lagrange order, and the small helper kernel.
//
// Orders 1-15 (odd), 21, 25, 31 and 41 have kernels with the pair count P = (order+1)/2 fixed at compile time (fully
// unrolled weight recurrences, everything in registers; instantiated by lr_inst.cu); any other odd order up
// to LR_MAX_ORDER runs the same code with P read at run time.
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

__global__ void source_basis_kernel(const double* __restrict__ angles, int64_t batch, double* __restrict__ basis) {
  const int64_t b = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (b >= batch) return;
  double o[9];
  source_basis(angles[3 * b], angles[3 * b + 1], angles[3 * b + 2], o);
#pragma unroll
  for (int a = 0; a < 9; ++a) basis[9 * b + a] = o[a];
}

int launch_source_basis(const double* angles, int64_t batch, double* basis, void* stream) {
  const int threads = 128;
  source_basis_kernel<<<(unsigned)((batch + threads - 1) / threads), threads, 0, (cudaStream_t)stream>>>(angles, batch,
                                                                                                       basis);
  g_launches.fetch_add(1);
  return (int)cudaGetLastError();
}

__global__ void source_basis_small_kernel(const SmallStage s, double* __restrict__ slot) {
  const int b = threadIdx.x, n = s.n;
  if (b >= n) return;
  const double* ang = s.v + 6 * n + 3 * b;
  double o[9];
  source_basis(ang[0], ang[1], ang[2], o);
#pragma unroll
  for (int a = 0; a < 9; ++a) slot[9 * b + a] = o[a];
  if (s.has_gb) {
#pragma unroll
    for (int a = 0; a < 6; ++a) slot[9 * n + 6 * b + a] = s.v[6 * b + a];
  }
}

int launch_source_basis_small(const SmallStage& s, double* slot, void* stream) {
  source_basis_small_kernel<<<1, 32, 0, (cudaStream_t)stream>>>(s, slot);
  g_launches.fetch_add(1);
  return (int)cudaGetLastError();
}

int launch_project(const Params& prm, int order, const double* hp, const double* hc, const double* basis,
                   double* y, int64_t batch, void* stream) {
  switch (order) {
    case 1: return launch_project_t<1>(prm, hp, hc, basis, y, batch, stream);
    case 3: return launch_project_t<2>(prm, hp, hc, basis, y, batch, stream);
    case 5: return launch_project_t<3>(prm, hp, hc, basis, y, batch, stream);
    case 7: return launch_project_t<4>(prm, hp, hc, basis, y, batch, stream);
    case 9: return launch_project_t<5>(prm, hp, hc, basis, y, batch, stream);
    case 11: return launch_project_t<6>(prm, hp, hc, basis, y, batch, stream);
    case 13: return launch_project_t<7>(prm, hp, hc, basis, y, batch, stream);
    case 15: return launch_project_t<8>(prm, hp, hc, basis, y, batch, stream);
    case 21: return launch_project_t<11>(prm, hp, hc, basis, y, batch, stream);
    case 31: return launch_project_t<16>(prm, hp, hc, basis, y, batch, stream);
    case 41: return launch_project_t<21>(prm, hp, hc, basis, y, batch, stream);
    case 25: return launch_project_t<13>(prm, hp, hc, basis, y, batch, stream);
    default: return launch_project_t<0>(prm, hp, hc, basis, y, batch, stream);
  }
}

int launch_tdi(const Params& prm, int order, int gen, int path, int channels, const double* y, double* out,
               int64_t batch, const FirPlanArgs& plan, void* stream) {
  switch (order) {
    case 1: return launch_tdi_t<1>(prm, gen, path, channels, y, out, batch, plan, stream);
    case 3: return launch_tdi_t<2>(prm, gen, path, channels, y, out, batch, plan, stream);
    case 5: return launch_tdi_t<3>(prm, gen, path, channels, y, out, batch, plan, stream);
    case 7: return launch_tdi_t<4>(prm, gen, path, channels, y, out, batch, plan, stream);
    case 9: return launch_tdi_t<5>(prm, gen, path, channels, y, out, batch, plan, stream);
    case 11: return launch_tdi_t<6>(prm, gen, path, channels, y, out, batch, plan, stream);
    case 13: return launch_tdi_t<7>(prm, gen, path, channels, y, out, batch, plan, stream);
    case 15: return launch_tdi_t<8>(prm, gen, path, channels, y, out, batch, plan, stream);
    case 21: return launch_tdi_t<11>(prm, gen, path, channels, y, out, batch, plan, stream);
    case 31: return launch_tdi_t<16>(prm, gen, path, channels, y, out, batch, plan, stream);
    case 41: return launch_tdi_t<21>(prm, gen, path, channels, y, out, batch, plan, stream);
    case 25: return launch_tdi_t<13>(prm, gen, path, channels, y, out, batch, plan, stream);
    default: return launch_tdi_t<0>(prm, gen, path, channels, y, out, batch, plan, stream);
  }
}

int launch_fir_plan(const Params& prm, int order, int gen, int path, double* coef, int* flags, int* list,
                    int plan_tiles, void* stream) {
  switch (order) {
    case 1: return launch_fir_plan_t<1>(prm, gen, path, coef, flags, list, plan_tiles, stream);
    case 3: return launch_fir_plan_t<2>(prm, gen, path, coef, flags, list, plan_tiles, stream);
    case 5: return launch_fir_plan_t<3>(prm, gen, path, coef, flags, list, plan_tiles, stream);
    case 7: return launch_fir_plan_t<4>(prm, gen, path, coef, flags, list, plan_tiles, stream);
    case 9: return launch_fir_plan_t<5>(prm, gen, path, coef, flags, list, plan_tiles, stream);
    case 11: return launch_fir_plan_t<6>(prm, gen, path, coef, flags, list, plan_tiles, stream);
    case 13: return launch_fir_plan_t<7>(prm, gen, path, coef, flags, list, plan_tiles, stream);
    case 15: return launch_fir_plan_t<8>(prm, gen, path, coef, flags, list, plan_tiles, stream);
    case 21: return launch_fir_plan_t<11>(prm, gen, path, coef, flags, list, plan_tiles, stream);
    case 31: return launch_fir_plan_t<16>(prm, gen, path, coef, flags, list, plan_tiles, stream);
    case 41: return launch_fir_plan_t<21>(prm, gen, path, coef, flags, list, plan_tiles, stream);
    case 25: return launch_fir_plan_t<13>(prm, gen, path, coef, flags, list, plan_tiles, stream);
    default: return launch_fir_plan_t<0>(prm, gen, path, coef, flags, list, plan_tiles, stream);
  }
}

}  // namespace lr
