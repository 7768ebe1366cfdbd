// lr_inst.cu — kernel instantiations for ONE compile-time pair count LR_INST_PT (build.py compiles this file
// once per fast order; LR_INST_PT = 0 is the run-time-P build that serves every other odd order).
#include <cuda_runtime.h>

#include <atomic>

#include "lr_kernels.cuh"

#ifndef LR_INST_PT
#error "compile with -DLR_INST_PT=<P>"
#endif

namespace lr {

extern std::atomic<int64_t> g_launches;

template <class K>
static cudaError_t prepare(K kernel, size_t smem) {
  if (smem > 48 * 1024) return cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  return cudaSuccess;
}

template <int PT>
int launch_project_t(const Params& prm, const double* hp, const double* hc, const double* basis, double* y,
                     int64_t batch, void* stream) {
  const size_t W = (size_t)kProjThreads + prm.halo_lo + prm.halo_hi;
  const size_t smem = 2 * W * sizeof(D2);
  cudaError_t e = prepare(project_kernel<PT>, smem);
  if (e != cudaSuccess) return (int)e;
  const int64_t grid = (int64_t)prm.ntiles * batch;
  if constexpr (proj_pairs(PT)) {
    if (prm.proj_pair && !prm.proj_ext) {
      const size_t smem2 = proj_pair_smem((int)W);
      if ((e = prepare(project_pair_kernel<PT>, smem2)) != cudaSuccess) return (int)e;
      project_pair_kernel<PT><<<(unsigned)grid, kProjPairThreads, smem2, (cudaStream_t)stream>>>(prm, hp, hc, basis, y);
      g_launches.fetch_add(1);
      return (int)cudaGetLastError();
    }
  }
  if (prm.proj_ext) {
    if ((e = prepare(project_kernel<PT, true>, smem)) != cudaSuccess) return (int)e;
    project_kernel<PT, true><<<(unsigned)grid, kProjThreads, smem, (cudaStream_t)stream>>>(prm, hp, hc, basis, y);
  } else {
    project_kernel<PT><<<(unsigned)grid, kProjThreads, smem, (cudaStream_t)stream>>>(prm, hp, hc, basis, y);
  }
  g_launches.fetch_add(1);
  return (int)cudaGetLastError();
}

template <int PT, int GEN>
static int launch_tdi_generic(const Params& prm, int channels, const double* y, double* out, int64_t batch,
                              cudaStream_t st) {
  const size_t W = (size_t)kTdiThreads + prm.halo_lo + prm.halo_hi;
  const size_t smem = 12 * W * sizeof(double);
  cudaError_t e = prepare(tdi_kernel<PT, GEN>, smem);
  if (e != cudaSuccess) return (int)e;
  const int64_t grid = (int64_t)prm.ntiles * batch;
  tdi_kernel<PT, GEN><<<(unsigned)grid, kTdiThreads, smem, st>>>(prm, y, out, channels);
  g_launches.fetch_add(1);
  return (int)cudaGetLastError();
}

// FIR path, plan: one CTA per tile of the whole series (prm.ntiles = plan_tiles, window = the whole series)
template <int PT, int GEN, int NN>
static int launch_fir_plan_g(const Params& prm, double* coef, int* flags, int* list, int plan_tiles, cudaStream_t st) {
  const int P = PT > 0 ? PT : prm.p;
  cudaError_t e;
  const size_t smem = ((sizeof(FirTile<GEN, NN>) + 15) / 16) * 16 +
                      (size_t)FirTile<GEN, NN>::NT * NN * (2 * P - 1) * sizeof(double);
  if ((e = prepare(tdi_fir_setup_kernel<PT, GEN, NN>, smem)) != cudaSuccess) return (int)e;
  if ((e = cudaMemsetAsync(list, 0, sizeof(int), st)) != cudaSuccess) return (int)e;
  tdi_fir_setup_kernel<PT, GEN, NN><<<(unsigned)plan_tiles, kFirSetupThreads, smem, st>>>(prm, coef, flags, list);
  g_launches.fetch_add(1);
  return (int)cudaGetLastError();
}

template <int PT>
int launch_fir_plan_t(const Params& prm, int gen, int path, double* coef, int* flags, int* list, int plan_tiles,
                      void* stream) {
  cudaStream_t st = (cudaStream_t)stream;
  if (path == kPathFir3)
    return gen == 1 ? launch_fir_plan_g<PT, 1, 3>(prm, coef, flags, list, plan_tiles, st)
                    : launch_fir_plan_g<PT, 2, 3>(prm, coef, flags, list, plan_tiles, st);
  return gen == 1 ? launch_fir_plan_g<PT, 1, 4>(prm, coef, flags, list, plan_tiles, st)
                  : launch_fir_plan_g<PT, 2, 4>(prm, coef, flags, list, plan_tiles, st);
}

// FIR path, apply: filter every tile the plan did not flag, and run the flagged tiles with per-sample weights
template <int PT, int GEN, int NN>
static int launch_tdi_fir(const Params& prm, int channels, const double* y, double* out, int64_t batch,
                          const FirPlanArgs& plan, cudaStream_t st) {
  cudaError_t e;
  const int W = kFirTile + prm.halo_lo + prm.halo_hi;
  const bool fixup = !plan.skip_fixup;
  if (fixup) {
    // fork: the flagged tiles (a handful, but each is a long dependent computation) run on the handle's side
    // stream while the apply kernel fills the GPU; the two write disjoint tiles of `out`
    cudaStream_t side = (cudaStream_t)plan.side;
    const size_t smem_fix = (size_t)12 * W * sizeof(double);
    if ((e = prepare(tdi_fir_fixup_kernel<PT, GEN>, smem_fix)) != cudaSuccess) return (int)e;
    if ((e = cudaEventRecord((cudaEvent_t)plan.fork, st)) != cudaSuccess) return (int)e;
    if ((e = cudaStreamWaitEvent(side, (cudaEvent_t)plan.fork, 0)) != cudaSuccess) return (int)e;
    tdi_fir_fixup_kernel<PT, GEN><<<plan.fixup_grid, kFirTile, smem_fix, side>>>(prm, y, out, channels, plan.list,
                                                                                 (int)batch);
    g_launches.fetch_add(1);
    if ((e = cudaGetLastError()) != cudaSuccess) return (int)e;
    if ((e = cudaEventRecord((cudaEvent_t)plan.join, side)) != cudaSuccess) return (int)e;
    if (plan.join_extra && (e = cudaEventRecord((cudaEvent_t)plan.join_extra, side)) != cudaSuccess) return (int)e;
  }

  const size_t smem = fir_apply_smem_bytes(W, prm.fir_wc);
  const int64_t grid = (int64_t)prm.ntiles * batch;
  if (prm.fir_uniform) {   // constant light times: the weights do not depend on tile time, k0 alone
    if ((e = prepare(tdi_fir_apply_kernel<1>, smem)) != cudaSuccess) return (int)e;
    tdi_fir_apply_kernel<1><<<(unsigned)grid, kFirThreads, smem, st>>>(prm, y, out, channels, plan.coef, plan.flags,
                                                                     (int)batch);
  } else if constexpr (NN == 4) {   // cubic plans: the tensor-path kernel (a full 8 x 8 x 4 FP64 MMA tile)
    const size_t smem_m = fir_mma_smem_bytes(W, prm.fir_wc);
    if ((e = prepare(tdi_fir_apply_mma_kernel<4>, smem_m)) != cudaSuccess) return (int)e;
    tdi_fir_apply_mma_kernel<4><<<(unsigned)grid, kFirMmaThreads, smem_m, st>>>(prm, y, out, channels, plan.coef,
                                                                              plan.flags, (int)batch);
  } else {
    if ((e = prepare(tdi_fir_apply_kernel<NN>, smem)) != cudaSuccess) return (int)e;
    tdi_fir_apply_kernel<NN><<<(unsigned)grid, kFirThreads, smem, st>>>(prm, y, out, channels, plan.coef, plan.flags,
                                                                      (int)batch);
  }
  g_launches.fetch_add(1);
  if ((e = cudaGetLastError()) != cudaSuccess) return (int)e;
  return fixup && plan.wait_join ? (int)cudaStreamWaitEvent(st, (cudaEvent_t)plan.join, 0) : 0;   // join
}

template <int PT>
int launch_tdi_t(const Params& prm, int gen, int path, int channels, const double* y, double* out, int64_t batch,
                 const FirPlanArgs& plan, void* stream) {
  cudaStream_t st = (cudaStream_t)stream;
  if (path == kPathFir3)
    return gen == 1 ? launch_tdi_fir<PT, 1, 3>(prm, channels, y, out, batch, plan, st)
                    : launch_tdi_fir<PT, 2, 3>(prm, channels, y, out, batch, plan, st);
  if (path == kPathFir4)
    return gen == 1 ? launch_tdi_fir<PT, 1, 4>(prm, channels, y, out, batch, plan, st)
                    : launch_tdi_fir<PT, 2, 4>(prm, channels, y, out, batch, plan, st);
  return gen == 1 ? launch_tdi_generic<PT, 1>(prm, channels, y, out, batch, st)
                  : launch_tdi_generic<PT, 2>(prm, channels, y, out, batch, st);
}

template int launch_project_t<LR_INST_PT>(const Params&, const double*, const double*, const double*, double*,
                                          int64_t, void*);
template int launch_fir_plan_t<LR_INST_PT>(const Params&, int, int, double*, int*, int*, int, void*);
template int launch_tdi_t<LR_INST_PT>(const Params&, int, int, int, const double*, double*, int64_t,
                                      const FirPlanArgs&, void*);

}  // namespace lr
