// lr_kernels.cuh — the two CUDA kernels of liblr (sm_100a) and their launchers' declarations.
//
//   project_kernel<PT>       : PAPER.md eqs. 10-16, one thread per time sample, all six links
//   tdi_kernel<PT,GEN>       : PAPER.md eqs. 17-21, one thread per time sample, X, Y, Z (+ A, E, T)
//   (lr_tdi_fir.cuh holds the fast TDI path: tdi_fir_setup_kernel + tdi_fir_apply_kernel)
//
// Both stage the window a tile of samples needs (raw samples and their exact first differences) in
// shared memory with coalesced loads, keep the Lagrange pair products in registers, and write coalesced
// fp64 along the time axis.  The path is bound by the FP64 pipe, so there is no tensor-core
// or TMA use: the staged windows are small (tens of KB) and each is read ~T times from shared memory.
#pragma once
#include "lr_device.cuh"

namespace lr {

// Launch shapes, tuned on B200: both kernels are bound by the FP64 pipe and want
// 12-24 resident warps per SM; letting ptxas take 160-250 registers per thread (one CTA per SM) halves the
// throughput.  The caps below keep the order-25 kernels spill-free.
constexpr int kProjThreads = 128;      // samples per projection tile (and threads of the one-sample-per-thread kernel)
constexpr int kProjPairThreads = 64;   // threads of the two-samples-per-thread kernel (same 128-sample tile)
constexpr int kTdiThreads = 256;
// elements of each half of the de-interleaved difference window of the pair kernel
__host__ __device__ constexpr int proj_pair_half(int W) { return (W >> 1) + 1; }
// dynamic shared memory of project_pair_kernel: raw[W], dif_e[H], dif_o[H] (D2), geo[kGeoFields][threads]
__host__ __device__ constexpr size_t proj_pair_smem(int W) {
  return (size_t)(W + 2 * proj_pair_half(W)) * sizeof(D2) + (size_t)kGeoFields * kProjPairThreads * sizeof(double);
}
// orders whose projection runs two samples per thread (compile-time P; the run-time-P build keeps one)
__host__ __device__ constexpr bool proj_pairs(int PT) { return PT >= 1; }
// (orders 31 and 41 spill 40-110 B at the 128 registers of 4 CTAs per SM and are still 2-4 % faster than at 3 CTAs)
__host__ __device__ constexpr int proj_min_blocks(int PT) { return PT == 0 ? 2 : 4; }
__host__ __device__ constexpr int tdi_min_blocks(int PT) { return PT == 0 ? 2 : PT <= 13 ? 3 : 2; }

// ---------------------------------------------------------------------------------------------- stage 1
// grid.x = ntiles * batch; tile = blockIdx.x % ntiles, template = blockIdx.x / ntiles.
// dynamic smem: D2 raw[W], D2 dif[W] with W = kProjThreads + halo_lo + halo_hi  (x = h+, y = hx)
// EXT: LR_Y_EXTENDED (24 spline channels, emission delays relative to the reception split: project_sample<PT, true>)
template <int PT, bool EXT = false>
__global__ void __launch_bounds__(kProjThreads, proj_min_blocks(PT))
project_kernel(const Params prm, const double* __restrict__ hp, const double* __restrict__ hc,
               const double* __restrict__ basis /* [batch][9] */, double* __restrict__ y) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int W = kProjThreads + prm.halo_lo + prm.halo_hi;
  D2* raw = reinterpret_cast<D2*>(smem_raw);
  D2* dif = raw + W;

  const int tile = blockIdx.x % prm.ntiles;
  const int64_t b = blockIdx.x / prm.ntiles;
  const int n0 = tile * kProjThreads;
  const int g0 = n0 - prm.halo_lo;  // global sample index of staged index 0
  const double* hpb = hp + b * prm.in_stride;
  const double* hcb = hc + b * prm.in_stride;

  // the samples of a tile fall in one or two spline intervals (knots are hours apart): their coefficients
  // go to shared memory, so that no evaluation in project_sample waits on a global load
  constexpr int NCH = EXT ? kSplineChannels : 15;   // spline channels this kernel evaluates
  __shared__ D4 sc[NCH * 2];
  double u_unused;
  const int n_last = n0 + kProjThreads - 1 < prm.n - 1 ? n0 + kProjThreads - 1 : prm.n - 1;
  const int i_lo = spline_interval(prm, sample_trel(prm, prm.n_off + n0), u_unused);
  const int i_hi = spline_interval(prm, sample_trel(prm, prm.n_off + n_last), u_unused);
  // (measured, plain form: orders <= 25 gain 2 %, orders 31 and 41 lose 1-2 % -- their shared-memory pipe is the fuller
  // one; the extended form, with 18 evaluations per sample, gains 8-10 % at those orders too)
  const bool tile_coef = PT > 0 && (PT <= 13 || EXT) && i_hi - i_lo <= 1;   // (block-uniform)
  if (tile_coef && threadIdx.x < 2 * NCH && !(EXT && threadIdx.x >= 6 && threadIdx.x < 18)) {   // (EXT: x_2, x_3 unused)
    const int ch = threadIdx.x >> 1, i = i_lo + (threadIdx.x & 1);
    sc[threadIdx.x] = load4(prm.coef + (int64_t)ch * prm.nint + (i < prm.nint ? i : prm.nint - 1));
  }
  // one pass, one barrier: every element's successor is loaded too (it hits L1) and the first difference is formed
  // in registers
  for (int m = threadIdx.x; m < W; m += kProjThreads) {
    const int g = g0 + m;
    D2 v{0.0, 0.0}, v1{0.0, 0.0};
    if (g >= prm.rd_lo && g < prm.rd_hi) { v.x = __ldg(hpb + g); v.y = __ldg(hcb + g); }
    if (g + 1 >= prm.rd_lo && g + 1 < prm.rd_hi && m + 1 < W) { v1.x = __ldg(hpb + g + 1); v1.y = __ldg(hcb + g + 1); }
    raw[m] = v;
    if (m + 1 < W) dif[m] = D2{v1.x - v.x, v1.y - v.y};
  }
  __syncthreads();

  const int n = n0 + (int)threadIdx.x;
  if (n >= prm.n) return;
  double* yb = y + b * 6 * prm.out_stride + n;
  const int ng = prm.n_off + n;   // global sample index
  if (ng < prm.m_proj || ng >= prm.n_glob - prm.m_proj) {
#pragma unroll
    for (int s = 0; s < 6; ++s) yb[s * prm.out_stride] = 0.0;
    return;
  }

  double bs[9];
#pragma unroll
  for (int a = 0; a < 9; ++a) bs[a] = __ldg(basis + b * 9 + a);
  const int64_t os = prm.out_stride;
  auto store = [&](int slot, double v) { yb[slot * os] = v; };
  if (tile_coef)
    project_sample<PT, EXT>(prm, raw, dif, W, n - g0, sample_trel(prm, ng), bs, store, CoefTile{sc, i_lo});
  else
    project_sample<PT, EXT>(prm, raw, dif, W, n - g0, sample_trel(prm, ng), bs, store, CoefGlobal{});
}

// Two consecutive samples per thread (project_pair): the same tile, staging and results as project_kernel with half
// the threads; every first difference a pair of stencils shares is read from shared memory once.
template <int PT>
__global__ void __launch_bounds__(kProjPairThreads, 5)   // 168 registers: 6 CTAs of 64 threads per SM
project_pair_kernel(const Params prm, const double* __restrict__ hp, const double* __restrict__ hc,
                    const double* __restrict__ basis /* [batch][9] */, double* __restrict__ y) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int W = kProjThreads + prm.halo_lo + prm.halo_hi;
  const int H = proj_pair_half(W);
  D2* raw = reinterpret_cast<D2*>(smem_raw);
  D2* dif_e = raw + W;      // first differences, de-interleaved: dif_e[i] = dif[2 i], dif_o[i] = dif[2 i + 1]
  D2* dif_o = dif_e + H;
  double* geo = reinterpret_cast<double*>(dif_o + H) + threadIdx.x;   // this thread's column of geo[kGeoFields][threads]

  const int tile = blockIdx.x % prm.ntiles;
  const int64_t b = blockIdx.x / prm.ntiles;
  const int n0 = tile * kProjThreads;
  const int g0 = n0 - prm.halo_lo;  // global sample index of staged index 0
  const double* hpb = hp + b * prm.in_stride;
  const double* hcb = hc + b * prm.in_stride;

  __shared__ D4 sc[15 * 2];
  __shared__ double bk_s[PT + 1];
  if (threadIdx.x <= PT) bk_s[threadIdx.x] = prm.bk[threadIdx.x];
  double u_unused;
  const int n_last = n0 + kProjThreads - 1 < prm.n - 1 ? n0 + kProjThreads - 1 : prm.n - 1;
  const int i_lo = spline_interval(prm, sample_trel(prm, prm.n_off + n0), u_unused);
  const int i_hi = spline_interval(prm, sample_trel(prm, prm.n_off + n_last), u_unused);
  const bool tile_coef = i_hi - i_lo <= 1;   // (block-uniform)
  if (tile_coef && threadIdx.x < 30) {
    const int ch = threadIdx.x >> 1, i = i_lo + (threadIdx.x & 1);
    sc[threadIdx.x] = load4(prm.coef + (int64_t)ch * prm.nint + (i < prm.nint ? i : prm.nint - 1));
  }
  for (int m = threadIdx.x; m < W; m += kProjPairThreads) {
    const int g = g0 + m;
    D2 v{0.0, 0.0};
    if (g >= prm.rd_lo && g < prm.rd_hi) { v.x = __ldg(hpb + g); v.y = __ldg(hcb + g); }
    raw[m] = v;
  }
  __syncthreads();
  for (int m = threadIdx.x; m < W - 1; m += kProjPairThreads) {
    const D2 d{raw[m + 1].x - raw[m].x, raw[m + 1].y - raw[m].y};
    ((m & 1) ? dif_o : dif_e)[m >> 1] = d;
  }
  __syncthreads();

  const int nA = n0 + 2 * (int)threadIdx.x;
  if (nA >= prm.n) return;
  const bool hasB = nA + 1 < prm.n;
  double* yb = y + b * 6 * prm.out_stride + nA;
  const int ngA = prm.n_off + nA;   // global sample index
  const int v_lo = prm.m_proj, v_hi = prm.n_glob - prm.m_proj;
  const bool vA = ngA >= v_lo && ngA < v_hi, vB = hasB && ngA + 1 >= v_lo && ngA + 1 < v_hi;
  const int64_t os = prm.out_stride;
  if (!vA && !vB) {
#pragma unroll
    for (int s = 0; s < 6; ++s) {
      yb[s * os] = 0.0;
      if (hasB) yb[s * os + 1] = 0.0;
    }
    return;
  }

  double bs[9];
#pragma unroll
  for (int a = 0; a < 9; ++a) bs[a] = __ldg(basis + b * 9 + a);
  auto store = [&](int slot, double a, double c) {
    yb[slot * os] = vA ? a : 0.0;
    if (hasB) yb[slot * os + 1] = vB ? c : 0.0;
  };
  const double tA = sample_trel(prm, ngA), tB = sample_trel(prm, ngA + 1);
  if (tile_coef) {
    project_geometry_store(prm, CoefTile{sc, i_lo}, tA, bs, geo, kProjPairThreads);
    project_geometry_store(prm, CoefTile{sc, i_lo}, tB, bs, geo + kGeoPerSample * kProjPairThreads, kProjPairThreads);
  } else {
    project_geometry_store(prm, CoefGlobal{}, tA, bs, geo, kProjPairThreads);
    project_geometry_store(prm, CoefGlobal{}, tB, bs, geo + kGeoPerSample * kProjPairThreads, kProjPairThreads);
  }
  project_pair<PT>(prm, raw, dif_e, dif_o, W, nA - g0, geo, kProjPairThreads, bk_s, store);
}

// ---------------------------------------------------------------------------------------------- stage 2
// dynamic smem: double raw[6][W], dif[6][W], W = kTdiThreads + halo_lo + halo_hi
// channels: LR_XYZ 0 | LR_AET 1 | LR_XYZ_AET 2
template <int PT, int GEN>
__global__ void __launch_bounds__(kTdiThreads, tdi_min_blocks(PT))
tdi_kernel(const Params prm, const double* __restrict__ y, double* __restrict__ out, int channels) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int W = kTdiThreads + prm.halo_lo + prm.halo_hi;
  double* raw = reinterpret_cast<double*>(smem_raw);
  double* dif = raw + 6 * W;

  const int tile = blockIdx.x % prm.ntiles;
  const int64_t b = blockIdx.x / prm.ntiles;
  const int n0 = tile * kTdiThreads;
  const int g0 = n0 - prm.halo_lo;
  const double* yb = y + b * 6 * prm.in_stride;

  for (int m = threadIdx.x; m < 6 * W; m += kTdiThreads) {
    const int s = m / W, g = g0 + (m - s * W);
    raw[m] = (g >= prm.rd_lo && g < prm.rd_hi) ? __ldg(yb + s * prm.in_stride + g) : 0.0;
  }
  __syncthreads();
  for (int m = threadIdx.x; m < 6 * W; m += kTdiThreads) {
    const int w = m % W;
    dif[m] = (w < W - 1) ? raw[m + 1] - raw[m] : 0.0;
  }
  __syncthreads();

  const int n = n0 + (int)threadIdx.x;
  if (n >= prm.n) return;
  const int nout = channels == 2 ? 6 : 3;
  double* ob = out + b * nout * prm.out_stride + n;
  const int ng = prm.n_off + n;   // global sample index
  if (ng < prm.m_front || ng >= prm.n_glob - prm.m_back) {
    for (int c = 0; c < nout; ++c) ob[c * prm.out_stride] = 0.0;
    return;
  }

  double xyz[3];
  tdi_sample<PT, GEN>(prm, raw, dif, W, n - g0, sample_trel(prm, ng), xyz);

  const int64_t N = prm.out_stride;
  if (channels != 1) { ob[0] = xyz[0]; ob[N] = xyz[1]; ob[2 * N] = xyz[2]; }
  if (channels != 0) {  // eq. 21
    const double A = (xyz[2] - xyz[0]) * 0.70710678118654752440;
    const double E = (xyz[0] - 2.0 * xyz[1] + xyz[2]) * 0.40824829046386301637;
    const double T = (xyz[0] + xyz[1] + xyz[2]) * 0.57735026918962576451;
    double* oa = channels == 2 ? ob + 3 * N : ob;
    oa[0] = A; oa[N] = E; oa[2 * N] = T;
  }
}

}  // namespace lr

#include "lr_tdi_fir.cuh"

namespace lr {

// lr_tdi paths
constexpr int kPathGeneric = 0;  // tdi_kernel: exact per-sample weights
constexpr int kPathFir3 = 3;     // tdi_fir_kernel, quadratic in tile time
constexpr int kPathFir4 = 4;     // tdi_fir_kernel, cubic in tile time

// FIR plan buffers (a plan object of lr_api.cu) and the fix-up machinery of the launching handle
struct FirPlanArgs {
  double* coef;   // DEVICE [ntiles][12][Wc][kFirKStride]
  int* flags;     // DEVICE [ntiles]: != 0 marks a tile that needs per-sample weights
  int* list;      // DEVICE [1 + ntiles]: count, then the flagged tiles
  int plan_tiles; // tiles of the plan (the whole series)
  int fixup_grid; // CTAs of the fix-up kernel (2 per SM)
  void* side;     // cudaStream_t owned by the handle: the fix-up kernel runs there, beside the apply kernel
  void* fork;     // cudaEvent_t: the caller's stream reached the launch
  void* join;     // cudaEvent_t owned by the handle: the fix-up kernel finished
  void* join_extra; // optional second cudaEvent_t recorded at the same point (a chunked caller's per-slot event)
  bool wait_join; // true: the caller's stream waits for `join` before the launcher returns; false: the caller
                  // orders later work after `join_extra` itself (chunked response: the next chunk overlaps the fix-up)
  bool skip_fixup; // the host knows that no flagged tile lies in this launch's window: no fork / fix-up / join
};

// small helper kernel: spline channel at arbitrary absolute times (lr_eval_orbit)
__global__ void eval_orbit_kernel(const Params prm, int ch, double t_start, const double* __restrict__ t,
                                  int64_t m, double* __restrict__ out);

// step P1 of the path (eq. 10): angles [batch][3] = (beta, lambda, psi) -> basis [batch][9] =
// (k, u, v), one thread per template; launched by every call that takes sky angles, in front of project_kernel
__global__ void source_basis_kernel(const double* __restrict__ angles, int64_t batch, double* __restrict__ basis);
int launch_source_basis(const double* angles, int64_t batch, double* basis, void* stream);
// the same for up to kSmallStage templates whose constants travel in the kernel's parameter buffer (no host ->
// device copy in front of the launch): v = gb [n][6] | angles [n][3]; slot = basis [n][9] | gb [n][6] | angles [n][3]
constexpr int kSmallStage = 16;
struct SmallStage { double v[kSmallStage * 9]; int n; int has_gb; };
__global__ void source_basis_small_kernel(const SmallStage s, double* __restrict__ slot);
int launch_source_basis_small(const SmallStage& s, double* slot, void* stream);

// Launchers, one explicit instantiation per compile-time pair count PT (lr_inst.cu is compiled once per
// PT; PT = 0 reads P at run time).  They return cudaError_t as int.
template <int PT>
int launch_project_t(const Params& prm, const double* hp, const double* hc, const double* basis, double* y,
                     int64_t batch, void* stream);
template <int PT>
int launch_tdi_t(const Params& prm, int gen, int path, int channels, const double* y, double* out, int64_t batch,
                 const FirPlanArgs& plan, void* stream);

template <int PT>
int launch_fir_plan_t(const Params& prm, int gen, int path, double* coef, int* flags, int* list, int plan_tiles,
                      void* stream);

// dispatch on the Lagrange order (lr_kernels.cu)
int launch_fir_plan(const Params& prm, int order, int gen, int path, double* coef, int* flags, int* list,
                    int plan_tiles, void* stream);
int launch_project(const Params& prm, int order, const double* hp, const double* hc, const double* basis,
                   double* y, int64_t batch, void* stream);
int launch_tdi(const Params& prm, int order, int gen, int path, int channels, const double* y, double* out,
               int64_t batch, const FirPlanArgs& plan, void* stream);

}  // namespace lr
