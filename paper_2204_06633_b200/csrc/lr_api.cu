// lr_api.cu — host side of liblr: the C ABI of include/lr.h.
//
// lr_create fits the orbit splines on the host (long double) and uploads per-interval cubic coefficients;
// lr_project / lr_tdi marshal arguments and launch the kernels of lr_kernels.cuh on the caller's stream.
// There is no CPU compute path: without a CUDA device every computing call returns LR_ECUDA.
#include <cuda_runtime.h>
#include <cufft.h>
#include <math.h>
#include <stdint.h>
#include <string.h>

#include <atomic>
#include <cmath>
#include <new>
#include <vector>

#include "../../include/lr.h"
#include "lr_host.hpp"
#include "lr_kernels.cuh"

namespace lr {
extern std::atomic<int64_t> g_launches;
int launch_gb_waveform(const double* gb_dev, double t0, double dt, int64_t batch, int64_t first, int64_t count,
                       int64_t stride, double* hp, double* hc, void* stream);   // lr_waveform.cu
}

namespace {

constexpr int kSlots = 4;  // ring of staging buffers for the per-template source basis

struct Stage {
  double* host = nullptr;  // pinned
  double* dev = nullptr;
  int64_t cap = 0;         // templates
  cudaEvent_t done = nullptr;
  bool pending = false;
};

}  // namespace

// lr_tdi's FIR plan (lr_tdi_fir.cuh): a function of the orbits and the time grid only, not of y.  Read-only once
// built, reference counted: the private plan of a handle (rebuilt when the grid or an option changes) or a plan
// made by lr_plan_create that any number of handles on the same orbits attach to (never rebuilt).
struct lr_plan {
  std::atomic<int> refs{1};
  bool shared = false;                  // made by lr_plan_create: immutable
  double* coef = nullptr;
  int* flags = nullptr;                 // [2 * ntiles + 1]: flags, then count + list of flagged tiles
  size_t coef_cap = 0, flags_cap = 0;   // elements
  bool valid = false;
  // what the plan was built for
  uint64_t orbit_id = 0;
  int64_t n = 0;
  double t0 = 0, dt = 0;
  int order = 0, gen = 0, chain = 0, path = 0;
  int tiles = 0;                        // plan tiles (1 for constant light times)
  cudaEvent_t ready = nullptr;
  // host copy of the list of flagged tiles (count, then the tiles), fetched once behind the plan kernel: a launch
  // whose window holds no flagged tile needs no fork / fix-up kernel / join
  int* list_host = nullptr;             // pinned, [1 + list_cap]
  size_t list_cap = 0;
  cudaEvent_t list_ev = nullptr;
  std::atomic<int> list_state{0};       // 0 unknown | 1 copy in flight | 2 known
};

static void plan_unref(lr_plan* pl) {
  if (!pl || pl->refs.fetch_sub(1) != 1) return;
  if (pl->ready) cudaEventDestroy(pl->ready);
  if (pl->list_ev) cudaEventDestroy(pl->list_ev);
  if (pl->list_host) cudaFreeHost(pl->list_host);
  if (pl->coef) cudaFree(pl->coef);
  if (pl->flags) cudaFree(pl->flags);
  delete pl;
}

struct lr_handle {
  // configuration
  double dt = 0, t_start = 0, knot_dt = 0, t0 = 0;
  int64_t n_knots = 0;
  int order = 0, p = 0, gen = 2, chain = LR_CHAIN_NESTED, channels = LR_XYZ;
  double r_max = 0, l_max = 0;
  double max_ldot = 0;   // max |dL_ij/dt| over the table (dimensionless), from the spline
  bool const_ltt = false; // every light-time table is constant: lr_tdi's plan is one tile (NEXT-4)
  int tdi_path = -1;     // LR_OPT_TDI_PATH: -1 auto | 0 generic | 3 | 4
  int plan_cache = 1;    // LR_OPT_TDI_PLAN_CACHE
  int proj_path = LR_PROJ_AUTO;   // LR_OPT_PROJ_PATH
  int y_precision = LR_Y_EXTENDED;   // LR_OPT_Y_PRECISION
  int sm_count = 0;
  int64_t chunk_samples = 0;   // LR_OPT_CHUNK_SAMPLES: 0 = automatic
  int64_t fft_length = 0;      // LR_OPT_FFT_LENGTH: 0 = n (no zero padding)
  uint64_t orbit_id = 0;       // hash of the spline coefficients and the knot grid: which orbits a plan belongs to
  lr_plan* plan = nullptr;     // this handle's own plan (implicit cache)
  lr_plan* attached = nullptr; // a shared plan (lr_plan_attach), used whenever it matches the call
  // the fix-up kernel of the FIR path runs on a side stream of the handle, forked from / joined to the caller's
  cudaStream_t fix_side = nullptr;
  cudaEvent_t fix_fork = nullptr, fix_join = nullptr;
  cudaEvent_t last_join = nullptr;   // the event most recently recorded behind a fix-up kernel (it reads plan->flags)
  // LR_OPT_TDI_PLAN_CACHE = 0 rebuilds the plan once per API call, not once per chunk of a chunked call
  bool in_call = false, built_in_call = false;
  double bk[lr::kPMax + 1];
  // device state
  lr::D4* coef = nullptr;
  Stage stage[kSlots];
  int next_slot = 0;
  Stage graph_stage;     // the slot of launches captured into CUDA graphs: never reallocated, never used by direct calls
  // scratch of lr_response / lr_response_host: y of one chunk, and for the host variant two staging
  // buffers each for h and out plus the copy streams of the three-stage pipeline
  double* y_scr = nullptr; size_t y_cap = 0;        // elements
  double* h_buf = nullptr; size_t h_cap = 0;
  double* o_buf = nullptr; size_t o_cap = 0;
  cudaStream_t s_in = nullptr, s_out = nullptr;
  cudaEvent_t ev_in[2] = {nullptr, nullptr}, ev_comp[2] = {nullptr, nullptr}, ev_out[2] = {nullptr, nullptr};
  cudaEvent_t ev_fix[2] = {nullptr, nullptr};       // fix-up kernel of the chunk in y slot 0 / 1 finished
  // lr_loglike_gb: spectra of one template chunk, partial sums of the inner product, the cached FFT plan
  double* f_buf = nullptr; size_t f_cap = 0;
  double* ip_work = nullptr; size_t ip_cap = 0;
  cufftHandle fft = 0; int64_t fft_n = 0;
  cudaStream_t s_fft = nullptr;                     // transforms + inner product of chunk c beside the response of c+1
  cudaEvent_t ev_resp[2] = {nullptr, nullptr}, ev_fft[2] = {nullptr, nullptr};
  int last_cuda = 0;

  int64_t m_proj() const {
    return (int64_t)ceil((1.001 * r_max / lr::kC + 1.001 * l_max) / dt) + p + 2;
  }
  int64_t tdi_reach(int g) const { return (int64_t)ceil((double)(g == 1 ? 4 : 8) * 1.001 * l_max / dt); }
  int64_t m_front(int g) const { return m_proj() + tdi_reach(g) + p + 2; }
  int64_t m_back() const { return m_proj() + p + 2; }
};

namespace {

struct TdiShape { int path, wc, taps, halo_lo, halo_hi; };
TdiShape tdi_shape(const lr_handle* h);

#define LR_CUDA(h, call)                      \
  do {                                        \
    cudaError_t e__ = (call);                 \
    if (e__ != cudaSuccess) {                 \
      (h)->last_cuda = (int)e__;              \
      return LR_ECUDA;                        \
    }                                         \
  } while (0)

// Is the caller recording `st` into a CUDA graph?  lr_project and lr_tdi can be captured (a launch-bound loop of
// small calls replays as one graph launch): they then wait on no event recorded outside the capture and record none
// that the handle would wait on later.
bool capturing(cudaStream_t st) {
  cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
  return cudaStreamIsCapturing(st, &cs) == cudaSuccess && cs == cudaStreamCaptureStatusActive;
}
// Event queries and allocations are among the calls a thread may not make while a global-mode capture is active:
// this guard switches the calling thread to the relaxed mode for its lifetime.
struct RelaxedCapture {
  cudaStreamCaptureMode mode = cudaStreamCaptureModeRelaxed;
  RelaxedCapture() { (void)cudaThreadExchangeStreamCaptureMode(&mode); }
  ~RelaxedCapture() { (void)cudaThreadExchangeStreamCaptureMode(&mode); }
};
// an event recorded outside the capture must have completed already: a capture cannot wait for it
bool event_done(cudaEvent_t ev) {
  RelaxedCapture relaxed;
  const bool done = cudaEventQuery(ev) == cudaSuccess;
  if (!done) (void)cudaGetLastError();
  return done;
}

lr::Params make_params(const lr_handle* h, int64_t n) {
  lr::Params P;
  memset(&P, 0, sizeof(P));
  P.coef = h->coef;
  P.nint = (int)(h->n_knots - 1);
  P.p = h->p;
  P.trel0 = (double)((long double)h->t0 - (long double)h->t_start);
  P.dt = h->dt;
  P.inv_h = 1.0 / h->knot_dt;
  P.inv_dt = 1.0 / h->dt;
  P.inv_cdt = 1.0 / (lr::kC * h->dt);
  P.n = (int)n; P.n_off = 0; P.n_glob = (int)n;          // default window: the whole series
  P.rd_lo = 0; P.rd_hi = (int)n;
  P.in_stride = n; P.out_stride = n;
  P.m_proj = (int)h->m_proj();
  P.m_front = (int)h->m_front(h->gen);
  P.m_back = (int)h->m_back();
  P.chain_sum = h->chain == LR_CHAIN_SUM ? 1 : 0;
  P.proj_ext = h->y_precision == LR_Y_EXTENDED ? 1 : 0;
  P.proj_pair = h->proj_path == LR_PROJ_PAIR ? 1 : 0;   // LR_PROJ_AUTO: one sample per thread (the faster one)
  memcpy(P.bk, h->bk, sizeof(P.bk));
  return P;
}

bool size_ok(int64_t batch, int64_t n) {
  return batch >= 1 && n >= 1 && n < ((int64_t)1 << 31) - ((int64_t)1 << 20) &&
         batch <= (((int64_t)1 << 31) - 1) / ((n + 63) / 64);
}

// the times the kernels evaluate the splines at must lie inside the knot table (no extrapolation)
bool in_table(const lr_handle* h, int64_t n_first, int64_t n_last, double back_reach) {
  const long double span = (long double)(h->n_knots - 1) * h->knot_dt;
  const long double rel0 = (long double)h->t0 - (long double)h->t_start;
  const long double lo = rel0 + (long double)n_first * h->dt - back_reach;
  const long double hi = rel0 + (long double)n_last * h->dt;
  return lo >= 0 && hi <= span;
}

// Stages the per-template constants of one launch.  Host -> device: the sky angles [batch][3] = (beta, lambda, psi)
// and, when `gb` is given, the waveform parameters [batch][6]; source_basis_kernel then writes the source basis
// [batch][9] (step P1 of the path) on the caller's stream.  Device layout of a slot: basis | gb | angles.
int stage_basis(lr_handle* h, const double* beta, const double* lam, const double* psi, int64_t batch,
                cudaStream_t st, Stage** used, const double* gb = nullptr, const double** gb_dev = nullptr) {
  if (capturing(st)) {
    // graph capture: only the parameter-buffer path (the constants become part of the kernel node), into a slot of
    // its own that no direct call touches and that is never reallocated (the graph keeps its address).  Captured
    // launches of one stream are ordered, so they may share it.
    if (batch > lr::kSmallStage) return LR_EINVAL;
    Stage& G = h->graph_stage;
    if (!G.dev) {
      RelaxedCapture relaxed;   // (allocation is not a capturable call)
      LR_CUDA(h, cudaMalloc(&G.dev, (size_t)lr::kSmallStage * 18 * sizeof(double)));
      G.cap = lr::kSmallStage;
    }
    lr::SmallStage ss;
    memset(&ss, 0, sizeof(ss));
    ss.n = (int)batch; ss.has_gb = gb ? 1 : 0;
    if (gb) memcpy(ss.v, gb, (size_t)batch * 6 * sizeof(double));
    for (int64_t b = 0; b < batch; ++b) {
      ss.v[6 * batch + 3 * b] = beta[b]; ss.v[6 * batch + 3 * b + 1] = lam[b]; ss.v[6 * batch + 3 * b + 2] = psi[b];
    }
    LR_CUDA(h, (cudaError_t)lr::launch_source_basis_small(ss, G.dev, (void*)st));
    if (gb_dev) *gb_dev = G.dev + 9 * batch;
    *used = &G;
    return LR_OK;
  }
  Stage& S = h->stage[h->next_slot];
  h->next_slot = (h->next_slot + 1) % kSlots;
  if (!S.done) LR_CUDA(h, cudaEventCreateWithFlags(&S.done, cudaEventDisableTiming));
  if (S.pending) {
    // the slot's earlier users must be done with it: only a rewrite of the pinned host side needs the HOST to wait;
    // the small path (constants in the kernel's parameter buffer) orders the device side on the stream instead
    if (batch <= lr::kSmallStage && S.cap >= batch) LR_CUDA(h, cudaStreamWaitEvent(st, S.done, 0));
    else LR_CUDA(h, cudaEventSynchronize(S.done));
    S.pending = false;
  }
  if (S.cap < batch) {
    if (S.host) cudaFreeHost(S.host);
    if (S.dev) cudaFree(S.dev);
    S.host = nullptr; S.dev = nullptr; S.cap = 0;
    LR_CUDA(h, cudaMallocHost(&S.host, (size_t)batch * 9 * sizeof(double)));
    LR_CUDA(h, cudaMalloc(&S.dev, (size_t)batch * 18 * sizeof(double)));
    S.cap = batch;
  }
  double* dev_gb = S.dev + 9 * batch;
  double* dev_ang = S.dev + 15 * batch;
  if (batch <= lr::kSmallStage) {   // the constants travel in the kernel's parameter buffer: no copy in front of it
    lr::SmallStage ss;
    memset(&ss, 0, sizeof(ss));
    ss.n = (int)batch; ss.has_gb = gb ? 1 : 0;
    if (gb) memcpy(ss.v, gb, (size_t)batch * 6 * sizeof(double));
    for (int64_t b = 0; b < batch; ++b) {
      ss.v[6 * batch + 3 * b] = beta[b]; ss.v[6 * batch + 3 * b + 1] = lam[b]; ss.v[6 * batch + 3 * b + 2] = psi[b];
    }
    LR_CUDA(h, (cudaError_t)lr::launch_source_basis_small(ss, S.dev, (void*)st));
    if (gb_dev) *gb_dev = dev_gb;
    *used = &S;
    return LR_OK;
  }
  // host side of the slot: gb [batch][6] | angles [batch][3] (the order they have on the device)
  double* ang = S.host + 6 * batch;
  for (int64_t b = 0; b < batch; ++b) { ang[3 * b] = beta[b]; ang[3 * b + 1] = lam[b]; ang[3 * b + 2] = psi[b]; }
  if (gb) memcpy(S.host, gb, (size_t)batch * 6 * sizeof(double));
  if (gb)
    LR_CUDA(h, cudaMemcpyAsync(dev_gb, S.host, (size_t)batch * 9 * sizeof(double), cudaMemcpyHostToDevice, st));
  else
    LR_CUDA(h, cudaMemcpyAsync(dev_ang, ang, (size_t)batch * 3 * sizeof(double), cudaMemcpyHostToDevice, st));
  LR_CUDA(h, (cudaError_t)lr::launch_source_basis(dev_ang, batch, S.dev, (void*)st));
  if (gb_dev) *gb_dev = dev_gb;
  *used = &S;
  return LR_OK;
}

}  // namespace

extern "C" {

int lr_create(const lr_orbits* orb, double dt, int order, int tdi_gen, lr_handle** out) {
  if (!orb || !out || !orb->x || !orb->ltt) return LR_EINVAL;
  if (!(dt > 0) || !(orb->knot_dt > 0) || orb->n_knots < 4 || orb->n_knots > ((int64_t)1 << 30)) return LR_EINVAL;
  if (order < 1 || order > LR_MAX_ORDER || order % 2 == 0) return LR_EINVAL;
  if (tdi_gen != 1 && tdi_gen != 2) return LR_EINVAL;
  const int64_t nk = orb->n_knots;
  for (int64_t i = 0; i < 9 * nk; ++i)
    if (!isfinite(orb->x[i])) return LR_EINVAL;
  for (int64_t i = 0; i < 6 * nk; ++i)
    if (!isfinite(orb->ltt[i]) || orb->ltt[i] < 0) return LR_EINVAL;

  lr_handle* h = new (std::nothrow) lr_handle();
  if (!h) return LR_ENOMEM;
  h->dt = dt; h->t_start = orb->t_start; h->knot_dt = orb->knot_dt; h->t0 = orb->t_start;
  h->n_knots = nk; h->order = order; h->p = (order + 1) / 2; h->gen = tdi_gen;

  // table maxima for the margins (reading A8)
  for (int64_t k = 0; k < nk; ++k)
    for (int i = 0; i < 3; ++i) {
      double r = 0;
      for (int a = 0; a < 3; ++a) { const double v = orb->x[((int64_t)i * 3 + a) * nk + k]; r += v * v; }
      r = sqrt(r);
      if (r > h->r_max) h->r_max = r;
    }
  for (int64_t k = 0; k < 6 * nk; ++k)
    if (orb->ltt[k] > h->l_max) h->l_max = orb->ltt[k];

  lr::pair_constants(h->p, h->bk);
  h->const_ltt = true;
  for (int s = 0; s < 6 && h->const_ltt; ++s)
    for (int64_t k = 1; k < nk; ++k)
      if (orb->ltt[s * nk + k] != orb->ltt[s * nk]) { h->const_ltt = false; break; }

  std::vector<lr::D4> coef;
  try { coef.resize((size_t)lr::kSplineChannels * (nk - 1)); } catch (...) { delete h; return LR_ENOMEM; }
  try {
    for (int ch = 0; ch < 9; ++ch) lr::fit_channel(orb->x + (int64_t)ch * nk, nk, orb->knot_dt, coef.data() + (size_t)ch * (nk - 1));
    for (int s = 0; s < 6; ++s) lr::fit_channel(orb->ltt + (int64_t)s * nk, nk, orb->knot_dt, coef.data() + (size_t)(9 + s) * (nk - 1));
    // channels 15..23: the three arm vectors x_i - x_j (arm a joins spacecraft a and (a+1)%3), splined from the exact
    // differences of the table values.  The spline fit is linear in the table, so these ARE spline(x_i) - spline(x_j)
    // -- but evaluated without the rounding of two ~1.5e11 m positions (LR_Y_EXTENDED)
    std::vector<long double> dif((size_t)nk);
    for (int arm = 0; arm < 3; ++arm)
      for (int a = 0; a < 3; ++a) {
        const double* xi = orb->x + ((int64_t)arm * 3 + a) * nk;
        const double* xj = orb->x + ((int64_t)((arm + 1) % 3) * 3 + a) * nk;
        for (int64_t k = 0; k < nk; ++k) dif[(size_t)k] = (long double)xi[k] - (long double)xj[k];
        lr::fit_channel(dif.data(), nk, orb->knot_dt, coef.data() + (size_t)(15 + arm * 3 + a) * (nk - 1));
      }
  } catch (...) { delete h; return LR_ENOMEM; }

  // largest light-time rate of the table: decides whether lr_tdi may treat the delays of a tile as a
  // low-degree polynomial in time (lr_tdi_fir.cuh)
  for (int s = 0; s < 6; ++s)
    for (int64_t i = 0; i + 1 < nk; ++i) {
      const lr::D4& c = coef[(size_t)(9 + s) * (nk - 1) + i];
      double m = fmax(fabs(c.y), fabs(c.y + 2.0 * c.z + 3.0 * c.w));
      if (c.w != 0.0) {
        const double u = -c.z / (3.0 * c.w);
        if (u > 0.0 && u < 1.0) m = fmax(m, fabs(c.y + u * (2.0 * c.z + 3.0 * c.w * u)));
      }
      h->max_ldot = fmax(h->max_ldot, m / orb->knot_dt);
    }

  {  // FNV-1a over the coefficients and the knot grid
    uint64_t id = 1469598103934665603ull;
    auto mix = [&](const void* p, size_t bytes) {
      const unsigned char* c = static_cast<const unsigned char*>(p);
      for (size_t i = 0; i < bytes; ++i) { id ^= c[i]; id *= 1099511628211ull; }
    };
    mix(coef.data(), coef.size() * sizeof(lr::D4));
    mix(&h->n_knots, sizeof(h->n_knots)); mix(&h->t_start, sizeof(h->t_start)); mix(&h->knot_dt, sizeof(h->knot_dt));
    h->orbit_id = id;
  }
  cudaError_t e = cudaMalloc(&h->coef, coef.size() * sizeof(lr::D4));
  if (e == cudaSuccess) e = cudaMemcpy(h->coef, coef.data(), coef.size() * sizeof(lr::D4), cudaMemcpyHostToDevice);
  if (e != cudaSuccess) {
    if (h->coef) cudaFree(h->coef);
    delete h;
    *out = nullptr;
    return LR_ECUDA;
  }
  *out = h;
  return LR_OK;
}

void lr_destroy(lr_handle* h) {
  if (!h) return;
  if (h->graph_stage.dev) cudaFree(h->graph_stage.dev);
  for (int s = 0; s < kSlots; ++s) {
    Stage& S = h->stage[s];
    if (S.pending) cudaEventSynchronize(S.done);
    if (S.done) cudaEventDestroy(S.done);
    if (S.host) cudaFreeHost(S.host);
    if (S.dev) cudaFree(S.dev);
  }
  if (h->fix_fork) cudaEventDestroy(h->fix_fork);
  if (h->fix_join) cudaEventDestroy(h->fix_join);
  if (h->fix_side) cudaStreamDestroy(h->fix_side);
  plan_unref(h->plan);
  plan_unref(h->attached);
  if (h->y_scr) cudaFree(h->y_scr);
  if (h->h_buf) cudaFree(h->h_buf);
  if (h->o_buf) cudaFree(h->o_buf);
  if (h->f_buf) cudaFree(h->f_buf);
  if (h->ip_work) cudaFree(h->ip_work);
  if (h->fft_n) cufftDestroy(h->fft);
  for (int i = 0; i < 2; ++i) {
    if (h->ev_in[i]) cudaEventDestroy(h->ev_in[i]);
    if (h->ev_comp[i]) cudaEventDestroy(h->ev_comp[i]);
    if (h->ev_out[i]) cudaEventDestroy(h->ev_out[i]);
    if (h->ev_fix[i]) cudaEventDestroy(h->ev_fix[i]);
    if (h->ev_resp[i]) cudaEventDestroy(h->ev_resp[i]);
    if (h->ev_fft[i]) cudaEventDestroy(h->ev_fft[i]);
  }
  if (h->s_fft) cudaStreamDestroy(h->s_fft);
  if (h->s_in) cudaStreamDestroy(h->s_in);
  if (h->s_out) cudaStreamDestroy(h->s_out);
  if (h->coef) cudaFree(h->coef);
  delete h;
}

int lr_set_option(lr_handle* h, int key, double value) {
  if (!h || !isfinite(value)) return LR_EINVAL;
  switch (key) {
    case LR_OPT_T0: h->t0 = value; return LR_OK;
    case LR_OPT_CHAIN:
      if (value != LR_CHAIN_NESTED && value != LR_CHAIN_SUM) return LR_EINVAL;
      h->chain = (int)value; return LR_OK;
    case LR_OPT_CHANNELS:
      if (value != LR_XYZ && value != LR_AET && value != LR_XYZ_AET) return LR_EINVAL;
      h->channels = (int)value; return LR_OK;
    case LR_OPT_TDI_GEN:
      if (value != 1 && value != 2) return LR_EINVAL;
      h->gen = (int)value; return LR_OK;
    case LR_OPT_TDI_PATH:
      if (value != LR_TDI_AUTO && value != LR_TDI_PER_SAMPLE && value != LR_TDI_FIR3 && value != LR_TDI_FIR4)
        return LR_EINVAL;
      h->tdi_path = (int)value; return LR_OK;
    case LR_OPT_Y_PRECISION:
      if (value != LR_Y_PLAIN && value != LR_Y_EXTENDED) return LR_EINVAL;
      h->y_precision = (int)value; return LR_OK;
    case LR_OPT_PROJ_PATH:
      if (value != LR_PROJ_AUTO && value != LR_PROJ_SINGLE && value != LR_PROJ_PAIR) return LR_EINVAL;
      h->proj_path = (int)value; return LR_OK;
    case LR_OPT_CHUNK_SAMPLES:
      if (value < 0 || value > 2147483647.0 || value != floor(value)) return LR_EINVAL;
      h->chunk_samples = (int64_t)value; return LR_OK;
    case LR_OPT_FFT_LENGTH:
      if (value < 0 || value > 2147483647.0 || value != floor(value)) return LR_EINVAL;
      h->fft_length = (int64_t)value; return LR_OK;
    case LR_OPT_TDI_PLAN_CACHE:
      if (value != 0 && value != 1) return LR_EINVAL;
      h->plan_cache = (int)value; if (h->plan) h->plan->valid = false; return LR_OK;
    default: return LR_EINVAL;
  }
}

int lr_get_option(const lr_handle* h, int key, double* value) {
  if (!h || !value) return LR_EINVAL;
  switch (key) {
    case LR_OPT_T0: *value = h->t0; return LR_OK;
    case LR_OPT_CHAIN: *value = h->chain; return LR_OK;
    case LR_OPT_CHANNELS: *value = h->channels; return LR_OK;
    case LR_OPT_TDI_GEN: *value = h->gen; return LR_OK;
    case LR_OPT_TDI_PATH: *value = h->tdi_path; return LR_OK;
    case LR_OPT_PROJ_PATH: *value = h->proj_path; return LR_OK;
    case LR_OPT_Y_PRECISION: *value = h->y_precision; return LR_OK;
    case LR_OPT_CHUNK_SAMPLES: *value = (double)h->chunk_samples; return LR_OK;
    case LR_OPT_FFT_LENGTH: *value = (double)h->fft_length; return LR_OK;
    case LR_OPT_TDI_PLAN_CACHE: *value = h->plan_cache; return LR_OK;
    case LR_INFO_TDI_PATH: *value = tdi_shape(h).path; return LR_OK;
    case LR_INFO_FIR_TAPS: *value = tdi_shape(h).taps; return LR_OK;
    case LR_INFO_FIR_POWERS: {
      const TdiShape t = tdi_shape(h);
      *value = t.path == LR_TDI_PER_SAMPLE ? 0 : h->const_ltt ? 1 : t.path == LR_TDI_FIR4 ? 4 : 3;
      return LR_OK;
    }
    default: return LR_EINVAL;
  }
}

int lr_get_margins(const lr_handle* h, int64_t* m_proj, int64_t* m_front, int64_t* m_back) {
  if (!h) return LR_EINVAL;
  if (m_proj) *m_proj = h->m_proj();
  if (m_front) *m_front = h->m_front(h->gen);
  if (m_back) *m_back = h->m_back();
  return LR_OK;
}

}  // extern "C"

namespace {

// A launch window: the kernels process global samples [off, off + n) of a series of n_glob samples; `in`
// points at the input row element of global sample `off` and may be read for global samples
// [rd_a, rd_b); rows of the input / output arrays are in_stride / out_stride elements apart.
struct Window {
  int64_t n_glob, off, n, rd_a, rd_b, in_stride, out_stride;
};

void apply_window(lr::Params& P, const Window& w) {
  P.n = (int)w.n; P.n_off = (int)w.off; P.n_glob = (int)w.n_glob;
  P.rd_lo = (int)(w.rd_a - w.off); P.rd_hi = (int)(w.rd_b - w.off);
  P.in_stride = w.in_stride; P.out_stride = w.out_stride;
}

int project_window(lr_handle* h, const double* hp, const double* hc, const double* basis_dev, int64_t batch,
                   const Window& w, double* y, void* stream) {
  lr::Params P = make_params(h, w.n_glob);
  apply_window(P, w);
  const int64_t mp = h->m_proj();
  P.halo_lo = (int)mp; P.halo_hi = (int)mp;
  P.ntiles = (int)((w.n + lr::kProjThreads - 1) / lr::kProjThreads);
  const int e = lr::launch_project(P, h->order, hp, hc, basis_dev, y, batch, stream);
  if (e != 0) { h->last_cuda = e; return LR_ECUDA; }
  return LR_OK;
}

// which lr_tdi path this handle takes, and the staged halo of that path's kernels

TdiShape tdi_shape(const lr_handle* h) {
  TdiShape t{h->tdi_path, 0, 0, 0, 0};
  const int64_t mf = h->m_front(h->gen);
  // per-tile polynomial FIR when the delays drift slowly enough, else exact per-sample weights
  const int nlinks = h->gen == 1 ? 3 : 7;  // links in the longest delayed term
  const double de = (double)nlinks * h->max_ldot * (double)lr::kFirTile;  // change of eps over one tile
  if (t.path == LR_TDI_AUTO) t.path = de <= 6e-6 ? LR_TDI_FIR3 : de <= 1.5e-4 ? LR_TDI_FIR4 : LR_TDI_PER_SAMPLE;
  if (t.path != LR_TDI_PER_SAMPLE) {
    const int imax = (int)h->tdi_reach(h->gen);
    t.taps = imax + 2 * h->p - 2;
    t.wc = ((t.taps + lr::kFirR - 1) / lr::kFirR) * lr::kFirR;
    const int back = t.wc - (h->p - 1);
    t.halo_lo = back > (int)(mf - h->m_proj()) ? back : (int)(mf - h->m_proj());
    t.halo_hi = h->p + lr::kFirR;
    // very long stencils: keep the per-sample kernel
    const int Wst = lr::kFirTile + t.halo_lo + t.halo_hi;
    if ((t.path == LR_TDI_FIR4 && !h->const_ltt ? lr::fir_mma_smem_bytes(Wst, t.wc) : lr::fir_apply_smem_bytes(Wst, t.wc)) >
        200 * 1024)
      t.path = LR_TDI_PER_SAMPLE;
  }
  if (t.path == LR_TDI_PER_SAMPLE) {
    t.wc = 0;
    t.halo_lo = (int)(mf - h->m_proj());
    t.halo_hi = h->p + 2;
  }
  return t;
}

bool plan_matches(const lr_plan* pl, const lr_handle* h, int64_t n_glob, int path) {
  return pl && pl->valid && pl->orbit_id == h->orbit_id && pl->n == n_glob && pl->t0 == h->t0 && pl->dt == h->dt &&
         pl->order == h->order && pl->gen == h->gen && pl->chain == h->chain && pl->path == path;
}

// FIR-path fields of the kernel parameters that do not depend on the launch window
void fir_params(const lr_handle* h, const TdiShape& ts, int64_t n_glob, lr::Params& P) {
  P.halo_lo = ts.halo_lo; P.halo_hi = ts.halo_hi; P.fir_wc = ts.wc; P.fir_taps = ts.taps;
  // the plan covers the whole series (global tiles); with constant light times every tile has the same
  // filters, so the plan is ONE tile (the constant-delay fast path of SURVEY.md §8(f) NEXT-4)
  const bool uniform = h->const_ltt;
  P.fir_uniform = uniform ? 1 : 0;
  P.fir_tile0 = uniform ? (int)(h->m_front(h->gen) / lr::kFirTile) : 0;
  P.ntiles = uniform ? 1 : (int)((n_glob + lr::kFirTile - 1) / lr::kFirTile);
}

// (Re)build `pl` for this handle's grid and options on `st`.  wait_list: block until the list of flagged tiles
// is on the host (lr_plan_create: the plan is then complete and immutable when the call returns).
int build_plan(lr_handle* h, lr_plan* pl, const TdiShape& ts, int64_t n_glob, cudaStream_t st, bool wait_list) {
  lr::Params P = make_params(h, n_glob);
  fir_params(h, ts, n_glob, P);
  const size_t need = (size_t)P.ntiles * lr::fir_plan_doubles_per_tile(P.fir_wc);
  pl->valid = false;
  pl->list_state = 0;
  if (pl->coef_cap < need) {
    if (pl->coef) { cudaFree(pl->coef); pl->coef = nullptr; pl->coef_cap = 0; }
    LR_CUDA(h, cudaMalloc(&pl->coef, need * sizeof(double)));
    pl->coef_cap = need;
  }
  if (pl->flags_cap < (size_t)P.ntiles) {
    if (pl->flags) { cudaFree(pl->flags); pl->flags = nullptr; pl->flags_cap = 0; }
    LR_CUDA(h, cudaMalloc(&pl->flags, (2 * (size_t)P.ntiles + 1) * sizeof(int)));
    pl->flags_cap = (size_t)P.ntiles;
  }
  if (!pl->ready) LR_CUDA(h, cudaEventCreateWithFlags(&pl->ready, cudaEventDisableTiming));
  // a fix-up kernel of an earlier launch may still be reading the list this build rewrites
  if (h->last_join) LR_CUDA(h, cudaStreamWaitEvent(st, h->last_join, 0));
  int* list = pl->flags + P.ntiles;
  const int e = lr::launch_fir_plan(P, h->order, h->gen, ts.path, pl->coef, pl->flags, list, P.ntiles, (void*)st);
  if (e != 0) { h->last_cuda = e; return LR_ECUDA; }
  LR_CUDA(h, cudaEventRecord(pl->ready, st));
  pl->orbit_id = h->orbit_id; pl->n = n_glob; pl->t0 = h->t0; pl->dt = h->dt; pl->order = h->order;
  pl->gen = h->gen; pl->chain = h->chain; pl->path = ts.path; pl->tiles = P.ntiles;
  pl->valid = true;
  // the list of flagged tiles comes to the host behind the plan kernel (no synchronisation unless asked: a later
  // call that finds the copy finished uses it, until then every launch runs the fix-up kernel)
  const size_t words = 1 + (size_t)P.ntiles;
  if (pl->list_cap < words) {
    if (pl->list_host) { cudaFreeHost(pl->list_host); pl->list_host = nullptr; pl->list_cap = 0; }
    if (cudaMallocHost(&pl->list_host, words * sizeof(int)) == cudaSuccess) pl->list_cap = words;
    else (void)cudaGetLastError();
  }
  if (!pl->list_ev && cudaEventCreateWithFlags(&pl->list_ev, cudaEventDisableTiming) != cudaSuccess) {
    pl->list_ev = nullptr;
    (void)cudaGetLastError();
  }
  if (pl->list_cap >= words && pl->list_ev) {
    LR_CUDA(h, cudaMemcpyAsync(pl->list_host, list, words * sizeof(int), cudaMemcpyDeviceToHost, st));
    LR_CUDA(h, cudaEventRecord(pl->list_ev, st));
    pl->list_state = 1;
    if (wait_list) {
      LR_CUDA(h, cudaEventSynchronize(pl->list_ev));
      pl->list_state = 2;
    }
  }
  return LR_OK;
}

// With LR_OPT_TDI_PLAN_CACHE = 0 the plan is rebuilt once per API call (before its first launch), not once per
// chunk of a chunked call: the entry points open a PlanCall on the TDI handle.
struct PlanCall {
  lr_handle* h; bool outer;
  explicit PlanCall(lr_handle* h_) : h(h_), outer(h_ && !h_->in_call) { if (outer) { h->in_call = true; h->built_in_call = false; } }
  ~PlanCall() { if (outer) h->in_call = false; }
};

// join_later: if non-null and the FIR path runs, the fix-up kernel's completion is recorded there and the
// caller's stream does NOT wait for it (set to nullptr by the per-sample path, which has no fix-up kernel).
int tdi_window(lr_handle* h, const double* y, int64_t batch, const Window& w, double* out, void* stream,
               cudaEvent_t* join_later = nullptr) {
  lr::Params P = make_params(h, w.n_glob);
  const TdiShape ts = tdi_shape(h);
  const int path = ts.path;
  cudaStream_t st = (cudaStream_t)stream;
  lr::FirPlanArgs pa{};
  pa.wait_join = true;
  P.halo_lo = ts.halo_lo; P.halo_hi = ts.halo_hi; P.fir_wc = ts.wc; P.fir_taps = ts.taps;
  if (path != LR_TDI_PER_SAMPLE) {
    if (w.off % lr::kFirTile != 0) return LR_EINVAL;   // windows of the FIR path start on a tile
    fir_params(h, ts, w.n_glob, P);
    const bool uniform = h->const_ltt;
    // which plan: a shared one that fits this call, else the handle's own (built on first use, kept while it fits)
    lr_plan* pl = plan_matches(h->attached, h, w.n_glob, path) ? h->attached : nullptr;
    if (!pl) {
      if (!h->plan) {
        h->plan = new (std::nothrow) lr_plan();
        if (!h->plan) return LR_ENOMEM;
      }
      pl = h->plan;
      const bool fresh = h->plan_cache || (h->in_call && h->built_in_call);
      if (!(fresh && plan_matches(pl, h, w.n_glob, path))) {
        if (capturing(st)) return LR_EINVAL;   // build the plan with one call outside the capture first
        const int rc = build_plan(h, pl, ts, w.n_glob, st, false);
        if (rc != LR_OK) return rc;
        h->built_in_call = true;
      }
    }
    if (capturing(st)) {
      if (!event_done(pl->ready)) return LR_EINVAL;      // (a capture cannot wait for work outside it)
    } else {
      LR_CUDA(h, cudaStreamWaitEvent(st, pl->ready, 0));   // the plan may have been built on another stream
    }
    pa.coef = pl->coef; pa.flags = pl->flags; pa.list = pl->flags + P.ntiles;
    pa.plan_tiles = P.ntiles;
    if (h->sm_count == 0) {
      int dev = 0;
      LR_CUDA(h, cudaGetDevice(&dev));
      LR_CUDA(h, cudaDeviceGetAttribute(&h->sm_count, cudaDevAttrMultiProcessorCount, dev));
    }
    pa.fixup_grid = 2 * h->sm_count;
    if (!h->fix_side) {
      // highest priority: the side stream starts a few microseconds behind the apply kernel (it waits for the fork
      // event), by which time the apply kernel's CTAs hold every SM; at equal priority the fix-up CTAs were only
      // dispatched once the apply grid had drained and became a 40 us tail of every lr_tdi call
      int prio_lo = 0, prio_hi = 0;
      LR_CUDA(h, cudaDeviceGetStreamPriorityRange(&prio_lo, &prio_hi));
      LR_CUDA(h, cudaStreamCreateWithPriority(&h->fix_side, cudaStreamNonBlocking, prio_hi));
      LR_CUDA(h, cudaEventCreateWithFlags(&h->fix_fork, cudaEventDisableTiming));
      LR_CUDA(h, cudaEventCreateWithFlags(&h->fix_join, cudaEventDisableTiming));
    }
    pa.side = h->fix_side; pa.fork = h->fix_fork; pa.join = h->fix_join;
    if (pl->list_state.load() == 1 && event_done(pl->list_ev)) pl->list_state = 2;
    if (pl->list_state.load() == 2) {
      const int cnt = pl->list_host[0];
      bool any = cnt > 0 && uniform;   // (one-tile plan: a flagged plan tile concerns every window)
      if (cnt > 0 && !uniform) {
        const int64_t t_lo = w.off / lr::kFirTile, t_hi = t_lo + (w.n + lr::kFirTile - 1) / lr::kFirTile;
        for (int i = 1; i <= cnt && !any; ++i) any = pl->list_host[i] >= t_lo && pl->list_host[i] < t_hi;
      }
      pa.skip_fixup = !any;
    }
    if (join_later) {
      if (pa.skip_fixup) *join_later = nullptr;   // nothing to wait for
      else { pa.join_extra = *join_later; pa.wait_join = false; }
    }
    if (!pa.skip_fixup && !capturing(st)) h->last_join = h->fix_join;
    apply_window(P, w);
    P.ntiles = (int)((w.n + lr::kFirTile - 1) / lr::kFirTile);
  } else {
    if (join_later) *join_later = nullptr;
    apply_window(P, w);
    P.ntiles = (int)((w.n + lr::kTdiThreads - 1) / lr::kTdiThreads);
  }
  const int e = lr::launch_tdi(P, h->order, h->gen, path, h->channels, y, out, batch, pa, stream);
  if (e != 0) { h->last_cuda = e; return LR_ECUDA; }
  return LR_OK;
}

int check_project(const lr_handle* h, int64_t batch, int64_t n) {
  if (!size_ok(batch, n) || n <= 2 * h->m_proj()) return LR_EINVAL;
  const int64_t mp = h->m_proj();
  return in_table(h, mp, n - mp - 1, 0.0) ? LR_OK : LR_ERANGE;
}

int check_tdi(const lr_handle* h, int64_t batch, int64_t n) {
  const int64_t mf = h->m_front(h->gen), mb = h->m_back();
  if (!size_ok(batch, n) || n <= mf + mb) return LR_EINVAL;
  const double reach = (double)(h->gen == 1 ? 4 : 8) * 1.001 * h->l_max;
  return in_table(h, mf, n - mb - 1, reach) ? LR_OK : LR_ERANGE;
}

}  // namespace

extern "C" {

int lr_project(lr_handle* h, const double* hp, const double* hc, const double* beta, const double* lam,
               const double* psi, int64_t batch, int64_t n, double* y, void* stream) {
  if (!h || !hp || !hc || !beta || !lam || !psi || !y) return LR_EINVAL;
  int rc = check_project(h, batch, n);
  if (rc != LR_OK) return rc;
  cudaStream_t st = (cudaStream_t)stream;
  Stage* S = nullptr;
  rc = stage_basis(h, beta, lam, psi, batch, st, &S);
  if (rc != LR_OK) return rc;
  const Window w{n, 0, n, 0, n, n, n};
  rc = project_window(h, hp, hc, S->dev, batch, w, y, stream);
  if (rc != LR_OK) return rc;
  if (!capturing(st)) {   // (a captured event could not be waited for by a later call)
    LR_CUDA(h, cudaEventRecord(S->done, st));
    S->pending = true;
  }
  return LR_OK;
}

int lr_tdi(lr_handle* h, const double* y, int64_t batch, int64_t n, double* out, void* stream) {
  if (!h || !y || !out) return LR_EINVAL;
  const int rc = check_tdi(h, batch, n);
  if (rc != LR_OK) return rc;
  const Window w{n, 0, n, 0, n, n, n};
  PlanCall call(h);
  return tdi_window(h, y, batch, w, out, stream);
}

}  // extern "C"

namespace {

constexpr int64_t gcd_(int64_t a, int64_t b) { return b == 0 ? a : gcd_(b, a % b); }
constexpr int64_t lcm_(int64_t a, int64_t b) { return a / gcd_(a, b) * b; }
// chunks of the one-call response start on a tile of every kernel: lcm of the tile sizes (128, 224, 256) = 1792
constexpr int64_t kChunkUnit = lcm_(lcm_(lr::kProjThreads, lr::kTdiThreads), lr::kFirTile);
// y of one chunk: longer chunks mean fewer kernel tails (one year: 0.88 ms at 40 MB, 0.83 ms in one chunk); L2
// residency of y buys nothing, the kernels are bound by FP64 issue.  Two slots of this size per handle at most.
constexpr int64_t kYSlotBytes = (int64_t)1024 << 20;

int ensure(lr_handle* h, double** buf, size_t* cap, size_t need) {
  if (*cap >= need) return LR_OK;
  if (*buf) { cudaFree(*buf); *buf = nullptr; *cap = 0; }
  LR_CUDA(h, cudaMalloc(buf, need * sizeof(double)));
  *cap = need;
  return LR_OK;
}

// One (template chunk, time chunk) of the two-stage path through the y scratch.  hp/hc: DEVICE rows of
// stride h_stride whose element 0 is global sample h_a and that hold global samples [h_a, h_b).
// out_chunk: DEVICE rows of stride o_stride whose element 0 is global sample a.
int response_chunk(lr_handle* hp_, lr_handle* ht_, const TdiShape& ts, const double* hp, const double* hc,
                   int64_t h_a, int64_t h_b, int64_t h_stride, const double* basis_dev, int64_t nb, int64_t n,
                   int64_t a, int64_t b, int64_t ly, double* out_chunk, int64_t o_stride, void* stream,
                   double* y_slot, cudaEvent_t* fix_done) {
  const int64_t ya = a - ts.halo_lo > 0 ? a - ts.halo_lo : 0;
  const int64_t yb = b + ts.halo_hi < n ? b + ts.halo_hi : n;
  const Window wp{n, ya, yb - ya, h_a, h_b, h_stride, ly};
  int rc = project_window(hp_, hp + (ya - h_a), hc + (ya - h_a), basis_dev, nb, wp, y_slot, stream);
  if (rc != LR_OK) return rc;
  const Window wt{n, a, b - a, ya, yb, ly, o_stride};
  rc = tdi_window(ht_, y_slot + (a - ya), nb, wt, out_chunk, stream, fix_done);
  if (rc != LR_OK) hp_->last_cuda = ht_->last_cuda;
  return rc;
}

// the two y slots alternate between chunks; a slot is rewritten only after the fix-up kernel that read it
int ensure_fix_events(lr_handle* h) {
  for (int i = 0; i < 2; ++i)
    if (!h->ev_fix[i]) LR_CUDA(h, cudaEventCreateWithFlags(&h->ev_fix[i], cudaEventDisableTiming));
  return LR_OK;
}

int64_t round_up(int64_t v, int64_t u) { return (v + u - 1) / u * u; }

}  // namespace

extern "C" {

int lr_get_span_halo(const lr_handle* hp_, const lr_handle* ht_, int64_t* lo, int64_t* hi, int64_t* unit) {
  if (!hp_ || !ht_) return LR_EINVAL;
  const TdiShape ts = tdi_shape(ht_);
  if (lo) *lo = ts.halo_lo + hp_->m_proj();
  if (hi) *hi = ts.halo_hi + hp_->m_proj();
  if (unit) *unit = kChunkUnit;
  return LR_OK;
}

int lr_response_span(lr_handle* hp_, lr_handle* ht_, const double* h_plus, const double* h_cross, int64_t h_first,
                     int64_t h_len, const double* beta, const double* lam, const double* psi, int64_t batch,
                     int64_t n, int64_t first, int64_t count, double* out, void* stream) {
  lr_handle* h = hp_;
  if (!h || !ht_ || !h_plus || !h_cross || !beta || !lam || !psi || !out) return LR_EINVAL;
  if (capturing((cudaStream_t)stream)) return LR_EINVAL;   // only lr_project and lr_tdi can be captured into a graph
  int rc = check_project(h, batch, n);
  if (rc == LR_OK) rc = check_tdi(ht_, batch, n);
  if (rc != LR_OK) return rc;
  const TdiShape ts = tdi_shape(ht_);
  const int64_t mp = h->m_proj();
  if (first < 0 || count < 1 || first + count > n || first % kChunkUnit != 0) return LR_EINVAL;
  if (h_first < 0 || h_len < 1 || h_first + h_len > n) return LR_EINVAL;
  // the h slice must hold every sample the span's kernels read: [first - halo_lo - m_proj, first+count+halo_hi+m_proj)
  const int64_t need_a = first - ts.halo_lo - mp > 0 ? first - ts.halo_lo - mp : 0;
  const int64_t need_b = first + count + ts.halo_hi + mp < n ? first + count + ts.halo_hi + mp : n;
  if (h_first > need_a || h_first + h_len < need_b) return LR_EINVAL;
  PlanCall call(ht_);
  cudaStream_t st = (cudaStream_t)stream;
  const int nout = ht_->channels == LR_XYZ_AET ? 6 : 3;
  // y of one chunk bounds the footprint: no [batch][6][n] buffer
  const int64_t bc = batch < 8 ? batch : 8;
  const int64_t budget = kYSlotBytes / (bc * 6 * (int64_t)sizeof(double));
  int64_t lc = budget / kChunkUnit * kChunkUnit;
  if (lc < 4 * kChunkUnit) lc = 4 * kChunkUnit;
  if (h->chunk_samples > 0) lc = round_up(h->chunk_samples, kChunkUnit);
  if (lc > round_up(count, kChunkUnit)) lc = round_up(count, kChunkUnit);
  const int64_t ly = round_up(lc + ts.halo_lo + ts.halo_hi, 2);
  rc = ensure(h, &h->y_scr, &h->y_cap, (size_t)(2 * bc * 6 * ly));
  if (rc == LR_OK) rc = ensure_fix_events(h);
  if (rc != LR_OK) return rc;
  cudaEvent_t pending[2] = {nullptr, nullptr};   // fix-up kernels still reading y slot 0 / 1
  int64_t c = 0;
  for (int64_t b0 = 0; b0 < batch; b0 += bc) {
    const int64_t nb = batch - b0 < bc ? batch - b0 : bc;
    Stage* S = nullptr;
    rc = stage_basis(h, beta + b0, lam + b0, psi + b0, nb, st, &S);
    if (rc != LR_OK) return rc;
    for (int64_t a = first; a < first + count; a += lc, ++c) {
      const int slot = (int)(c & 1);
      const int64_t b = a + lc < first + count ? a + lc : first + count;
      if (pending[slot]) LR_CUDA(h, cudaStreamWaitEvent(st, pending[slot], 0));
      pending[slot] = h->ev_fix[slot];
      rc = response_chunk(h, ht_, ts, h_plus + b0 * h_len, h_cross + b0 * h_len, h_first, h_first + h_len, h_len,
                          S->dev, nb, n, a, b, ly, out + b0 * nout * count + (a - first), count, stream,
                          h->y_scr + (size_t)slot * bc * 6 * ly, &pending[slot]);
      if (rc != LR_OK) return rc;
    }
    LR_CUDA(h, cudaEventRecord(S->done, st));
    S->pending = true;
  }
  for (int i = 0; i < 2; ++i)   // join the last fix-up kernels
    if (pending[i]) LR_CUDA(h, cudaStreamWaitEvent(st, pending[i], 0));
  return LR_OK;
}

int lr_response(lr_handle* hp_, lr_handle* ht_, const double* h_plus, const double* h_cross, const double* beta,
                const double* lam, const double* psi, int64_t batch, int64_t n, double* out, void* stream) {
  return lr_response_span(hp_, ht_, h_plus, h_cross, 0, n, beta, lam, psi, batch, n, 0, n, out, stream);
}

int lr_response_host(lr_handle* hp_, lr_handle* ht_, const double* h_plus, const double* h_cross, const double* beta,
                     const double* lam, const double* psi, int64_t batch, int64_t n, double* out, void* stream) {
  lr_handle* h = hp_;
  if (!h || !ht_ || !h_plus || !h_cross || !beta || !lam || !psi || !out) return LR_EINVAL;
  if (capturing((cudaStream_t)stream)) return LR_EINVAL;   // only lr_project and lr_tdi can be captured into a graph
  int rc = check_project(h, batch, n);
  if (rc == LR_OK) rc = check_tdi(ht_, batch, n);
  if (rc != LR_OK) return rc;
  {   // the 2-D copies below use the row pitch n * 8 bytes
    int dev = 0, max_pitch = 0;
    LR_CUDA(h, cudaGetDevice(&dev));
    LR_CUDA(h, cudaDeviceGetAttribute(&max_pitch, cudaDevAttrMaxPitch, dev));
    if (n * (int64_t)sizeof(double) > (int64_t)max_pitch) return LR_EINVAL;
  }
  PlanCall call(ht_);
  cudaStream_t st = (cudaStream_t)stream;
  const TdiShape ts = tdi_shape(ht_);
  const int nout = ht_->channels == LR_XYZ_AET ? 6 : 3;
  const int64_t mp = h->m_proj();
  // three-stage pipeline over (template chunk, time chunk): H2D of the next chunk's h and D2H of the previous
  // chunk's out run on the handle's copy streams while the kernels of the current chunk run on `stream`
  const int64_t bc = batch < 8 ? batch : 8;
  // Chunk lengths.  The call is bound by the device-to-host copy of `out` (3-6 rows per template against 2 rows of
  // h going in), so the first copy should start as early as possible and every chunk costs a fixed ~10 us per
  // stream: the chunks double from n/32 up to the largest the 80 MB slots hold (6 chunks for one year of one
  // template instead of 8 equal ones: 3.26 -> 3.16 ms on a box whose D2H of the 151 MB alone takes 2.66 ms; n/64 first
  // is no better).  LR_OPT_CHUNK_SAMPLES asks for equal chunks of that length.
  const int64_t cap = ((int64_t)80 << 20) / (bc * 6 * (int64_t)sizeof(double)) / kChunkUnit * kChunkUnit;
  int64_t lc = cap < 4 * kChunkUnit ? 4 * kChunkUnit : cap;               // the longest chunk
  int64_t lc_first = round_up((n + 31) / 32, kChunkUnit);
  if (lc_first < 4 * kChunkUnit) lc_first = 4 * kChunkUnit;
  if (h->chunk_samples > 0) lc = lc_first = round_up(h->chunk_samples, kChunkUnit);
  if (lc > round_up(n, kChunkUnit)) lc = round_up(n, kChunkUnit);
  if (lc_first > lc) lc_first = lc;
  const int64_t ly = round_up(lc + ts.halo_lo + ts.halo_hi, 2);
  const int64_t lh = ly + 2 * mp;
  rc = ensure(h, &h->y_scr, &h->y_cap, (size_t)(2 * bc * 6 * ly));
  if (rc == LR_OK) rc = ensure_fix_events(h);
  if (rc == LR_OK) rc = ensure(h, &h->h_buf, &h->h_cap, (size_t)(2 * 2 * bc * lh));
  if (rc == LR_OK) rc = ensure(h, &h->o_buf, &h->o_cap, (size_t)(2 * bc * nout * lc));
  if (rc != LR_OK) return rc;
  if (!h->s_in) {
    LR_CUDA(h, cudaStreamCreateWithFlags(&h->s_in, cudaStreamNonBlocking));
    LR_CUDA(h, cudaStreamCreateWithFlags(&h->s_out, cudaStreamNonBlocking));
    for (int i = 0; i < 2; ++i) {
      LR_CUDA(h, cudaEventCreateWithFlags(&h->ev_in[i], cudaEventDisableTiming));
      LR_CUDA(h, cudaEventCreateWithFlags(&h->ev_comp[i], cudaEventDisableTiming));
      LR_CUDA(h, cudaEventCreateWithFlags(&h->ev_out[i], cudaEventDisableTiming));
    }
  }
  // the copy streams start after whatever the caller enqueued on `stream` before this call
  LR_CUDA(h, cudaEventRecord(h->ev_comp[0], st));
  LR_CUDA(h, cudaStreamWaitEvent(h->s_in, h->ev_comp[0], 0));
  LR_CUDA(h, cudaStreamWaitEvent(h->s_out, h->ev_comp[0], 0));
  int64_t c = 0;
  cudaEvent_t pending[2] = {nullptr, nullptr};   // fix-up kernels still reading y slot 0 / 1
  const size_t dsz = sizeof(double);
  for (int64_t b0 = 0; b0 < batch; b0 += bc) {
    const int64_t nb = batch - b0 < bc ? batch - b0 : bc;
    Stage* S = nullptr;
    rc = stage_basis(h, beta + b0, lam + b0, psi + b0, nb, st, &S);
    if (rc != LR_OK) return rc;
    int64_t len = lc_first;
    for (int64_t a = 0, b = 0; a < n; a = b, ++c, len = 2 * len < lc ? 2 * len : lc) {
      const int slot = (int)(c & 1);
      b = a + len < n ? a + len : n;
      // a short remainder joins this chunk if the slots hold it (one year: 5 chunks instead of 5 + a 98k-sample tail,
      // whose copies would wait for the longest chunk's: 0.1 ms)
      if (n - b > 0 && n - b < len / 2 && n - a <= lc) b = n;
      const int64_t ya = a - ts.halo_lo > 0 ? a - ts.halo_lo : 0, yb = b + ts.halo_hi < n ? b + ts.halo_hi : n;
      const int64_t ha = ya - mp > 0 ? ya - mp : 0, hb = yb + mp < n ? yb + mp : n;
      double* hp_d = h->h_buf + (size_t)slot * 2 * bc * lh;
      double* hc_d = hp_d + (size_t)bc * lh;
      double* o_d = h->o_buf + (size_t)slot * bc * nout * lc;
      // stage 1: H2D (the kernels of chunk c-2 must be done with this slot's h buffer)
      if (c >= 2) LR_CUDA(h, cudaStreamWaitEvent(h->s_in, h->ev_comp[slot], 0));
      LR_CUDA(h, cudaMemcpy2DAsync(hp_d, lh * dsz, h_plus + b0 * n + ha, n * dsz, (hb - ha) * dsz, nb,
                                   cudaMemcpyHostToDevice, h->s_in));
      LR_CUDA(h, cudaMemcpy2DAsync(hc_d, lh * dsz, h_cross + b0 * n + ha, n * dsz, (hb - ha) * dsz, nb,
                                   cudaMemcpyHostToDevice, h->s_in));
      LR_CUDA(h, cudaEventRecord(h->ev_in[slot], h->s_in));
      // stage 2: kernels (the D2H of chunk c-2 must be done with this slot's out buffer)
      LR_CUDA(h, cudaStreamWaitEvent(st, h->ev_in[slot], 0));
      if (c >= 2) LR_CUDA(h, cudaStreamWaitEvent(st, h->ev_out[slot], 0));
      if (pending[slot]) LR_CUDA(h, cudaStreamWaitEvent(st, pending[slot], 0));
      pending[slot] = h->ev_fix[slot];
      rc = response_chunk(h, ht_, ts, hp_d, hc_d, ha, hb, lh, S->dev, nb, n, a, b, ly, o_d, lc, stream,
                          h->y_scr + (size_t)slot * bc * 6 * ly, &pending[slot]);
      if (rc != LR_OK) return rc;
      LR_CUDA(h, cudaEventRecord(h->ev_comp[slot], st));
      // stage 3: D2H (after the chunk's kernels, the fix-up kernel on its side stream included)
      LR_CUDA(h, cudaStreamWaitEvent(h->s_out, h->ev_comp[slot], 0));
      if (pending[slot]) LR_CUDA(h, cudaStreamWaitEvent(h->s_out, pending[slot], 0));
      // rows [template][channel] have one pitch on either side (n on the host, lc in the staging buffer): one copy
      LR_CUDA(h, cudaMemcpy2DAsync(out + b0 * nout * n + a, (size_t)n * dsz, o_d, (size_t)lc * dsz, (b - a) * dsz,
                                   (size_t)nb * nout, cudaMemcpyDeviceToHost, h->s_out));
      LR_CUDA(h, cudaEventRecord(h->ev_out[slot], h->s_out));
    }
    LR_CUDA(h, cudaEventRecord(S->done, st));
    S->pending = true;
  }
  // join: `stream` waits for the last copies, then the call waits for `stream`
  LR_CUDA(h, cudaStreamWaitEvent(st, h->ev_out[0], 0));
  if (c >= 2) LR_CUDA(h, cudaStreamWaitEvent(st, h->ev_out[1], 0));
  LR_CUDA(h, cudaStreamSynchronize(st));
  return LR_OK;
}

int lr_gb_waveform(lr_handle* h, const double* gb, int64_t batch, int64_t n, double* h_plus, double* h_cross,
                   void* stream) {
  if (!h || !gb || !h_plus || !h_cross || !size_ok(batch, n)) return LR_EINVAL;
  if (capturing((cudaStream_t)stream)) return LR_EINVAL;
  for (int64_t i = 0; i < batch * 6; ++i)
    if (!std::isfinite(gb[i])) return LR_EINVAL;
  cudaStream_t st = (cudaStream_t)stream;
  for (int64_t b0 = 0; b0 < batch; b0 += 32768) {   // grid.y limit
    const int64_t nb = batch - b0 < 32768 ? batch - b0 : 32768;
    std::vector<double> zero((size_t)nb, 0.0);
    Stage* S = nullptr;
    const double* gb_dev = nullptr;
    int rc = stage_basis(h, zero.data(), zero.data(), zero.data(), nb, st, &S, gb + b0 * 6, &gb_dev);
    if (rc != LR_OK) return rc;
    LR_CUDA(h, (cudaError_t)lr::launch_gb_waveform(gb_dev, h->t0, h->dt, nb, 0, n, n, h_plus + b0 * n,
                                                   h_cross + b0 * n, stream));
    LR_CUDA(h, cudaEventRecord(S->done, st));
    S->pending = true;
  }
  return LR_OK;
}

}  // extern "C"

namespace {
// lr_response_gb with a row stride for out ([batch][3|6] rows of o_stride >= n doubles)
int response_gb(lr_handle* hp_, lr_handle* ht_, const double* gb, const double* beta, const double* lam,
                const double* psi, int64_t batch, int64_t n, double* out, int64_t o_stride, void* stream) {
  lr_handle* h = hp_;
  if (!h || !ht_ || !gb || !beta || !lam || !psi || !out) return LR_EINVAL;
  if (capturing((cudaStream_t)stream)) return LR_EINVAL;   // only lr_project and lr_tdi can be captured into a graph
  int rc = check_project(h, batch, n);
  if (rc == LR_OK) rc = check_tdi(ht_, batch, n);
  if (rc != LR_OK) return rc;
  for (int64_t i = 0; i < batch * 6; ++i)
    if (!std::isfinite(gb[i])) return LR_EINVAL;
  PlanCall call(ht_);
  cudaStream_t st = (cudaStream_t)stream;
  const TdiShape ts = tdi_shape(ht_);
  const int nout = ht_->channels == LR_XYZ_AET ? 6 : 3;
  const int64_t mp = h->m_proj();
  // the chunk loop of lr_response with one more kernel in front: the chunk's h (with the halos of both stages)
  // is generated into a scratch of the handle, like y
  const int64_t bc = batch < 8 ? batch : 8;
  const int64_t budget = kYSlotBytes / (bc * 6 * (int64_t)sizeof(double));
  int64_t lc = budget / kChunkUnit * kChunkUnit;
  if (lc < 4 * kChunkUnit) lc = 4 * kChunkUnit;
  if (h->chunk_samples > 0) lc = round_up(h->chunk_samples, kChunkUnit);
  if (lc > round_up(n, kChunkUnit)) lc = round_up(n, kChunkUnit);
  const int64_t ly = round_up(lc + ts.halo_lo + ts.halo_hi, 2);
  const int64_t lh = ly + 2 * mp;
  rc = ensure(h, &h->y_scr, &h->y_cap, (size_t)(2 * bc * 6 * ly));
  if (rc == LR_OK) rc = ensure_fix_events(h);
  if (rc == LR_OK) rc = ensure(h, &h->h_buf, &h->h_cap, (size_t)(2 * 2 * bc * lh));
  if (rc != LR_OK) return rc;
  cudaEvent_t pending[2] = {nullptr, nullptr};   // fix-up kernels still reading y slot 0 / 1
  int64_t c = 0;
  for (int64_t b0 = 0; b0 < batch; b0 += bc) {
    const int64_t nb = batch - b0 < bc ? batch - b0 : bc;
    Stage* S = nullptr;
    const double* gb_dev = nullptr;
    rc = stage_basis(h, beta + b0, lam + b0, psi + b0, nb, st, &S, gb + b0 * 6, &gb_dev);
    if (rc != LR_OK) return rc;
    for (int64_t a = 0; a < n; a += lc, ++c) {
      const int slot = (int)(c & 1);
      const int64_t b = a + lc < n ? a + lc : n;
      const int64_t ya = a - ts.halo_lo > 0 ? a - ts.halo_lo : 0, yb = b + ts.halo_hi < n ? b + ts.halo_hi : n;
      const int64_t ha = ya - mp > 0 ? ya - mp : 0, hb = yb + mp < n ? yb + mp : n;
      double* hp_d = h->h_buf + (size_t)slot * 2 * bc * lh;
      double* hc_d = hp_d + (size_t)bc * lh;
      LR_CUDA(h, (cudaError_t)lr::launch_gb_waveform(gb_dev, h->t0, h->dt, nb, ha, hb - ha, lh, hp_d, hc_d, stream));
      if (pending[slot]) LR_CUDA(h, cudaStreamWaitEvent(st, pending[slot], 0));
      pending[slot] = h->ev_fix[slot];
      rc = response_chunk(h, ht_, ts, hp_d, hc_d, ha, hb, lh, S->dev, nb, n, a, b, ly,
                          out + b0 * nout * o_stride + a, o_stride, stream, h->y_scr + (size_t)slot * bc * 6 * ly,
                          &pending[slot]);
      if (rc != LR_OK) return rc;
    }
    LR_CUDA(h, cudaEventRecord(S->done, st));
    S->pending = true;
  }
  for (int i = 0; i < 2; ++i)   // join the last fix-up kernels
    if (pending[i]) LR_CUDA(h, cudaStreamWaitEvent(st, pending[i], 0));
  return LR_OK;
}

}  // namespace

extern "C" {

int lr_response_gb(lr_handle* hp_, lr_handle* ht_, const double* gb, const double* beta, const double* lam,
                   const double* psi, int64_t batch, int64_t n, double* out, void* stream) {
  return response_gb(hp_, ht_, gb, beta, lam, psi, batch, n, out, n, stream);
}

int lr_loglike_gb(lr_handle* hp_, lr_handle* ht_, const double* gb, const double* beta, const double* lam,
                  const double* psi, int64_t batch, int64_t n, const double* data_f, const double* inv_psd,
                  double scale, int mode, double* out, void* stream) {
  lr_handle* h = hp_;
  if (!h || !ht_ || !gb || !beta || !lam || !psi || !data_f || !inv_psd || !out) return LR_EINVAL;
  if (ht_->channels == LR_XYZ_AET || n < 2 || n > 0x7fffffff) return LR_EINVAL;   // three channels per template
  if (mode != LR_IP_CROSS && mode != LR_IP_DIFF) return LR_EINVAL;
  {   // sizes before any allocation (batch < 1 is LR_EINVAL, not a failed cudaMalloc)
    int rc0 = check_project(h, batch, n);
    if (rc0 == LR_OK) rc0 = check_tdi(ht_, batch, n);
    if (rc0 != LR_OK) return rc0;
  }
  PlanCall call(ht_);
  cudaStream_t st = (cudaStream_t)stream;
  const int64_t nt = h->fft_length > 0 ? h->fft_length : n;   // transform length (zero padded beyond n)
  if (nt < n) return LR_EINVAL;
  const int64_t nf = nt / 2 + 1;
  const int64_t bc = batch < 8 ? batch : 8;
  const int64_t np = nt + (nt & 1);   // row stride of the channels: cuFFT wants 16-byte aligned transforms
  // More than one template chunk: two slots of channels and spectra, and the transforms + inner product of chunk c
  // run on a stream of the handle beside the response of chunk c+1 (the response is bound by FP64 issue, the
  // transforms mostly by HBM: they share the SMs well).  One chunk: everything on the caller's stream.
  const int nslot = batch > bc ? 2 : 1;
  const size_t o_slot = (size_t)(bc * 3 * np), f_slot = (size_t)(bc * 3 * nf * 2);
  int rc = ensure(h, &h->o_buf, &h->o_cap, nslot * o_slot);
  if (rc == LR_OK) rc = ensure(h, &h->f_buf, &h->f_cap, nslot * f_slot);
  if (rc == LR_OK) rc = ensure(h, &h->ip_work, &h->ip_cap, (size_t)(bc * LR_IP_BLOCKS));
  if (rc != LR_OK) return rc;
  if (nslot == 2 && !h->s_fft) {
    // highest priority: the transforms' CTAs take SM slots as the response's CTAs retire instead of queueing
    // behind the whole grid of the response kernel launched before them
    int prio_lo = 0, prio_hi = 0;
    LR_CUDA(h, cudaDeviceGetStreamPriorityRange(&prio_lo, &prio_hi));
    LR_CUDA(h, cudaStreamCreateWithPriority(&h->s_fft, cudaStreamNonBlocking, prio_hi));
    for (int i = 0; i < 2; ++i) {
      LR_CUDA(h, cudaEventCreateWithFlags(&h->ev_resp[i], cudaEventDisableTiming));
      LR_CUDA(h, cudaEventCreateWithFlags(&h->ev_fft[i], cudaEventDisableTiming));
    }
  }
  if (h->fft_n != nt) {   // one plan of three real-to-complex transforms (the channels of one template), kept
    if (h->fft_n) { cufftDestroy(h->fft); h->fft_n = 0; }
    int len = (int)nt;
    int in_len = (int)np, out_len = (int)nf;
    const cufftResult fr = cufftPlanMany(&h->fft, 1, &len, &in_len, 1, (int)np, &out_len, 1, (int)nf, CUFFT_D2Z, 3);
    if (fr != CUFFT_SUCCESS) {
      h->last_cuda = 10000 + (int)fr;   // cuFFT result codes are reported as 10000 + cufftResult
      return LR_ECUDA;
    }
    h->fft_n = nt;
  }
  cudaStream_t sf = nslot == 2 ? h->s_fft : st;
  if (cufftSetStream(h->fft, sf) != CUFFT_SUCCESS) { h->last_cuda = 10000; return LR_ECUDA; }
  bool busy[2] = {false, false};   // ev_fft[slot] recorded and not yet waited for by the caller's stream
  int64_t c = 0;
  for (int64_t b0 = 0; b0 < batch; b0 += bc, ++c) {
    const int64_t nb = batch - b0 < bc ? batch - b0 : bc;
    const int slot = nslot == 2 ? (int)(c & 1) : 0;
    double* ob = h->o_buf + slot * o_slot;
    double* fb = h->f_buf + slot * f_slot;
    if (busy[slot]) {   // the transforms of chunk c-2 have read this slot
      LR_CUDA(h, cudaStreamWaitEvent(st, h->ev_fft[slot], 0));
      busy[slot] = false;
    }
    rc = response_gb(hp_, ht_, gb + b0 * 6, beta + b0, lam + b0, psi + b0, nb, n, ob, np, stream);
    if (rc != LR_OK) return rc;
    if (nt > n)   // the zero padding of every row (the response writes [0, n) only)
      LR_CUDA(h, cudaMemset2DAsync(ob + n, (size_t)np * sizeof(double), 0, (size_t)(nt - n) * sizeof(double),
                                   (size_t)nb * 3, st));
    if (nslot == 2) {
      LR_CUDA(h, cudaEventRecord(h->ev_resp[slot], st));
      LR_CUDA(h, cudaStreamWaitEvent(sf, h->ev_resp[slot], 0));
    }
    for (int64_t b = 0; b < nb; ++b) {
      const cufftResult fr = cufftExecD2Z(h->fft, ob + b * 3 * np, reinterpret_cast<cufftDoubleComplex*>(fb) + b * 3 * nf);
      if (fr != CUFFT_SUCCESS) {
        h->last_cuda = 20000 + (int)fr;   // 20000 + cufftResult: the transform itself
        return LR_ECUDA;
      }
    }
    // (ip_work is shared by the slots: the inner products run one after the other on sf)
    rc = lr_inner_product(fb, data_f, inv_psd, scale, mode, nb, 1, 3, nf, h->ip_work, out + b0, (void*)sf);
    if (rc != LR_OK) return rc;
    if (nslot == 2) {
      LR_CUDA(h, cudaEventRecord(h->ev_fft[slot], sf));
      busy[slot] = true;
    }
  }
  for (int i = 0; i < 2; ++i)   // join: `out` is complete on the caller's stream
    if (busy[i]) LR_CUDA(h, cudaStreamWaitEvent(st, h->ev_fft[i], 0));
  return LR_OK;
}

int lr_plan_create(lr_handle* h, int64_t n, void* stream, lr_plan** out) {
  if (!h || !out) return LR_EINVAL;
  *out = nullptr;
  if (capturing((cudaStream_t)stream)) return LR_EINVAL;
  const int rc = check_tdi(h, 1, n);
  if (rc != LR_OK) return rc;
  const TdiShape ts = tdi_shape(h);
  if (ts.path == LR_TDI_PER_SAMPLE) return LR_EINVAL;   // the per-sample path has no plan
  lr_plan* pl = new (std::nothrow) lr_plan();
  if (!pl) return LR_ENOMEM;
  pl->shared = true;
  const int rb = build_plan(h, pl, ts, n, (cudaStream_t)stream, true);
  if (rb != LR_OK) { plan_unref(pl); return rb; }
  *out = pl;
  return LR_OK;
}

int lr_plan_attach(lr_handle* h, lr_plan* plan) {
  if (!h) return LR_EINVAL;
  if (plan && (plan->orbit_id != h->orbit_id || plan->dt != h->dt || plan->order != h->order)) return LR_EINVAL;
  if (plan) plan->refs.fetch_add(1);
  plan_unref(h->attached);
  h->attached = plan;
  return LR_OK;
}

void lr_plan_release(lr_plan* plan) { plan_unref(plan); }

int64_t lr_plan_bytes(const lr_plan* plan) {
  return plan ? (int64_t)(plan->coef_cap * sizeof(double) + (2 * plan->flags_cap + 1) * sizeof(int)) : 0;
}

int lr_gb_parameters(double A, double f0, double fdot, double phi0, double iota, int form, double* gb) {
  if (!gb || (form != LR_GB_PAPER && form != LR_GB_CONFIG) || !(f0 > 0)) return LR_EINVAL;
  if (!std::isfinite(A) || !std::isfinite(f0) || !std::isfinite(fdot) || !std::isfinite(phi0) || !std::isfinite(iota))
    return LR_EINVAL;
  const double ci = cos(iota);
  const double plus = A * (1.0 + ci * ci), cross = -2.0 * A * ci;   // eq. 9's inclination factors
  gb[0] = form == LR_GB_PAPER ? -plus : plus;                        // eq. 9 carries a minus sign on h+ too
  gb[1] = cross;
  gb[2] = f0;
  gb[3] = fdot;
  gb[4] = form == LR_GB_PAPER ? 11.0 / 3.0 * fdot * fdot / f0 : 0.0;  // eq. 8
  gb[5] = phi0;
  return LR_OK;
}

int64_t lr_fft_good_length(int64_t n) {
  if (n < 1 || n > 2147483647) return -1;
  for (int64_t m = n;; ++m) {   // smallest m >= n with no prime factor above 7
    int64_t r = m;
    for (int p : {2, 3, 5, 7})
      while (r % p == 0) r /= p;
    if (r == 1) return m;
  }
}

int lr_eval_orbit(lr_handle* h, int channel, const double* t, int64_t m, double* out, void* stream) {
  if (!h || !t || !out || channel < 0 || channel >= lr::kSplineChannels || m < 1) return LR_EINVAL;
  lr::Params P = make_params(h, 1);
  const int threads = 256;
  const int64_t blocks = (m + threads - 1) / threads;
  if (blocks > 0x7fffffff) return LR_EINVAL;
  lr::eval_orbit_kernel<<<(unsigned)blocks, threads, 0, (cudaStream_t)stream>>>(P, channel, h->t_start, t, m, out);
  lr::g_launches.fetch_add(1);
  LR_CUDA(h, cudaGetLastError());
  return LR_OK;
}

int64_t lr_launch_count(void) { return lr::g_launches.load(); }

int lr_last_cuda_error(const lr_handle* h) { return h ? h->last_cuda : 0; }

const char* lr_strerror(int code) {
  switch (code) {
    case LR_OK: return "success";
    case LR_EINVAL: return "invalid argument";
    case LR_ERANGE: return "sample span (with the delays' backward reach) is not covered by the orbit table";
    case LR_ECUDA: return "CUDA error (see lr_last_cuda_error)";
    case LR_ENOMEM: return "host allocation failed";
    case LR_ELIMIT: return "size exceeds the fixed capacity of this no-allocation entry point (see include/lr.h)";
    default: return "unknown error code";
  }
}

}  // extern "C"
