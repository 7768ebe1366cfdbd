/* lr.h — C ABI of liblr: the generic time-domain LISA response on one B200 (sm_100a).
 *
 * The library computes the data-parallel hot path of arXiv:2204.06633:
 *   stage 1  lr_project : the six single-link responses y_ij(t)          (eqs. 10-16)
 *   stage 2  lr_tdi     : first/second-generation TDI X,Y,Z and A,E,T     (eqs. 17-21)
 * over arbitrary orbits given as a table that lr_create turns into device-resident cubic splines
 * ("interpolated and then evaluated at each evenly-spaced time step"), with centred
 * Lagrange fractional-delay interpolation of user-defined order, batched over templates
 * (one response per walker per MCMC step).
 *
 * Conventions (DESIGN.md §3 lists the readings A1..A16 behind them)
 *   - every array is fp64, C-contiguous; "DEVICE" = CUDA device memory of the current device,
 *     "HOST" = ordinary host memory.  The caller owns every buffer it passes.
 *   - link slots are ordered [12, 23, 31, 13, 32, 21]; link ij is received on spacecraft i and was
 *     emitted by spacecraft j.
 *   - sample n of every series (h, y, out) is at time t0 + n*dt (LR_OPT_T0, default orbits->t_start).
 *   - "order" is the polynomial degree of the Lagrange interpolant: order+1 taps, order odd (1..65).
 *   - L_ij are light travel TIMES in seconds ("the delay time").
 *   - outputs are fully written; samples inside the fixed margins (lr_get_margins) are exactly 0.0.
 *   - lr_project / lr_tdi enqueue work on `cuda_stream` (a cudaStream_t, NULL = legacy default stream)
 *     and return without synchronising.  lr_response_host is synchronous.
 *   - lr_project (batch <= 16) and lr_tdi may be captured into a CUDA graph (cudaStreamBeginCapture on `cuda_stream`):
 *     they then wait on nothing outside the capture.  Call lr_tdi once outside a capture first, with the same n and
 *     options (the graph keeps the addresses of the handle's TDI plan: do not change LR_OPT_* or call lr_tdi with
 *     another n on that handle while the graph is in use, which would rebuild the plan), replay the graph on one stream
 *     at a time, and destroy it before the handle.  Every other computing call returns LR_EINVAL on a capturing
 *     stream.
 *   - all entry points return 0 on success or a negative LR_E* code; they never abort, throw or print.
 *     Inputs are not scanned for NaN (NaN propagates).
 *   - a handle keeps per-call staging state (and lr_tdi's plan): use one handle from one host thread and one
 *     stream at a time; different handles are independent.
 *   - there is no CPU fallback: every call that computes needs a CUDA device and fails with LR_ECUDA
 *     otherwise.
 */
#ifndef LR_H_
#define LR_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct lr_handle lr_handle; /* opaque; owns the device spline coefficients and small staging buffers */

/* Orbit table on uniform knots (§IV.D: positions and light travel times as
 * delivered by an orbit product).  lr_create copies it; the caller may free it on return. */
typedef struct {
  int64_t n_knots;   /* >= 4 */
  double t_start;    /* time of knot 0 [s] */
  double knot_dt;    /* uniform knot spacing [s] (> 0), e.g. 86400 */
  const double* x;   /* HOST [3 spacecraft][3 xyz][n_knots], metres, SSB frame */
  const double* ltt; /* HOST [6 links: 12,23,31,13,32,21][n_knots], seconds */
} lr_orbits;

/* error codes */
#define LR_OK 0
#define LR_EINVAL (-1)  /* null pointer, bad order / generation / dt / sizes */
#define LR_ERANGE (-2)  /* the sample span (with the backward reach of the delays) leaves the knot table */
#define LR_ECUDA (-3)   /* a CUDA call failed; lr_last_cuda_error gives the CUDA code */
#define LR_ENOMEM (-4)  /* host allocation failed */
#define LR_ELIMIT (-5)  /* a size exceeds the fixed capacity of a no-allocation entry point (lr_inner_product_static) */

/* option keys for lr_set_option */
#define LR_OPT_T0 1       /* time of sample 0 [s]; default orbits->t_start */
#define LR_OPT_CHAIN 2    /* LR_CHAIN_NESTED (default) | LR_CHAIN_SUM */
#define LR_OPT_CHANNELS 3 /* LR_XYZ (default) | LR_AET | LR_XYZ_AET */
#define LR_OPT_TDI_GEN 4  /* 1 | 2: changes the generation given to lr_create */
#define LR_OPT_TDI_PATH 5 /* LR_TDI_AUTO (default) | LR_TDI_PER_SAMPLE | LR_TDI_FIR3 | LR_TDI_FIR4 */
#define LR_OPT_CHUNK_SAMPLES 7 /* time-chunk length of lr_response / lr_response_host (rounded up to 1792); 0 = automatic */
#define LR_OPT_FFT_LENGTH 8 /* transform length of lr_loglike_gb (>= n, zero padded); 0 (default) = n */
#define LR_OPT_TDI_PLAN_CACHE 6 /* 1 (default): keep the FIR plan between lr_tdi calls; 0: rebuild every call */
#define LR_OPT_PROJ_PATH 9 /* LR_PROJ_AUTO (default) | LR_PROJ_SINGLE | LR_PROJ_PAIR */
#define LR_OPT_Y_PRECISION 10 /* LR_Y_EXTENDED (default) | LR_Y_PLAIN */

/* How lr_project forms the delayed times (the end-to-end accuracy of the path).
 * The same eq. 16 either way; the difference is where fp64 rounding enters.
 *   LR_Y_PLAIN    : every delay is an fp64 number of samples (t - k.x_i/c is ~50-100 samples away: 7e-15 samples of
 *                   rounding), y agrees with the long-double oracle to ~2e-14 (the round-1 kernel, bit for bit).
 *   LR_Y_EXTENDED : the emission time of a link is placed relative to the split (integer, fraction) of its reception
 *                   time, from L_ij/dt and k.(x_i - x_j)/(c dt) with the arm vectors x_i - x_j splined from the exact
 *                   differences of the table; y agrees with the oracle to ~1e-15, and the end-to-end T channel
 *                   (which amplifies errors of y by up to 1e6 at 0.1 mHz) improves by the same factor.  Costs 2 % of
 *                   lr_project and is the default; runs the one-sample-per-thread kernel. */
#define LR_Y_PLAIN 0
#define LR_Y_EXTENDED 1

/* Read-only keys of lr_get_option: what lr_tdi will do with the handle's current orbits and options.
 *   LR_INFO_TDI_PATH   : the path LR_TDI_AUTO resolves to (LR_TDI_PER_SAMPLE | LR_TDI_FIR3 | LR_TDI_FIR4)
 *   LR_INFO_FIR_TAPS   : taps per series of the merged FIR filters (0 on the per-sample path)
 *   LR_INFO_FIR_POWERS : accumulators per output sample = powers of tile time (1 for constant light times, 3, 4; 0 on
 *                        the per-sample path).  The FIR path executes 3 channels x 4 series x taps x powers FMAs per
 *                        sample (bench.py's `executed_ops_per_sample`). */
#define LR_INFO_TDI_PATH 101
#define LR_INFO_FIR_TAPS 102
#define LR_INFO_FIR_POWERS 103

/* How lr_project maps time samples to threads (the results are the same bit for bit).
 *   LR_PROJ_SINGLE : one sample per thread.
 *   LR_PROJ_PAIR   : two consecutive samples per thread; the two Lagrange stencils of every interpolation time share
 *                    all but one of their first differences, which are then read from shared memory once (half the
 *                    shared-memory traffic; orders with a compile-time kernel, any other order runs LR_PROJ_SINGLE).
 *                    Measured on B200 it is 5-7 % slower than LR_PROJ_SINGLE at order 25 (166 registers per thread
 *                    leave 11 warps per SM against 16), so it is not the default.
 *   LR_PROJ_AUTO   : the faster of the two on B200 (LR_PROJ_SINGLE). */
#define LR_PROJ_AUTO (-1)
#define LR_PROJ_SINGLE 1
#define LR_PROJ_PAIR 2

/* How lr_tdi evaluates the Lagrange weights (same result to rounding).
 *   LR_TDI_PER_SAMPLE : every delayed term gets its own weight set at every sample.
 *   LR_TDI_FIR3/4     : per tile of 224 samples the weights are a quadratic/cubic polynomial in time fitted
 *                       through 3/4 nodes, and all terms of a series merge into one short FIR filter; tiles
 *                       in which a delay crosses a whole number of samples use the per-sample code.
 *                       The per-tile filters (the "plan") depend on the orbits and the time grid (n, t0, dt,
 *                       generation, chain mode) only, not on y: one plan serves every template of a batch and,
 *                       with LR_OPT_TDI_PLAN_CACHE = 1, every later call on the same grid (the paper keeps its
 *                       orbit arrays on the device "for the entirety of the sampling run").  The
 *                       plan costs 12*Wc*32 B per tile (about 60 B per sample at order 25) of device memory.
 *   LR_TDI_AUTO       : FIR3 / FIR4 / PER_SAMPLE by the largest light-time rate of the orbit table. */
#define LR_TDI_AUTO (-1)
#define LR_TDI_PER_SAMPLE 0
#define LR_TDI_FIR3 3
#define LR_TDI_FIR4 4

/* Chained delays D_{i1 i2 ... in} (eqs. 19-20).
 *   LR_CHAIN_SUM    : eq. 20 verbatim, the sum of the L's all taken at t.
 *   LR_CHAIN_NESTED : d_0 = 0, d_k = d_{k-1} + L_{i_k i_{k+1}}(t - d_{k-1}) (leftmost pair at t); the whole
 *                     chain is applied as ONE interpolation at t - d_n. */
#define LR_CHAIN_NESTED 0
#define LR_CHAIN_SUM 1

/* Output channels of lr_tdi (eq. 21). LR_XYZ_AET writes [X,Y,Z,A,E,T]. */
#define LR_XYZ 0
#define LR_AET 1
#define LR_XYZ_AET 2

#define LR_MAX_ORDER 65

/* Build a response object: fit a not-a-knot cubic spline to each of the 15 orbit channels on the host,
 * upload the per-interval coefficients, fix the margins.  dt = sample spacing of h, y and out [s];
 * lagrange_order odd in [1, LR_MAX_ORDER]; tdi_gen in {1, 2}.  *out receives the handle.
 * Errors: LR_EINVAL, LR_ENOMEM, LR_ECUDA. */
int lr_create(const lr_orbits* orbits, double dt, int lagrange_order, int tdi_gen, lr_handle** out);

/* Free the handle and its device memory (NULL is allowed).  Work enqueued earlier must have finished. */
void lr_destroy(lr_handle* h);

/* Set an option (see LR_OPT_*).  Errors: LR_EINVAL for an unknown key or value. */
int lr_set_option(lr_handle* h, int key, double value);

/* Read an option back (*value receives what lr_set_option stored, or the default).  The binding uses
 * LR_OPT_CHANNELS to check the size of `out` before a call writes 3 or 6 rows per template.
 * Errors: LR_EINVAL for a null pointer or an unknown key. */
int lr_get_option(const lr_handle* h, int key, double* value);

/* Fixed margins in samples (reading A8), computed once from the table maxima R_max = max|x_i|
 * and L_max = max L_ij over the knots, p = (order+1)/2:
 *   m_proj      = ceil((1.001 R_max/c + 1.001 L_max)/dt) + p + 2          y is 0 outside [m_proj, n - m_proj)
 *   m_tdi_front = m_proj + ceil(G 1.001 L_max/dt) + p + 2, G = 4 (gen 1) | 8 (gen 2)
 *   m_tdi_back  = m_proj + p + 2                              out is 0 outside [m_tdi_front, n - m_tdi_back)
 * Any of the three pointers may be NULL. */
int lr_get_margins(const lr_handle* h, int64_t* m_proj, int64_t* m_tdi_front, int64_t* m_tdi_back);

/* Stage 1 (eqs. 10-16).  For every template b and sample n in [m_proj, n - m_proj), t = t0 + n dt:
 *   k,u,v from (beta, lambda) per eq. 10, (u,v) rotated by psi (equivalent to eq. 9's rotation of h by 2 psi);
 *   n_ij = (x_i(t) - x_j(t))/|.|, xi+ = (u.n)^2 - (v.n)^2, xix = 2 (u.n)(v.n)                    (eq. 12)
 *   y_ij = [xi+ (h+(t_e) - h+(t_r)) + xix (hx(t_e) - hx(t_r))] / (2 (1 - k.n_ij))               (eq. 16)
 *   t_e = t - L_ij(t) - k.x_j(t)/c,  t_r = t - k.x_i(t)/c, h evaluated by Lagrange interpolation.
 * h_plus, h_cross : DEVICE [batch][n];  beta (ecliptic latitude), lambda (ecliptic longitude), psi : HOST [batch]
 * (the three angles are copied to the device as they are; k, u, v are computed there by a one-thread-per-template
 * kernel in front of the projection kernel).  y_out : DEVICE [batch][6][n].  Requires n > 2 m_proj and n < 2^31 - 2^20.
 * Errors: LR_EINVAL, LR_ERANGE, LR_ECUDA. */
int lr_project(lr_handle* h, const double* h_plus, const double* h_cross, const double* beta,
               const double* lambda, const double* psi, int64_t batch, int64_t n, double* y_out,
               void* cuda_stream);

/* Stage 2 (eqs. 17-21).  y : DEVICE [batch][6][n] (any handle's lr_project output — a handle with
 * other orbits gives the paper's hybrid templates).  out : DEVICE [batch][3][n] (LR_XYZ,
 * LR_AET) or [batch][6][n] (LR_XYZ_AET).  Requires n > m_tdi_front + m_tdi_back.
 * Errors: LR_EINVAL, LR_ERANGE, LR_ECUDA. */
int lr_tdi(lr_handle* h, const double* y, int64_t batch, int64_t n, double* out, void* cuda_stream);

/* Both stages with DEVICE buffers and no [batch][6][n] array: h_plus, h_cross DEVICE [batch][n] -> out DEVICE
 * [batch][3|6][n], bit-identical to lr_project followed by lr_tdi.  The path runs in chunks of time (and of
 * 8 templates) through a y scratch of two slots of <= 1 GB owned by h_proj, so the device footprint
 * is h + out + that scratch (the paper's real call is waveform -> projection -> TDI with nothing
 * in between leaving the GPU).  Enqueues on `cuda_stream` and returns without synchronising.
 * beta, lambda, psi: HOST [batch].  Errors: as lr_project / lr_tdi. */
int lr_response(lr_handle* h_proj, lr_handle* h_tdi, const double* h_plus, const double* h_cross,
                const double* beta, const double* lambda, const double* psi, int64_t batch, int64_t n, double* out,
                void* cuda_stream);

/* The same for a SPAN of the time axis (one long template split over several GPUs, each rank
 * recomputing its halo instead of exchanging it — no collective).  Computes out for the global samples
 * [first, first+count) of a series of n samples; time, margins and results are those of the whole-series
 * call, bit for bit.  h_plus, h_cross: DEVICE [batch][h_len] holding the global samples
 * [h_first, h_first+h_len), which must include [first - lo, first+count+hi) clipped to [0, n) with (lo, hi)
 * from lr_get_span_halo; out: DEVICE [batch][3|6][count].  `first` must be a multiple of the span unit
 * (lr_get_span_halo's `unit`, 1792 samples).  Errors: LR_EINVAL for a bad span or a too-short h slice, else as
 * lr_response. */
int lr_response_span(lr_handle* h_proj, lr_handle* h_tdi, const double* h_plus, const double* h_cross,
                     int64_t h_first, int64_t h_len, const double* beta, const double* lambda, const double* psi,
                     int64_t batch, int64_t n, int64_t first, int64_t count, double* out, void* cuda_stream);

/* Samples of h a span needs before (lo) and after (hi) itself, and the alignment unit of `first`.  Any pointer
 * may be NULL. */
int lr_get_span_halo(const lr_handle* h_proj, const lr_handle* h_tdi, int64_t* lo, int64_t* hi, int64_t* unit);

/* Both stages with HOST buffers: copies h_plus/h_cross [batch][n] to the device, runs lr_project on
 * `h_proj` and lr_tdi on `h_tdi` (may be the same handle), copies out [batch][3|6][n] back and waits.
 * The call is a three-stage pipeline over chunks of time: the H2D copy of the next chunk and the D2H copy of
 * the previous one overlap the kernels (pinned host buffers are needed for the overlap; pageable ones work,
 * serially).  Device scratch is owned by h_proj and grown on demand (kept until lr_destroy).
 * `cuda_stream` as above.  Errors: as lr_project / lr_tdi, LR_ECUDA for a failed allocation or copy. */
int lr_response_host(lr_handle* h_proj, lr_handle* h_tdi, const double* h_plus, const double* h_cross,
                     const double* beta, const double* lambda, const double* psi, int64_t batch, int64_t n,
                     double* out, void* cuda_stream);

/* A shareable TDI plan (the orbit information is "pre-computed and stored for the entirety of the
 * sampling run").  lr_tdi's FIR path keeps, per tile of 224 samples, the merged Lagrange filters of eqs. 17-20 (the
 * "plan": a function of the orbits, dt, order, n, t0, generation and chain mode, not of y).  By default every handle
 * builds and caches its own on first use.  An MCMC driver that runs several handles / streams on the same orbits can
 * instead build the plan ONCE and attach it to all of them:
 *   lr_plan_create : builds the plan for h's current options (LR_OPT_T0, generation, chain, path) and a series of n
 *                    samples on `cuda_stream`, waits for it, and returns an object that is read-only from then on
 *                    (reference count 1).  LR_EINVAL if h's lr_tdi path is LR_TDI_PER_SAMPLE (no plan), else errors
 *                    as lr_tdi.
 *   lr_plan_attach : h uses `plan` (one more reference) for every lr_tdi / lr_response* call whose grid and options
 *                    equal the plan's; any other call falls back to h's own cached plan.  The plan must come from a
 *                    handle with the same orbit table, dt and order (LR_EINVAL otherwise).  NULL detaches.
 *   lr_plan_release: drops the caller's reference; the device memory goes when the last attached handle is destroyed.
 * Results with an attached plan are bit-identical to those with the handle's own.  Handles that share a plan may be
 * used from different host threads and streams at the same time (each handle still from one thread at a time). */
typedef struct lr_plan lr_plan;
int lr_plan_create(lr_handle* h, int64_t n, void* cuda_stream, lr_plan** out);
int lr_plan_attach(lr_handle* h, lr_plan* plan);
void lr_plan_release(lr_plan* plan);
/* Device bytes the plan holds (0 for NULL). */
int64_t lr_plan_bytes(const lr_plan* plan);

/* Template generator (eqs. 5-9; SURVEY.md §8(f) NEXT-1 "generate the GB waveform
 * from the parameters").  One template is LR_GB_NPAR doubles
 *   gb = { a_plus, a_cross, f0 [Hz], fdot [Hz/s], fddot [Hz/s^2], phi0 [rad] }
 * and its polarisations at t_n = t0 + n dt (t0 = LR_OPT_T0 of the handle, dt = the handle's) are
 *   h_plus[n]  = a_plus  cos( 2 pi (f0 t_n + fdot t_n^2 / 2 + fddot t_n^3 / 6) + phi0 )      eq. 5a
 *   h_cross[n] = a_cross sin( same argument )                                                eq. 5b
 * Eq. 9's inclination factors and signs are the caller's amplitudes (paper: a_plus = -A (1 + cos^2 iota),
 * a_cross = -2 A cos iota; BASELINE.json's configs: a_plus = +A (1 + cos^2 iota)); eq. 9's rotation by 2 psi
 * is applied by lr_project to the basis (reading A4); eq. 8 gives the paper's fddot = 11/3 fdot^2 / f0.
 * The phase is reduced modulo one cycle in double-double arithmetic before it is rounded, so the samples are
 * correct to a few ulp of the amplitude however many cycles have gone by.
 * gb: HOST [batch][LR_GB_NPAR] (read before the call returns); h_plus, h_cross: DEVICE [batch][n].
 * Errors: LR_EINVAL (null pointer, non-finite parameter, bad sizes), LR_ECUDA. */
#define LR_GB_NPAR 6
int lr_gb_waveform(lr_handle* h, const double* gb, int64_t batch, int64_t n, double* h_plus, double* h_cross,
                   void* cuda_stream);

/* The six numbers of lr_gb_waveform from the physical parameters (HOST arithmetic, no device needed):
 *   LR_GB_PAPER : eqs. 8-9 — a_plus = -A (1 + cos^2 iota), a_cross = -2 A cos iota, fddot = 11/3 fdot^2 / f0
 *   LR_GB_CONFIG: BASELINE.json's configs — a_plus = +A (1 + cos^2 iota), a_cross = -2 A cos iota, fddot = 0
 * gb: HOST [LR_GB_NPAR] (written).  Errors: LR_EINVAL (null pointer, unknown form, f0 <= 0, non-finite input). */
#define LR_GB_PAPER 0
#define LR_GB_CONFIG 1
int lr_gb_parameters(double A, double f0, double fdot, double phi0, double iota, int form, double* gb);

/* Parameters -> TDI channels in one call: lr_gb_waveform, lr_project (on h_proj) and lr_tdi (on h_tdi, may be
 * the same handle) chunk by chunk along time; neither h nor y exists as a whole array, both live in scratch
 * of h_proj.  out: DEVICE [batch][3|6][n], bit-identical to
 * lr_response on the output of lr_gb_waveform.  gb, beta, lambda, psi: HOST, read before the call returns.
 * Errors: as lr_gb_waveform and lr_response. */
int lr_response_gb(lr_handle* h_proj, lr_handle* h_tdi, const double* gb, const double* beta, const double* lambda,
                   const double* psi, int64_t batch, int64_t n, double* out, void* cuda_stream);

/* Noise-weighted inner product of frequency-domain channels (eqs. 2-3, 22):
 *   LR_IP_CROSS : out[b] = scale * sum_{ch,k} Re( conj(fa[b][ch][k]) fb[b'][ch][k] ) * inv_psd[ch][k]
 *   LR_IP_DIFF  : out[b] = scale * sum_{ch,k} | fa[b][ch][k] - fb[b'][ch][k] |^2   * inv_psd[ch][k]
 * with b' = b (batch_b == batch) or 0 (batch_b == 1: one data set d against every template).  With
 * a~ = dt * rfft(a), df = 1/(n dt) and inv_psd = 1/S_n (0 in the DC bin), scale = 4 df gives <a|b> of eq. 2
 * summed over the channels (eq. 22) and, in LR_IP_DIFF mode, scale = -2 df gives log L = -<d-h|d-h>/2 of eq. 3.
 * The Fourier transforms are the caller's (a library FFT).  fa: DEVICE [batch][nch][nf] complex128 (re, im
 * interleaved), fb: DEVICE [batch_b][nch][nf], inv_psd: DEVICE [nch][nf], work: DEVICE scratch of
 * batch * LR_IP_BLOCKS doubles, out: DEVICE [batch].  Deterministic (fixed reduction tree).  batch <= 65535.
 * Enqueues on `cuda_stream`.  Errors: LR_EINVAL, LR_ECUDA. */
#define LR_IP_CROSS 0
#define LR_IP_DIFF 1
#define LR_IP_BLOCKS 1024
int lr_inner_product(const double* fa, const double* fb, const double* inv_psd, double scale, int mode,
                     int64_t batch, int64_t batch_b, int nch, int64_t nf, double* work, double* out,
                     void* cuda_stream);

/* lr_inner_product for callers that cannot allocate (code under CUDA graph capture, tight serving loops, harnesses
 * that forbid cudaMalloc): the same kernels and the same results bit for bit, with the scratch of the reduction (the
 * per-block partial sums) in a device array that is part of the library image instead of a caller-supplied `work`
 * buffer.  The call allocates nothing: no cudaMalloc, cudaFree or allocating library routine; its first call on a
 * device resolves the array's address (cudaGetSymbolAddress, with that device current) and caches it.
 *   - limit: batch <= LR_IP_STATIC_MAX_BATCH (64); a larger batch returns LR_ELIMIT and launches nothing (split
 *     the batch, or use lr_inner_product).  The array is LR_IP_STATIC_MAX_BATCH * LR_IP_BLOCKS doubles = 512 KB of
 *     device memory on every GPU that loads the library, held until the process exits.
 *   - ALL calls on a device share the one array: two calls whose kernels can overlap on the GPU (different streams
 *     without an ordering between them, or two host threads) race on it and give wrong results.  Calls on one
 *     stream, or otherwise ordered, are safe.  Nothing in it needs clearing between calls: stage 1 overwrites every
 *     element stage 2 reads.
 * Arguments as lr_inner_product without `work`.  Errors: LR_EINVAL, LR_ELIMIT, LR_ECUDA. */
#define LR_IP_STATIC_MAX_BATCH 64
int lr_inner_product_static(const double* fa, const double* fb, const double* inv_psd, double scale, int mode,
                            int64_t batch, int64_t batch_b, int nch, int64_t nf, double* out, void* cuda_stream);

/* One likelihood evaluation per template, parameters in, one scalar out ("only the scalar
 * returns"; eqs. 2-3, 5-9, 10-22): lr_response_gb into scratch, the library's real-to-complex FFT (cuFFT, fp64)
 * of the three TDI channels, lr_inner_product against one data set:
 *   out[b] = scale * sum_{ch,k} inv_psd[ch][k] * ( mode LR_IP_DIFF ? |H_b[ch][k] - data_f[ch][k]|^2
 *                                                                   : Re( conj(H_b[ch][k]) data_f[ch][k] ) )
 * with H_b[ch][k] = sum_n out_b[ch][n] exp(-2 pi i k n / N), k = 0 .. N/2 — the UNNORMALISED forward DFT of the
 * channels (margins are zeros); data_f must be in the same convention.  log L of eq. 3 with a~ = dt * DFT is
 * scale = -2 dt / N, mode LR_IP_DIFF, inv_psd[ch][0] = 0.
 * With LR_OPT_FFT_LENGTH = M > n set on h_proj the channels are zero padded to M samples before the transform
 * (N = M in the formulas above: data_f and inv_psd then have M/2+1 bins on the grid k / (M dt)); a length without
 * prime factors above 7 (lr_fft_good_length) makes the transform 2-3x faster than e.g. 3,153,600 = 2^6 3^3 5^2 73.
 * h_tdi must produce three channels (LR_XYZ or LR_AET).  gb, beta, lambda, psi: HOST [batch]...; data_f: DEVICE
 * complex [3][N/2+1] (interleaved re, im); inv_psd: DEVICE [3][N/2+1]; out: DEVICE [batch].  Scratch (the
 * channels and spectra of 8 templates — twice that for batch > 8 — and the FFT plan) is owned by h_proj and kept
 * until lr_destroy.  Templates are processed in chunks of 8; for batch > 8 the transforms and the inner product of
 * one chunk run on a stream of the handle beside the response of the next chunk and are joined to `cuda_stream`
 * before the call returns, so the caller sees ordinary stream ordering.
 * Errors: LR_EINVAL (as lr_response_gb, or six output channels), LR_ECUDA (CUDA or cuFFT failure). */
int lr_loglike_gb(lr_handle* h_proj, lr_handle* h_tdi, const double* gb, const double* beta, const double* lambda,
                  const double* psi, int64_t batch, int64_t n, const double* data_f, const double* inv_psd,
                  double scale, int mode, double* out, void* cuda_stream);

/* Smallest length >= n whose prime factors are 2, 3, 5, 7 (HOST arithmetic); -1 for n outside [1, 2^31). */
int64_t lr_fft_good_length(int64_t n);

/* Evaluate the device spline of one orbit channel (0..8 = x[i][a] as i*3+a, 9..14 = L link slots) at
 * `m` times t (DEVICE [m]) into out (DEVICE [m]); used by the tests to pin the orbit ingestion. */
int lr_eval_orbit(lr_handle* h, int channel, const double* t, int64_t m, double* out, void* cuda_stream);

/* Measure this device's FP64 issue rate with a DFMA-only kernel that runs for about `seconds` (8 chains per thread,
 * acc = acc * register + uniform register: the operand form with which the pipe reaches its 64 DFMA per SM and clock;
 * chains with three register operands stop at 58.7, see lr_peak.cu):
 * *inst_per_s = FP64 thread-instructions per second (one DFMA = 1).  The roofline denominator of bench.py.
 * Synchronous.  Errors: LR_EINVAL, LR_ECUDA. */
int lr_measure_fp64_peak(double seconds, double* inst_per_s);

/* Number of kernels liblr has launched in this process (all handles); bench.py's gpu_launches. */
int64_t lr_launch_count(void);

/* CUDA error code (cudaError_t as int) of the last failed CUDA call on this handle, 0 if none.  A failed cuFFT
 * call in lr_loglike_gb is reported as 10000 + cufftResult (planning) or 20000 + cufftResult (execution). */
int lr_last_cuda_error(const lr_handle* h);

/* Static description of an LR_* code. */
const char* lr_strerror(int code);

#ifdef __cplusplus
}
#endif
#endif /* LR_H_ */
