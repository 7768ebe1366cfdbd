// lr_waveform.cu — the template generator in front of the response: the Galactic-
// binary waveform of PAPER.md eqs. 5-9 evaluated on the device, so that h+ and hx never
// come from the host.
//
//   cycles(t) = f0 t + fdot t^2 / 2 + fddot t^3 / 6,   h+ = a+ cos(2 pi cycles + phi0),  hx = ax sin(...)
//
// at t_n = t0 + n dt.  After a year a mHz source has run through 1e5-1e6 cycles, so the phase has to be
// reduced modulo one before it is rounded: t_n and the cubic are evaluated in double-double arithmetic
// (error-free products by FMA, about 1e-32 relative), the nearest integer is removed from the high word, and
// only the remaining fraction meets 2 pi.  The sine and cosine are the CUDA math library's fp64 sincos (1-2 ulp).
#include <cuda_runtime.h>

#include <atomic>
#include <cstdint>

namespace lr {

extern std::atomic<int64_t> g_launches;

namespace {

struct DD { double hi, lo; };

__device__ __forceinline__ DD two_sum(double a, double b) {
  const double s = a + b, bb = s - a;
  return {s, (a - (s - bb)) + (b - bb)};
}
__device__ __forceinline__ DD quick_two_sum(double a, double b) {   // |a| >= |b|
  const double s = a + b;
  return {s, b - (s - a)};
}
__device__ __forceinline__ DD two_prod(double a, double b) {
  const double p = a * b;
  return {p, fma(a, b, -p)};
}
__device__ __forceinline__ DD dd_add_d(DD a, double b) {
  DD s = two_sum(a.hi, b);
  return quick_two_sum(s.hi, s.lo + a.lo);
}
__device__ __forceinline__ DD dd_mul(DD a, DD b) {
  DD p = two_prod(a.hi, b.hi);
  p.lo += a.hi * b.lo + a.lo * b.hi;
  return quick_two_sum(p.hi, p.lo);
}

// gb: DEVICE [batch][6] = a_plus, a_cross, f0, fdot, fddot, phi0.  Writes the global samples [first, first+count)
// of every template into rows of `stride` doubles whose element 0 is global sample `first`.
__global__ void __launch_bounds__(256)
gb_waveform_kernel(const double* __restrict__ gb, double t0, double dt, int64_t first, int64_t count, int64_t stride,
                   double* __restrict__ hp, double* __restrict__ hc) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= count) return;
  const int64_t b = blockIdx.y;
  const double* g = gb + b * 6;
  const double ap = __ldg(g), ac = __ldg(g + 1), f0 = __ldg(g + 2), c2 = 0.5 * __ldg(g + 3), fddot = __ldg(g + 4),
               phi0 = __ldg(g + 5);
  DD c3;                                         // fddot / 6 in two words (fddot - 6 c3.hi is exact in one FMA)
  c3.hi = fddot / 6.0;
  c3.lo = fma(-6.0, c3.hi, fddot) / 6.0;
  // t = t0 + n dt, exactly to double-double precision (n < 2^53 is exact in fp64)
  const DD ndt = two_prod((double)(first + i), dt);
  const DD t = dd_add_d(two_sum(ndt.hi, t0), ndt.lo);
  // Horner in double-double: cycles = t (f0 + t (c2 + t c3))
  DD c = dd_mul(t, c3);
  c = dd_add_d(c, c2);
  c = dd_mul(c, t);
  c = dd_add_d(c, f0);
  c = dd_mul(c, t);
  const double whole = rint(c.hi);
  double frac = (c.hi - whole) + c.lo;          // in [-1/2, 1/2] (+ a rounding of the low word)
  // 2 pi in two words
  const double tp_hi = 6.283185307179586232, tp_lo = 2.4492935982947064e-16;
  const double ang = fma(frac, tp_hi, fma(frac, tp_lo, phi0));
  double s, co;
  sincos(ang, &s, &co);
  hp[b * stride + i] = ap * co;
  hc[b * stride + i] = ac * s;
}

}  // namespace

int launch_gb_waveform(const double* gb_dev, double t0, double dt, int64_t batch, int64_t first, int64_t count,
                       int64_t stride, double* hp, double* hc, void* stream) {
  const int threads = 256;
  const dim3 grid((unsigned)((count + threads - 1) / threads), (unsigned)batch);
  gb_waveform_kernel<<<grid, threads, 0, (cudaStream_t)stream>>>(gb_dev, t0, dt, first, count, stride, hp, hc);
  g_launches.fetch_add(1);
  return (int)cudaGetLastError();
}

}  // namespace lr
