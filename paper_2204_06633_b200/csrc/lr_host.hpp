// lr_host.hpp — host-side numerics of lr_create: spline fit and Lagrange constants.
#pragma once
#include <stdint.h>

#include <vector>

#include "lr_device.cuh"

namespace lr {

// Not-a-knot cubic spline on uniform knots, solved for the knot slopes s_i (Hermite form):
//   s_{i-1} + 4 s_i + s_{i+1} = 3 (y_{i+1} - y_{i-1}) / h                       i = 1..n-2
//   s_0 + 2 s_1 = (-5 y_0 + 4 y_1 + y_2) / (2h),   2 s_{n-2} + s_{n-1} = (5 y_{n-1} - 4 y_{n-2} - y_{n-3}) / (2h)
// (the end rows are the interior row combined with continuity of the third derivative at knots 1 and n-2).
// Writes the per-interval coefficients of c0 + c1 u + c2 u^2 + c3 u^3, u = (t - t_i)/h.
template <class In>
inline void fit_channel(const In* y, int64_t n, double h_, lr::D4* out) {
  typedef long double R;
  const R h = (R)h_;
  std::vector<R> dg(n), up(n), rhs(n), s(n);
  dg[0] = 1; up[0] = 2;
  rhs[0] = (-(R)5 * y[0] + (R)4 * y[1] + (R)y[2]) / ((R)2 * h);
  for (int64_t i = 1; i + 1 < n; ++i) {
    dg[i] = 4; up[i] = 1;
    rhs[i] = (R)3 * ((R)y[i + 1] - (R)y[i - 1]) / h;
  }
  dg[n - 1] = 1; up[n - 1] = 0;
  rhs[n - 1] = ((R)5 * y[n - 1] - (R)4 * y[n - 2] - (R)y[n - 3]) / ((R)2 * h);
  // forward elimination; sub-diagonal is 1 except the last row, where it is 2
  for (int64_t i = 1; i < n; ++i) {
    const R lo = (i == n - 1) ? (R)2 : (R)1;
    const R f = lo / dg[i - 1];
    dg[i] -= f * up[i - 1];
    rhs[i] -= f * rhs[i - 1];
  }
  s[n - 1] = rhs[n - 1] / dg[n - 1];
  for (int64_t i = n - 2; i >= 0; --i) s[i] = (rhs[i] - up[i] * s[i + 1]) / dg[i];
  for (int64_t i = 0; i + 1 < n; ++i) {
    const R dy = (R)y[i + 1] - (R)y[i];
    out[i].x = (double)y[i];
    out[i].y = (double)(h * s[i]);
    out[i].z = (double)((R)3 * dy - h * ((R)2 * s[i] + s[i + 1]));
    out[i].w = (double)(-(R)2 * dy + h * (s[i] + s[i + 1]));
  }
}

// b_k = 1 / prod_{m != k} (k - m), m = -P+1..P  ( = (-1)^(P-k) / ((k+P-1)! (P-k)!) ), k = 1..P
inline void pair_constants(int P, double* bk /* [kPMax+1] */) {
  for (int k = 0; k <= kPMax; ++k) bk[k] = 0.0;
  for (int k = 1; k <= P; ++k) {
    long double den = 1;
    for (int m = -P + 1; m <= P; ++m)
      if (m != k) den *= (long double)(k - m);
    bk[k] = (double)(1.0L / den);
  }
}

}  // namespace lr
