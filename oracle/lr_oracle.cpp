// lr_oracle.cpp — CPU ORACLE for the generic time-domain LISA response.
//
// THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke()
// and bench.py's cpu_baseline / `--impl reference` legs may build, load or call it.
// It shares no code, header, table or constant generator with the CUDA library under
// paper_2204_06633_b200/csrc/, and neither side includes or imports the other.
//
// What it is: a plain, slow, step-by-step statement of the algorithm of
// arXiv:2204.06633, written in the paper's order and notation, templated
// on the scalar type S (long double = parity truth, double = the timed CPU baseline).
// There is no blocking, fusion, reordering or fast weight formula: every Lagrange
// weight is the naive O(T^2) product.  The method is a discretisation (Lagrange
// interpolation of sampled series over splined orbits), so the oracle is the
// algorithm itself; the continuous-time definition pins it from outside
// (tests/test_oracle_pins.py, pins P1-P11 of SURVEY.md §8(c) / DESIGN.md §4).
//
// Passages followed (PAPER.md line : equation):
//   source basis k,u,v ............ 130-136 : eq. 10
//   polarisation rotation by psi .. 105-108 : eq. 9 (rotation matrix only; the iota
//                                     factors belong to the caller's waveform, reading A4)
//   antenna terms xi+, xix ........ 152-157 : eq. 12;   H_ij: 142 : eq. 11
//   single-link response y_ij ..... 181     : eq. 16
//   TDI X1, X2 ..................... 193-197 : eqs. 17-18; Y, Z by 1->2->3->1 (116, 210)
//   delay operator, chained delays  203-208 : eqs. 19-20 (SUM); NESTED per BASELINE north_star
//   A, E, T ........................ 216-223 : eq. 21
//   orbit interpolation ........... 263 ("interpolated and then evaluated at each time step")
//   centred Lagrange interpolation  265
// Readings of silent / ambiguous points (A1..A16) are listed in DESIGN.md §3.
//
// Pins: every function below is pinned (no "parity unpinned" entries):
//   lagrange_weight/interp -> P1 ; Spline -> P9 ; project -> P2, P5, P8, P4 ;
//   tdi -> P2, P3, P5, P7, P10, P4 ; aet -> P6 ; margins -> brute-force reach test.

#include <cmath>
#include <cstdint>
#include <cstring>
#include <new>
#include <vector>

namespace {

constexpr double C_LIGHT = 299792458.0;  // m/s (reading A13)

// link slots [12, 23, 31, 13, 32, 21]: receiver i, emitter j
constexpr int LINK_I[6] = {1, 2, 3, 1, 3, 2};
constexpr int LINK_J[6] = {2, 3, 1, 3, 2, 1};

int slot_of(int i, int j) {
  for (int s = 0; s < 6; ++s)
    if (LINK_I[s] == i && LINK_J[s] == j) return s;
  return -1;
}

// ------------------------------------------------------------------ O1: cubic spline
// C^2 cubic spline on uniform knots with not-a-knot ends (reading A9), stored as knot
// values y and knot second derivatives m.
template <class S>
struct Spline {
  int64_t nk = 0;
  S t0 = 0, h = 1;
  std::vector<S> y, m;

  void fit(const double* v, int64_t n, double t_start, double knot_dt) {
    nk = n; t0 = (S)t_start; h = (S)knot_dt;
    y.resize(n); m.assign(n, (S)0);
    for (int64_t i = 0; i < n; ++i) y[i] = (S)v[i];
    // interior C^2 conditions: m[i-1] + 4 m[i] + m[i+1] = r[i] = 6 (y[i-1] - 2 y[i] + y[i+1]) / h^2
    std::vector<S> r(n, (S)0);
    for (int64_t i = 1; i + 1 < n; ++i) r[i] = (S)6 * (y[i - 1] - (S)2 * y[i] + y[i + 1]) / (h * h);
    // not-a-knot: third derivative continuous at knots 1 and n-2:
    //   m[0] - 2 m[1] + m[2] = 0   and   m[n-3] - 2 m[n-2] + m[n-1] = 0.
    // Substituted into rows 1 and n-2 they give 6 m[1] = r[1] and 6 m[n-2] = r[n-2].
    m[1] = r[1] / (S)6;
    m[n - 2] = r[n - 2] / (S)6;
    int64_t lo = 2, hi = n - 3;  // remaining unknowns, tridiagonal (1, 4, 1)
    if (hi >= lo) {
      int64_t k = hi - lo + 1;
      std::vector<S> cp(k), dp(k);
      for (int64_t a = 0; a < k; ++a) {
        int64_t i = lo + a;
        S rhs = r[i];
        if (i == lo) rhs -= m[1];
        if (i == hi) rhs -= m[n - 2];
        S sub = (a == 0) ? (S)0 : (S)1, sup = (a == k - 1) ? (S)0 : (S)1;
        S den = (S)4 - sub * (a ? cp[a - 1] : (S)0);
        cp[a] = sup / den;
        dp[a] = (rhs - sub * (a ? dp[a - 1] : (S)0)) / den;
      }
      for (int64_t a = k - 1; a >= 0; --a) m[lo + a] = dp[a] - ((a == k - 1) ? (S)0 : cp[a] * m[lo + a + 1]);
    }
    m[0] = (S)2 * m[1] - m[2];
    m[n - 1] = (S)2 * m[n - 2] - m[n - 3];
  }

  S eval(S t) const {
    S s = (t - t0) / h;
    int64_t i = (int64_t)std::floor(s);
    if (i < 0) i = 0;
    if (i > nk - 2) i = nk - 2;
    S u = (t - (t0 + (S)i * h)) / h, v = (S)1 - u;
    return v * y[i] + u * y[i + 1] + h * h / (S)6 * ((v * v * v - v) * m[i] + (u * u * u - u) * m[i + 1]);
  }
};

// ------------------------------------------------------------------ O6: Lagrange
// Weight of tap j (j = -p+1 .. p) at fractional position eps in [0,1):
//   w_j(eps) = prod_{m != j} (eps - m) / (j - m)          (naive product, reading A5)
template <class S>
S lagrange_weight(int p, int j, S eps) {
  S w = 1;
  for (int mm = -p + 1; mm <= p; ++mm)
    if (mm != j) w *= (eps - (S)mm) / (S)(j - mm);
  return w;
}

// x evaluated D samples before sample n:  I = ceil(D), eps = I - D, q = n - I,
// result = sum_j w_j(eps) x[q + j].  n stays an integer throughout.
template <class S, class In>
S interp(const In* x, int64_t n, S D, int p) {
  S I = std::ceil(D);
  S eps = I - D;
  int64_t q = n - (int64_t)I;
  S acc = 0;
  for (int j = -p + 1; j <= p; ++j) acc += lagrange_weight<S>(p, j, eps) * (S)x[q + j];
  return acc;
}

template <class S>
struct Orbits {
  Spline<S> x[3][3];  // [spacecraft][xyz]
  Spline<S> L[6];     // light travel times [s], link slots
};

struct Margins { int64_t proj, tdi_front, tdi_back; };

}  // namespace

struct orc_handle {
  double dt, t0;
  int order, p;
  double r_max, l_max, t_first, t_last;
  Orbits<long double> ld;
  Orbits<double> d;
  template <class S> const Orbits<S>& orb() const;
  Margins margins(int gen) const {
    // reading A8: fixed margins from table maxima; outputs inside them are exactly 0
    Margins mg;
    mg.proj = (int64_t)std::ceil((1.001 * r_max / C_LIGHT + 1.001 * l_max) / dt) + p + 2;
    int64_t nl = (gen == 1) ? 4 : 8;
    mg.tdi_front = mg.proj + (int64_t)std::ceil((double)nl * 1.001 * l_max / dt) + p + 2;
    mg.tdi_back = mg.proj + p + 2;
    return mg;
  }
};
template <> const Orbits<long double>& orc_handle::orb<long double>() const { return ld; }
template <> const Orbits<double>& orc_handle::orb<double>() const { return d; }

namespace {

// ------------------------------------------------------------------ O2-O7: projection
template <class S, class In, class Out>
void project(const orc_handle& H, const In* hp, const In* hc, int64_t n, double beta_, double lam_, double psi_,
             int64_t lo, int64_t hi, Out* y) {
  const Orbits<S>& O = H.orb<S>();
  const int p = H.p;
  const S dt = (S)H.dt, t0 = (S)H.t0, c = (S)C_LIGHT;
  const S beta = (S)beta_, lam = (S)lam_, psi = (S)psi_;
  // O2, eq. 10
  const S er[3] = {std::cos(beta) * std::cos(lam), std::cos(beta) * std::sin(lam), std::sin(beta)};
  const S eth[3] = {std::sin(beta) * std::cos(lam), std::sin(beta) * std::sin(lam), -std::cos(beta)};
  const S eph[3] = {-std::sin(lam), std::cos(lam), (S)0};
  S k[3], u[3], v[3];
  for (int a = 0; a < 3; ++a) { k[a] = -er[a]; u[a] = -eph[a]; v[a] = -eth[a]; }
  // O3, eq. 9: the waveform is rotated by 2 psi (done per tap below)
  const S c2 = std::cos((S)2 * psi), s2 = std::sin((S)2 * psi);
  const Margins mg = H.margins(1);

#pragma omp parallel for schedule(static)
  for (int64_t nn = lo; nn < hi; ++nn) {
    if (nn < mg.proj || nn >= n - mg.proj) {
      for (int s = 0; s < 6; ++s) y[(int64_t)s * n + nn] = (Out)0;
      continue;
    }
    const S t = t0 + (S)nn * dt;
    S x[3][3];
    for (int i = 0; i < 3; ++i)
      for (int a = 0; a < 3; ++a) x[i][a] = O.x[i][a].eval(t);
    for (int s = 0; s < 6; ++s) {
      const int i = LINK_I[s] - 1, j = LINK_J[s] - 1;
      // O4: link unit vector, emitter j -> receiver i, both positions at reception time t (A2)
      S d[3], dn = 0;
      for (int a = 0; a < 3; ++a) { d[a] = x[i][a] - x[j][a]; dn += d[a] * d[a]; }
      dn = std::sqrt(dn);
      S un = 0, vn = 0, kn = 0, kxi = 0, kxj = 0;
      for (int a = 0; a < 3; ++a) {
        const S na = d[a] / dn;
        un += u[a] * na; vn += v[a] * na; kn += k[a] * na;
        kxi += k[a] * x[i][a]; kxj += k[a] * x[j][a];
      }
      const S xip = un * un - vn * vn, xic = (S)2 * un * vn;  // eq. 12
      // O5: delays in samples (A1: L is a light travel TIME)
      const S Dr = (kxi / c) / dt;
      const S De = (O.L[s].eval(t) + kxj / c) / dt;
      // O6: rotated waveform at emission and reception times
      // (the rotation is linear, so rotating the interpolated values equals interpolating
      //  the rotated series; done on the values to keep one code path for In = double)
      const S hpe = interp<S, In>(hp, nn, De, p), hce = interp<S, In>(hc, nn, De, p);
      const S hpr = interp<S, In>(hp, nn, Dr, p), hcr = interp<S, In>(hc, nn, Dr, p);
      const S Hpe = c2 * hpe - s2 * hce, Hce = s2 * hpe + c2 * hce;
      const S Hpr = c2 * hpr - s2 * hcr, Hcr = s2 * hpr + c2 * hcr;
      // O7, eq. 16 with eq. 11
      y[(int64_t)s * n + nn] = (Out)((xip * (Hpe - Hpr) + xic * (Hce - Hcr)) / ((S)2 * ((S)1 - kn)));
    }
  }
}

// ------------------------------------------------------------------ O8-O9: TDI
struct Term { int sign; const char* chain; int si, sj; };
// eqs. 17-18 for X, in the paper's order; first 8 terms are X1.
const Term X_TERMS[16] = {
    {+1, "", 1, 3},        {+1, "13", 3, 1},       {+1, "131", 1, 2},      {+1, "1312", 2, 1},
    {-1, "", 1, 2},        {-1, "12", 2, 1},       {-1, "121", 1, 3},      {-1, "1213", 3, 1},
    {+1, "13121", 1, 2},   {+1, "131212", 2, 1},   {+1, "1312121", 1, 3},  {+1, "13121213", 3, 1},
    {-1, "12131", 1, 3},   {-1, "121313", 3, 1},   {-1, "1213131", 1, 2},  {-1, "12131312", 2, 1}};

inline int rot(int i, int times) {  // circular permutation 1->2->3->1 applied `times` times
  return (i - 1 + times) % 3 + 1;
}

template <class S, class In, class Out>
void tdi(const orc_handle& H, const In* y, int64_t n, int gen, int nested, int channels, int64_t lo, int64_t hi,
         Out* out) {
  const Orbits<S>& O = H.orb<S>();
  const int p = H.p;
  const S dt = (S)H.dt, t0 = (S)H.t0;
  const Margins mg = H.margins(gen);
  const int nterms = (gen == 1) ? 8 : 16;
  const int nout = (channels == 2) ? 6 : 3;
  const S r2 = std::sqrt((S)2), r3 = std::sqrt((S)3), r6 = std::sqrt((S)6);

#pragma omp parallel for schedule(static)
  for (int64_t nn = lo; nn < hi; ++nn) {
    if (nn < mg.tdi_front || nn >= n - mg.tdi_back) {
      for (int c = 0; c < nout; ++c) out[(int64_t)c * n + nn] = (Out)0;
      continue;
    }
    const S t = t0 + (S)nn * dt;
    S xyz[3];
    for (int ch = 0; ch < 3; ++ch) {  // X, Y, Z: indices rotated ch times (A11)
      S acc = 0;
      for (int k = 0; k < nterms; ++k) {
        const Term& T = X_TERMS[k];
        const int len = (int)std::strlen(T.chain);
        S d = 0;  // chain delay in seconds
        for (int a = 0; a + 1 < len; ++a) {
          const int i = rot(T.chain[a] - '0', ch), j = rot(T.chain[a + 1] - '0', ch);
          const int s = slot_of(i, j);
          // eq. 20 (SUM): every L at t.  NESTED (A6): d_k = d_{k-1} + L(t - d_{k-1}), leftmost first.
          d += nested ? O.L[s].eval(t - d) : O.L[s].eval(t);
        }
        const int ss = slot_of(rot(T.si, ch), rot(T.sj, ch));
        const In* ys = y + (int64_t)ss * n;
        const S val = (len == 0) ? (S)ys[nn] : interp<S, In>(ys, nn, d / dt, p);
        acc += (S)T.sign * val;
      }
      xyz[ch] = acc;
    }
    const S A = (xyz[2] - xyz[0]) / r2, E = (xyz[0] - (S)2 * xyz[1] + xyz[2]) / r6,
            T = (xyz[0] + xyz[1] + xyz[2]) / r3;  // eq. 21
    if (channels == 0) { for (int c = 0; c < 3; ++c) out[(int64_t)c * n + nn] = (Out)xyz[c]; }
    else if (channels == 1) { out[nn] = (Out)A; out[n + nn] = (Out)E; out[2 * n + nn] = (Out)T; }
    else {
      for (int c = 0; c < 3; ++c) out[(int64_t)c * n + nn] = (Out)xyz[c];
      out[3 * n + nn] = (Out)A; out[4 * n + nn] = (Out)E; out[5 * n + nn] = (Out)T;
    }
  }
}

}  // namespace

// =========================================================================== C ABI
extern "C" {

// x: [3][3][n_knots] metres; ltt: [6][n_knots] seconds; t0 = time of sample 0.
int orc_create(int64_t n_knots, double t_start, double knot_dt, const double* x, const double* ltt, double dt,
               double t0, int order, orc_handle** out) {
  if (!x || !ltt || !out || n_knots < 4 || dt <= 0 || knot_dt <= 0 || order < 1 || order % 2 == 0) return -1;
  orc_handle* H = new (std::nothrow) orc_handle();
  if (!H) return -2;
  H->dt = dt; H->t0 = t0; H->order = order; H->p = (order + 1) / 2;
  H->t_first = t_start; H->t_last = t_start + (double)(n_knots - 1) * knot_dt;
  H->r_max = 0; H->l_max = 0;
  for (int64_t k = 0; k < n_knots; ++k)
    for (int i = 0; i < 3; ++i) {
      double r = 0;
      for (int a = 0; a < 3; ++a) { double v = x[((int64_t)i * 3 + a) * n_knots + k]; r += v * v; }
      r = std::sqrt(r);
      if (r > H->r_max) H->r_max = r;
    }
  for (int64_t k = 0; k < 6 * n_knots; ++k)
    if (ltt[k] > H->l_max) H->l_max = ltt[k];
  for (int i = 0; i < 3; ++i)
    for (int a = 0; a < 3; ++a) {
      H->ld.x[i][a].fit(x + ((int64_t)i * 3 + a) * n_knots, n_knots, t_start, knot_dt);
      H->d.x[i][a].fit(x + ((int64_t)i * 3 + a) * n_knots, n_knots, t_start, knot_dt);
    }
  for (int s = 0; s < 6; ++s) {
    H->ld.L[s].fit(ltt + (int64_t)s * n_knots, n_knots, t_start, knot_dt);
    H->d.L[s].fit(ltt + (int64_t)s * n_knots, n_knots, t_start, knot_dt);
  }
  *out = H;
  return 0;
}

void orc_destroy(orc_handle* H) { delete H; }

int orc_margins(const orc_handle* H, int tdi_gen, int64_t* m_proj, int64_t* m_front, int64_t* m_back) {
  Margins mg = H->margins(tdi_gen);
  *m_proj = mg.proj; *m_front = mg.tdi_front; *m_back = mg.tdi_back;
  return 0;
}

// channel 0..8 = x[i][a] (i*3+a), 9..14 = L slots
int orc_spline_eval_ld(const orc_handle* H, int channel, const long double* t, int64_t m, long double* out) {
  for (int64_t k = 0; k < m; ++k)
    out[k] = (channel < 9) ? H->ld.x[channel / 3][channel % 3].eval(t[k]) : H->ld.L[channel - 9].eval(t[k]);
  return 0;
}

// (long double scalars travel by pointer: ctypes would round a by-value long double to double)
int orc_lagrange_weights_ld(int order, const long double* eps, long double* w) {
  const int p = (order + 1) / 2;
  for (int j = -p + 1; j <= p; ++j) w[j + p - 1] = lagrange_weight<long double>(p, j, *eps);
  return 0;
}

// x[len] evaluated D samples before sample n
int orc_interp_ld(const long double* x, int64_t n, const long double* D, int order, long double* out) {
  *out = interp<long double, long double>(x, n, *D, (order + 1) / 2);
  return 0;
}

#define ORC_CHECK_RANGE(n, lo, hi) if (!H || lo < 0 || hi > n || lo > hi) return -1

// y[6][n]; only samples [lo, hi) are written.  Inputs fp64, arithmetic long double.
int orc_project_ld(const orc_handle* H, const double* hp, const double* hc, int64_t n, double beta, double lam,
                   double psi, int64_t lo, int64_t hi, long double* y) {
  ORC_CHECK_RANGE(n, lo, hi);
  project<long double, double, long double>(*H, hp, hc, n, beta, lam, psi, lo, hi, y);
  return 0;
}
int orc_project_ldin(const orc_handle* H, const long double* hp, const long double* hc, int64_t n, double beta,
                     double lam, double psi, int64_t lo, int64_t hi, long double* y) {
  ORC_CHECK_RANGE(n, lo, hi);
  project<long double, long double, long double>(*H, hp, hc, n, beta, lam, psi, lo, hi, y);
  return 0;
}
// the timed CPU baseline: fp64 arithmetic
int orc_project_d(const orc_handle* H, const double* hp, const double* hc, int64_t n, double beta, double lam,
                  double psi, int64_t lo, int64_t hi, double* y) {
  ORC_CHECK_RANGE(n, lo, hi);
  project<double, double, double>(*H, hp, hc, n, beta, lam, psi, lo, hi, y);
  return 0;
}

// y[6][n] -> out[3 or 6][n].  gen 1|2; nested 1 = NESTED, 0 = SUM (eq. 20);
// channels 0 = XYZ, 1 = AET, 2 = XYZ then AET.
int orc_tdi_ld(const orc_handle* H, const double* y, int64_t n, int gen, int nested, int channels, int64_t lo,
               int64_t hi, long double* out) {
  ORC_CHECK_RANGE(n, lo, hi);
  tdi<long double, double, long double>(*H, y, n, gen, nested, channels, lo, hi, out);
  return 0;
}
int orc_tdi_ldin(const orc_handle* H, const long double* y, int64_t n, int gen, int nested, int channels,
                 int64_t lo, int64_t hi, long double* out) {
  ORC_CHECK_RANGE(n, lo, hi);
  tdi<long double, long double, long double>(*H, y, n, gen, nested, channels, lo, hi, out);
  return 0;
}
int orc_tdi_d(const orc_handle* H, const double* y, int64_t n, int gen, int nested, int channels, int64_t lo,
              int64_t hi, double* out) {
  ORC_CHECK_RANGE(n, lo, hi);
  tdi<double, double, double>(*H, y, n, gen, nested, channels, lo, hi, out);
  return 0;
}

}  // extern "C"
