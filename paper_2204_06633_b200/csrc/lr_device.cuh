// lr_device.cuh — per-sample arithmetic of the LISA response (device functions).
//
// Everything here is the product's own restatement of arXiv:2204.06633 (eqs. 10-21); it shares
// nothing with oracle/.  The functions are LR_HD (__host__ __device__) so that a host harness can single-
// step them while debugging; the library itself only ever calls them from kernels.
//
// Numerical design:
//   * the sample index stays an integer; a delay D (in samples) is split as I = ceil(D), eps = I - D in
//     [0,1), and the stencil is addressed with integers only;
//   * Lagrange weights come from the pair factorisation (eps-k)(eps-1+k) = z - k(k-1), z = eps^2 - eps,
//     with prefix/suffix products over the P = (order+1)/2 pairs: no division, regular at eps = 0;
//   * an interpolated value is returned as  x[a] - S  with a = the sample just above the target and S a
//     weighted sum of exact first differences (summation by parts, the constant mode removed
//     structurally), so that differences of interpolations of one series (Delta h in eq. 16, the +/- pairs
//     of eqs. 17-18) lose no digits to cancellation.
#pragma once
#include <math.h>
#include <stdint.h>

#ifdef __CUDACC__
#define LR_HD __host__ __device__ __forceinline__
#else
#define LR_HD inline
#define __host__
#define __device__
#endif

namespace lr {

constexpr int kPMax = 33;        // order <= 65
constexpr double kC = 299792458.0;  // m/s
constexpr int kSplineChannels = 24; // 9 positions, 6 light times, 9 arm-vector components (x_a - x_{a+1})

struct alignas(16) D2 { double x, y; };
struct alignas(32) D4 { double x, y, z, w; };

// link slots [12,23,31,13,32,21] -> receiver / emitter (0-based spacecraft)
__host__ __device__ constexpr int link_rx(int s) { return s == 0 ? 0 : s == 1 ? 1 : s == 2 ? 2 : s == 3 ? 0 : s == 4 ? 2 : 1; }
__host__ __device__ constexpr int link_tx(int s) { return s == 0 ? 1 : s == 1 ? 2 : s == 2 ? 0 : s == 3 ? 2 : s == 4 ? 1 : 0; }
// slot of link (rx i, tx j), 0-based
__host__ __device__ constexpr int link_slot(int i, int j) {
  return (i == 0 && j == 1) ? 0 : (i == 1 && j == 2) ? 1 : (i == 2 && j == 0) ? 2
       : (i == 0 && j == 2) ? 3 : (i == 2 && j == 1) ? 4 : 5;
}
// the circular permutation 1->2->3->1 applied r times to a slot
__host__ __device__ constexpr int rot_slot(int s, int r) {
  return link_slot((link_rx(s) + r) % 3, (link_tx(s) + r) % 3);
}

// Kernel parameters shared by both stages (passed by value).
struct Params {
  const D4* coef;      // DEVICE [kSplineChannels][nint] cubic coefficients (c0,c1,c2,c3) in u = (t - t_i)/h in [0,1)
  int nint;            // spline intervals = n_knots - 1
  int p;               // P = (order+1)/2
  double trel0;        // t0 - t_start  [s]
  double dt;           // sample spacing [s]
  double inv_h;        // 1 / knot_dt
  double inv_dt;       // 1 / dt
  double inv_cdt;      // 1 / (c dt)
  int n;               // samples this launch processes: local indices [0, n)
  int n_off;           // global sample index of local sample 0 (time and margins are global)
  int n_glob;          // samples of the whole series
  int rd_lo, rd_hi;    // local index range [rd_lo, rd_hi) in which the input rows may be read (0 outside)
  int64_t in_stride;   // elements between rows (and templates: rows x in_stride) of the input arrays
  int64_t out_stride;  // same for the output array
  int m_proj, m_front, m_back;
  int halo_lo, halo_hi;  // staged window = [n0 - halo_lo, n0 + B + halo_hi)
  int ntiles;
  int fir_wc;            // FIR path: taps per series as stored (padded to a multiple of kFirR)
  int fir_uniform;       // FIR path: 1 = all light times are constant: ONE plan tile (slot 0) serves every tile
  int fir_tile0;         // FIR path: global tile whose geometry plan slot 0 is built from
  int fir_taps;          // FIR path: taps per series that can be non-zero (<= fir_wc; the padding is at the front)
  int chain_sum;         // 0: nested delays (default), 1: eq. 20 sums of the L at t
  int proj_ext;          // 1: LR_Y_EXTENDED (emission delays relative to the reception split, arm-vector splines)
  int proj_pair;         // 1: projection with two consecutive samples per thread (LR_PROJ_PAIR; same bits)
  double bk[kPMax + 1];  // bk[k] = 1 / prod_{m != k} (k - m), m = -P+1..P, for k = 1..P
};

LR_HD D4 load4(const D4* p) {
#ifdef __CUDA_ARCH__
  const double2 lo = __ldg(reinterpret_cast<const double2*>(p));
  const double2 hi = __ldg(reinterpret_cast<const double2*>(p) + 1);
  return D4{lo.x, lo.y, hi.x, hi.y};
#else
  return *p;
#endif
}

LR_HD double inv_sqrt(double x) {
#ifdef __CUDA_ARCH__
  return rsqrt(x);
#else
  return 1.0 / sqrt(x);
#endif
}

// time of sample n relative to knot 0
LR_HD double sample_trel(const Params& P, int n) { return fma((double)n, P.dt, P.trel0); }

// cubic spline channel `ch` at relative time trel (reading A9)
LR_HD int spline_interval(const Params& P, double trel, double& u) {
  const double s = trel * P.inv_h;
  int i = (int)floor(s);
  i = i < 0 ? 0 : (i > P.nint - 1 ? P.nint - 1 : i);
  u = s - (double)i;
  return i;
}
// where the coefficients of interval i come from: the table in global memory, or the copy of the (at most
// two) intervals of a tile that a kernel staged in shared memory
struct CoefGlobal {
  LR_HD D4 get(const Params& P, int ch, int i) const { return load4(P.coef + (int64_t)ch * P.nint + i); }
};
struct CoefTile {
  const D4* sc;   // [channels staged][2]
  int i0;
  LR_HD D4 get(const Params&, int ch, int i) const { return sc[ch * 2 + (i - i0)]; }
};
template <class Coef>
LR_HD double spline_eval(const Params& P, const Coef& src, int ch, double trel) {
  double u;
  const int i = spline_interval(P, trel, u);
  const D4 c = src.get(P, ch, i);
  return fma(fma(fma(c.w, u, c.z), u, c.y), u, c.x);
}
LR_HD double spline_eval(const Params& P, int ch, double trel) { return spline_eval(P, CoefGlobal{}, ch, trel); }

// Split a delay of D samples: anchor index a = n - ceil(D) + 1 (the sample just above the target
// n - D), eps = ceil(D) - D in [0,1).  Stencil taps are a-P .. a+P-1.
LR_HD void split_delay(double D, int n, int& a, double& eps) {
  const double I = ceil(D);
  eps = I - D;
  a = n - (int)I + 1;
}

// Centred Lagrange interpolation of NS series that share one target, in summation-by-parts form.
//   value_s = raw_s[a] - S[s],   S[s] = sum_{j=1-P}^{0} C_j dif_s[a-1+j] - sum_{j=1}^{P-1} E_j dif_s[a-1+j]
// with C_j = sum_{j'<=j} w_j', E_j = sum_{j'>j} w_j' and dif_s[m] = raw_s[m+1] - raw_s[m].
// `dif(m, out)` fetches the NS first differences at staged index m.  PT > 0 fixes P at compile time.
template <int PT, int NS, class Dif>
LR_HD void interp_sbp(const Params& prm, double eps, int a, Dif dif, double (&S)[NS]) {
  const int P = PT > 0 ? PT : prm.p;
  double R[PT > 0 ? PT : kPMax];
  const double z = fma(eps, eps, -eps);
  // ascending pass: R[k-1] = b_k * prod_{k'<k} G_k',  G_k = (eps-k)(eps-1+k) = z - k(k-1)
  double pre = 1.0;
#pragma unroll
  for (int k = 1; k <= P; ++k) {
    R[k - 1] = pre * prm.bk[k];
    pre *= z - (double)(k * (k - 1));
  }
  // descending pass: complete the pair products, build running sums C (taps below the target, outside
  // in) and E (taps above, outside in), and accumulate against the first differences.
  double suf = 1.0, C = 0.0, E = 0.0;
  double lo[NS], hi[NS];
#pragma unroll
  for (int s = 0; s < NS; ++s) { lo[s] = 0.0; hi[s] = 0.0; }
  const int q = a - 1;
#pragma unroll
  for (int k = P; k >= 1; --k) {
    const double Rk = R[k - 1] * suf;            // b_k prod_{k' != k} G_k'
    suf *= z - (double)(k * (k - 1));
    C = fma(Rk, (double)k - eps, C);             // += w_{1-k}
    double d[NS];
    dif(q + 1 - k, d);
#pragma unroll
    for (int s = 0; s < NS; ++s) lo[s] = fma(C, d[s], lo[s]);
    if (k >= 2) {
      E = fma(Rk, eps + (double)(k - 1), E);     // += w_k
      dif(q + k - 1, d);
#pragma unroll
      for (int s = 0; s < NS; ++s) hi[s] = fma(E, d[s], hi[s]);
    }
  }
#pragma unroll
  for (int s = 0; s < NS; ++s) S[s] = lo[s] - hi[s];
}

// The same for TWO consecutive samples A (anchor a) and B (anchor a + 1) whose targets eps_A, eps_B differ: the two
// stencils overlap in 2P - 2 of their 2P - 1 first differences, so every difference is fetched ONCE (2P fetches
// for the pair instead of 2 (2P - 1)) and used with both weight sets.  Iteration k fetches dif[q+1-k] and dif[q+k],
// q = a - 1: sample A uses them for its low step k and its high step k+1, sample B for its low step k+1 and its
// high step k (B's low step 1 reuses the upper fetch of iteration 1).  Every accumulator receives exactly the
// operations of interp_sbp in the same order, so the results equal two interp_sbp calls bit for bit.
// Compile-time P only.  win(c, out) fetches the NS first differences at index q + c, q = a - 1 (c is a compile-time
// constant after unrolling: the caller can lay the window out so that c becomes an immediate offset).
template <int PT, int NS, class Win>
LR_HD void interp_sbp2(const Params& prm, double epsA, double epsB, Win win, double (&SA)[NS], double (&SB)[NS]) {
  static_assert(PT > 0, "interp_sbp2 needs a compile-time pair count");
  constexpr int P = PT;
  double RA[P], RB[P];
  const double zA = fma(epsA, epsA, -epsA), zB = fma(epsB, epsB, -epsB);
  double preA = 1.0, preB = 1.0;
#pragma unroll
  for (int k = 1; k <= P; ++k) {
    RA[k - 1] = preA * prm.bk[k];
    preA *= zA - (double)(k * (k - 1));
    RB[k - 1] = preB * prm.bk[k];
    preB *= zB - (double)(k * (k - 1));
  }
  double sufA = 1.0, CA = 0.0, EA = 0.0, sufB = 1.0, CB = 0.0, EB = 0.0;
  double loA[NS], hiA[NS], loB[NS], hiB[NS];
#pragma unroll
  for (int s = 0; s < NS; ++s) { loA[s] = 0.0; hiA[s] = 0.0; loB[s] = 0.0; hiB[s] = 0.0; }
#pragma unroll
  for (int k = P; k >= 1; --k) {
    double dL[NS], dH[NS];
    win(1 - k, dL);
    win(k, dH);
    // sample A: low step k; high step k+1 with the E of the previous iteration
    const double RkA = RA[k - 1] * sufA;
    sufA *= zA - (double)(k * (k - 1));
    CA = fma(RkA, (double)k - epsA, CA);
#pragma unroll
    for (int s = 0; s < NS; ++s) loA[s] = fma(CA, dL[s], loA[s]);
    if (k < P) {
#pragma unroll
      for (int s = 0; s < NS; ++s) hiA[s] = fma(EA, dH[s], hiA[s]);
    }
    if (k >= 2) EA = fma(RkA, epsA + (double)(k - 1), EA);
    // sample B (anchor a + 1): low step k+1 with the C of the previous iteration; high step k
    if (k < P) {
#pragma unroll
      for (int s = 0; s < NS; ++s) loB[s] = fma(CB, dL[s], loB[s]);
    }
    const double RkB = RB[k - 1] * sufB;
    sufB *= zB - (double)(k * (k - 1));
    CB = fma(RkB, (double)k - epsB, CB);
    if (k >= 2) {
      EB = fma(RkB, epsB + (double)(k - 1), EB);
#pragma unroll
      for (int s = 0; s < NS; ++s) hiB[s] = fma(EB, dH[s], hiB[s]);
    } else {
#pragma unroll
      for (int s = 0; s < NS; ++s) loB[s] = fma(CB, dH[s], loB[s]);   // B's low step 1: dif[q + 1]
    }
  }
#pragma unroll
  for (int s = 0; s < NS; ++s) { SA[s] = loA[s] - hiA[s]; SB[s] = loB[s] - hiB[s]; }
}

// ---------------------------------------------------------------------------------------------- stage 1
// Geometry of one time sample (eqs. 10-12 and the reception delays of eq. 16): everything that needs the positions
// and the basis, so that only 15 doubles per sample stay live across the nine interpolations.
struct ProjGeom {
  double Dr[3];                          // reception delay k.x_i/c [samples]
  double xip[3], xic[3], kn[3], rden[3]; // per arm (links 12, 23, 31 and their reverses): xi+, xix, k.n, 1/(2(1-k.n)(1+k.n))
};

template <class Coef>
LR_HD void project_geometry(const Params& prm, const Coef& coef, double trel, const double* bs, ProjGeom& g) {
  const double k0 = bs[0], k1 = bs[1], k2 = bs[2];
  const double u0 = bs[3], u1 = bs[4], u2 = bs[5];
  const double v0 = bs[6], v1 = bs[7], v2 = bs[8];
  double x[3][3];
#pragma unroll
  for (int i = 0; i < 3; ++i) {
#pragma unroll
    for (int a = 0; a < 3; ++a) x[i][a] = spline_eval(prm, coef, i * 3 + a, trel);
    g.Dr[i] = (k0 * x[i][0] + k1 * x[i][1] + k2 * x[i][2]) * prm.inv_cdt;   // reception delay k.x_i/c [samples]
  }
  // three arms: arm a joins receiver i = a and emitter j = (a+1)%3 (links 12, 23, 31); the reverse links
  // 21, 32, 13 share xi+ and xix and flip the sign of k.n
#pragma unroll
  for (int arm = 0; arm < 3; ++arm) {
    const int i = arm, j = (arm + 1) % 3;
    const double d0 = x[i][0] - x[j][0], d1 = x[i][1] - x[j][1], d2 = x[i][2] - x[j][2];
    const double inv = inv_sqrt(d0 * d0 + d1 * d1 + d2 * d2);
    const double n0v = d0 * inv, n1v = d1 * inv, n2v = d2 * inv;  // emitter j -> receiver i
    const double un = u0 * n0v + u1 * n1v + u2 * n2v;
    const double vn = v0 * n0v + v1 * n1v + v2 * n2v;
    g.kn[arm] = k0 * n0v + k1 * n1v + k2 * n2v;
    // eq. 16 divides by 2 (1 - k.n) on one link of the arm and by 2 (1 + k.n) on the other: one reciprocal,
    // 1 / (2 (1 - k.n)(1 + k.n)), computed here, serves both (an fp64 division is ~25 instructions and a branch;
    // six of them at the end of the links' dependency chains, plus 1/sqrt as two operations, were 8 % of the
    // kernel)
    g.rden[arm] = 1.0 / (2.0 * ((1.0 - g.kn[arm]) * (1.0 + g.kn[arm])));
    g.xip[arm] = un * un - vn * vn;   // eq. 12
    g.xic[arm] = 2.0 * un * vn;
  }
}

LR_HD int clamp_anchor(int v, int lo, int hi) { return v < lo ? lo : (v > hi ? hi : v); }

// One time sample of eqs. 10-16 for all six links.  raw/dif: staged (h+, hx) pairs and their first
// differences, W entries; nl = this sample's staged index; bs = k(3), u(3), v(3).  y6[slot] receives y_ij.
//
// EXT (LR_Y_EXTENDED): the same sample with the delays formed so that y is good to a few fp64 roundings instead of ~2e-14.
// What limits the plain form is not the interpolation but the DELAYS: k.x_i/c is ~500 s (50-100 samples), so the
// fp64 value of a delay carries 7e-15 samples of rounding, and Delta h = h(t_e) - h(t_r) with t_e - t_r ~ 1 sample sees
// it as a relative error of 1e-14 (which TDI then amplifies by up to 1e6 in the T channel).  Here
//   * the arm vectors x_i - x_j come from their own splines (channels 15..23, fitted to the exact differences of the
//     table values: the same function, without the rounding of two 1.5e11 m positions); only spacecraft 1 is located
//     by its position spline, k.x_2/c and k.x_3/c follow from the arm vectors (18 spline evaluations per sample), and
//   * an emission time is placed RELATIVE to its reception time: with D_r = I_r - eps_r split exactly,
//     D_e - D_r = L_ij/dt -+ k.(x_i - x_j)/(c dt) =: dD is a small number known to ~1e-16 samples, and
//     u = dD - eps_r, I_e = I_r + ceil(u), eps_e = ceil(u) - u.  The rounding of D_r itself then moves BOTH times
//     together, which changes Delta h by w dt * 7e-15 only.
template <int PT, bool EXT, class Store, class Coef = CoefGlobal>
LR_HD void project_sample(const Params& prm, const D2* raw, const D2* dif, int W, int nl, double trel,
                          const double* bs, Store store, const Coef& coef = Coef{}) {
  // geometry first (everything that needs the positions and the basis), so that only 12 doubles stay live
  // across the nine interpolations: Dr[3] and, per arm, xi+, xix, k.n
  double Dr[3], xip[3], xic[3], kn[3], rden[3];
  double kd[EXT ? 3 : 1];   // EXT: k.(x_i - x_j)/c [samples] per arm
  {
    const double k0 = bs[0], k1 = bs[1], k2 = bs[2];
    const double u0 = bs[3], u1 = bs[4], u2 = bs[5];
    const double v0 = bs[6], v1 = bs[7], v2 = bs[8];
    double x[3][3];
    if constexpr (EXT) {   // reception delay of spacecraft 1 from its position; the other two follow from the arms
#pragma unroll
      for (int a = 0; a < 3; ++a) x[0][a] = spline_eval(prm, coef, a, trel);
      Dr[0] = (k0 * x[0][0] + k1 * x[0][1] + k2 * x[0][2]) * prm.inv_cdt;
    } else {
#pragma unroll
      for (int i = 0; i < 3; ++i) {
#pragma unroll
        for (int a = 0; a < 3; ++a) x[i][a] = spline_eval(prm, coef, i * 3 + a, trel);
        Dr[i] = (k0 * x[i][0] + k1 * x[i][1] + k2 * x[i][2]) * prm.inv_cdt;   // reception delay k.x_i/c [samples]
      }
    }
    // three arms: arm a joins receiver i = a and emitter j = (a+1)%3 (links 12, 23, 31); the reverse links
    // 21, 32, 13 share xi+ and xix and flip the sign of k.n
#pragma unroll
    for (int arm = 0; arm < 3; ++arm) {
      const int i = arm, j = (arm + 1) % 3;
      double d0, d1, d2;
      if constexpr (EXT) {
        d0 = spline_eval(prm, coef, 15 + arm * 3, trel);
        d1 = spline_eval(prm, coef, 16 + arm * 3, trel);
        d2 = spline_eval(prm, coef, 17 + arm * 3, trel);
        kd[arm] = (k0 * d0 + k1 * d1 + k2 * d2) * prm.inv_cdt;
        if (arm < 2) Dr[arm + 1] = Dr[arm] - kd[arm];   // k.x_j/c = k.x_i/c - k.(x_i - x_j)/c
      } else {
        d0 = x[i][0] - x[j][0]; d1 = x[i][1] - x[j][1]; d2 = x[i][2] - x[j][2];
      }
      const double inv = inv_sqrt(d0 * d0 + d1 * d1 + d2 * d2);
      const double n0v = d0 * inv, n1v = d1 * inv, n2v = d2 * inv;  // emitter j -> receiver i
      const double un = u0 * n0v + u1 * n1v + u2 * n2v;
      const double vn = v0 * n0v + v1 * n1v + v2 * n2v;
      kn[arm] = k0 * n0v + k1 * n1v + k2 * n2v;
      // eq. 16 divides by 2 (1 - k.n) on one link of the arm and by 2 (1 + k.n) on the other: one reciprocal,
      // 1 / (2 (1 - k.n)(1 + k.n)), computed here, serves both (an fp64 division is ~25 instructions and a branch;
      // six of them at the end of the links' dependency chains, plus 1/sqrt as two operations, were 8 % of the
      // kernel)
      rden[arm] = 1.0 / (2.0 * ((1.0 - kn[arm]) * (1.0 + kn[arm])));
      xip[arm] = un * un - vn * vn;   // eq. 12
      xic[arm] = 2.0 * un * vn;
    }
  }

  auto fetch = [&](int m, double (&d)[2]) {
    const D2 v = dif[m];
    d[0] = v.x; d[1] = v.y;
  };
  const int a_min = PT > 0 ? PT : prm.p, a_max = W - (PT > 0 ? PT : prm.p);
  auto clampi = [](int v, int lo, int hi) { return v < lo ? lo : (v > hi ? hi : v); };

  // receiver by receiver: h at the reception time t - k.x_i/c (shared by the two links received at i), then the two
  // emission times of those links; only one receiver's reception sums are live at a time
#pragma unroll
  for (int i = 0; i < 3; ++i) {
    double Sr[2], er;
    int ar;
    split_delay(Dr[i], nl, ar, er);
    ar = clampi(ar, a_min, a_max);   // (only ever moves the anchor of a sample inside the margins: zeroed)
    interp_sbp<PT, 2>(prm, er, ar, fetch, Sr);
    const D2 rr = raw[ar];
#pragma unroll
    for (int l = 0; l < 2; ++l) {
      // the links received at i: from j = (i+1)%3 (slot i: arm i, direction ij) and from (i+2)%3 (the reverse link of
      // arm (i+2)%3)
      const int arm = l == 0 ? i : (i + 2) % 3;
      const int tx = l == 0 ? (i + 1) % 3 : (i + 2) % 3;
      const int slot = link_slot(i, tx);
      const double kappa = l == 0 ? kn[arm] : -kn[arm];
      // emission: t - L_rx,tx(t) - k.x_tx(t)/c.  EXT: relative to the reception split, D_e - D_r = L/dt +
      // k.(x_tx - x_rx)/(c dt) with x_tx - x_rx = -(x_a - x_b) for the link ab of arm ab and +(x_a - x_b) for link ba
      const double De = EXT ? fma(spline_eval(prm, coef, 9 + slot, trel), prm.inv_dt, l == 0 ? -kd[EXT ? arm : 0] : kd[EXT ? arm : 0]) - er
                            : fma(spline_eval(prm, coef, 9 + slot, trel), prm.inv_dt, Dr[tx]);
      int ae;
      double eps, Se[2];
      split_delay(De, EXT ? ar - 1 : nl, ae, eps);
      ae = clampi(ae, a_min, a_max);
      interp_sbp<PT, 2>(prm, eps, ae, fetch, Se);
      const D2 re = raw[ae];
      const double dhp = (re.x - rr.x) - Se[0] + Sr[0];
      const double dhc = (re.y - rr.y) - Se[1] + Sr[1];
      store(slot, (xip[arm] * dhp + xic[arm] * dhc) * ((1.0 + kappa) * rden[arm]));  // eq. 16: / (2 (1 - kappa))
    }
  }
}

// Two consecutive samples per thread (staged indices nl = A and nl + 1 = B).  Each of the nine interpolation times of
// B lies ~1e-4 samples from A's shifted by one sample (|d/dt (k.x/c)| <= 1e-4, |dL/dt| <= 1e-7), so the stencils of a
// pair share all but one first difference and interp_sbp2 fetches each from shared memory once.  Where the integer
// parts of the two delays differ (the fraction wrapped between A and B: about one pair in 1e4) the pair takes two
// single-sample interpolations (out of line: it is rare and would triple the code).  Results equal project_sample's
// bit for bit.
//
// To keep the register count of the pair near that of a single sample, the thread first writes the geometry of both
// samples (project_geometry's 15 numbers, the six emission delays and the six link factors (1 +- k.n) / (2 (1 -
// k.n)(1 + k.n))) to a private column of shared memory, geo[kGeoFields][nthreads], and then walks the three RECEIVERS
// in a rolled loop: reception at i, then the two links received at i.
constexpr int kGeoDr = 0, kGeoDe = 3, kGeoXip = 9, kGeoXic = 12, kGeoF = 15, kGeoPerSample = 21;
constexpr int kGeoFields = 2 * kGeoPerSample;

template <class Coef>
LR_HD void project_geometry_store(const Params& prm, const Coef& coef, double trel, const double* bs, double* geo,
                                  int stride) {
  ProjGeom g;
  project_geometry(prm, coef, trel, bs, g);
#pragma unroll
  for (int i = 0; i < 3; ++i) {
    geo[(kGeoDr + i) * stride] = g.Dr[i];
    geo[(kGeoXip + i) * stride] = g.xip[i];
    geo[(kGeoXic + i) * stride] = g.xic[i];
  }
#pragma unroll
  for (int arm = 0; arm < 3; ++arm) {
    const int i = arm, j = (arm + 1) % 3;
#pragma unroll
    for (int dir = 0; dir < 2; ++dir) {
      const int rx = dir == 0 ? i : j, tx = dir == 0 ? j : i;
      const int slot = link_slot(rx, tx);
      const double kappa = dir == 0 ? g.kn[arm] : -g.kn[arm];
      // emission: t - L_rx,tx(t) - k.x_tx(t)/c
      geo[(kGeoDe + slot) * stride] = fma(spline_eval(prm, coef, 9 + slot, trel), prm.inv_dt, g.Dr[tx]);
      geo[(kGeoF + slot) * stride] = (1.0 + kappa) * g.rden[arm];   // eq. 16: 1 / (2 (1 - kappa))
    }
  }
}

#ifdef __CUDACC__
// interp_sbp<PT, 2> on the staged (h+, hx) differences as an out-of-line call with rolled loops (the rare path of
// project_pair; bk: the pair constants in shared memory, so that no kernel parameter has its address taken).  Same
// operations in the same order as interp_sbp, hence the same bits.
template <int PT>
__device__ __noinline__ void interp_sbp_rolled(const double* bk, double eps, int a, const D2* dif_e, const D2* dif_o,
                                               double* S) {
  auto dif_at = [&](int m) { return (m & 1) ? dif_o[m >> 1] : dif_e[m >> 1]; };
  double R[PT];
  const double z = fma(eps, eps, -eps);
  double pre = 1.0;
#pragma unroll 1
  for (int k = 1; k <= PT; ++k) {
    R[k - 1] = pre * bk[k];
    pre *= z - (double)(k * (k - 1));
  }
  double suf = 1.0, C = 0.0, E = 0.0, lo0 = 0.0, lo1 = 0.0, hi0 = 0.0, hi1 = 0.0;
  const int q = a - 1;
#pragma unroll 1
  for (int k = PT; k >= 1; --k) {
    const double Rk = R[k - 1] * suf;
    suf *= z - (double)(k * (k - 1));
    C = fma(Rk, (double)k - eps, C);
    const D2 d = dif_at(q + 1 - k);
    lo0 = fma(C, d.x, lo0);
    lo1 = fma(C, d.y, lo1);
    if (k >= 2) {
      E = fma(Rk, eps + (double)(k - 1), E);
      const D2 e = dif_at(q + k - 1);
      hi0 = fma(E, e.x, hi0);
      hi1 = fma(E, e.y, hi1);
    }
  }
  S[0] = lo0 - hi0;
  S[1] = lo1 - hi1;
}

// geo: this thread's column (element f of sample A at geo[f * stride], of sample B at geo[(kGeoPerSample + f) * stride]).
// The first differences are staged DE-INTERLEAVED, dif_e[i] = dif[2 i], dif_o[i] = dif[2 i + 1]: the lanes of a warp
// own every other sample, so with the plain layout their 16-byte reads of one tap would be 32 bytes apart (a two-way
// bank conflict on every load: measured, 52.7 M conflicts in one year); de-interleaved, the lanes read consecutive
// elements.  For a window anchored at q the tap q + c lies at (c even ? pe : po)[c >> 1] with two base pointers chosen
// by the parity of q, so every tap is still an immediate offset.
// bk_s: prm.bk in shared memory.  store(slot, yA, yB).
template <int PT, class Store>
__device__ __forceinline__ void project_pair(const Params& prm, const D2* raw, const D2* dif_e, const D2* dif_o, int W,
                                             int nl, const double* geo, int stride, const double* bk_s, Store store) {
  constexpr int a_min = PT;
  const int a_max = W - PT;
  auto interp2 = [&](double DA, double DB, int& aA, int& aB, double (&SA)[2], double (&SB)[2]) {
    double eA, eB;
    split_delay(DA, nl, aA, eA);
    split_delay(DB, nl + 1, aB, eB);
    aA = clamp_anchor(aA, a_min, a_max);
    aB = clamp_anchor(aB, a_min, a_max);
    if (aB == aA + 1) {
      const int q = aA - 1, q2 = q >> 1;
      const D2* pe = (q & 1) ? dif_o + q2 : dif_e + q2;        // taps q + c, c even
      const D2* po = (q & 1) ? dif_e + q2 + 1 : dif_o + q2;    // taps q + c, c odd
      auto win = [&](int c, double (&d)[2]) {
        const D2 v = (c & 1) ? po[c >> 1] : pe[c >> 1];
        d[0] = v.x; d[1] = v.y;
      };
      interp_sbp2<PT, 2>(prm, eA, eB, win, SA, SB);
    } else {
      interp_sbp_rolled<PT>(bk_s, eA, aA, dif_e, dif_o, SA);
      interp_sbp_rolled<PT>(bk_s, eB, aB, dif_e, dif_o, SB);
    }
  };
  const double* gA = geo;
  const double* gB = geo + kGeoPerSample * stride;
#pragma unroll 1
  for (int i = 0; i < 3; ++i) {   // receiver
    double SrA[2], SrB[2];
    int arA, arB;
    interp2(gA[(kGeoDr + i) * stride], gB[(kGeoDr + i) * stride], arA, arB, SrA, SrB);
    const D2 rrA = raw[arA], rrB = raw[arB];
#pragma unroll
    for (int l = 0; l < 2; ++l) {
      // the two links received at i: from (i+1)%3 (slot i, arm i) and from (i+2)%3 (the reverse link of arm (i+2)%3)
      const int slot = l == 0 ? i : (i == 0 ? 3 : i == 1 ? 5 : 4);
      const int arm = l == 0 ? i : (i == 0 ? 2 : i - 1);
      int aeA, aeB;
      double SeA[2], SeB[2];
      interp2(gA[(kGeoDe + slot) * stride], gB[(kGeoDe + slot) * stride], aeA, aeB, SeA, SeB);
      double yA, yB;
      {
        const D2 re = raw[aeA];
        const double dhp = (re.x - rrA.x) - SeA[0] + SrA[0];
        const double dhc = (re.y - rrA.y) - SeA[1] + SrA[1];
        yA = (gA[(kGeoXip + arm) * stride] * dhp + gA[(kGeoXic + arm) * stride] * dhc) * gA[(kGeoF + slot) * stride];
      }
      {
        const D2 re = raw[aeB];
        const double dhp = (re.x - rrB.x) - SeB[0] + SrB[0];
        const double dhc = (re.y - rrB.y) - SeB[1] + SrB[1];
        yB = (gB[(kGeoXip + arm) * stride] * dhp + gB[(kGeoXic + arm) * stride] * dhc) * gB[(kGeoF + slot) * stride];
      }
      store(slot, yA, yB);
    }
  }
}
#endif

// ---------------------------------------------------------------------------------------------- stage 2
// X's two delay chains (eqs. 17-18): term k of chain A is + y_{A[k]} delayed by the
// first k links of A, term k of chain B is - y_{B[k]} delayed by the first k links of B; k = 0..3 is the
// first generation, k = 0..7 the second.  Term k^2 of A and term k of B carry the same series.
// slots: chain A = 13 31 12 21 12 21 13 31, chain B = 12 21 13 31 13 31 12 21
__host__ __device__ constexpr int chain_a(int k) { return k == 0 ? 3 : k == 1 ? 2 : k == 2 ? 0 : k == 3 ? 5 : k == 4 ? 0 : k == 5 ? 5 : k == 6 ? 3 : 2; }
__host__ __device__ constexpr int chain_b(int k) { return k == 0 ? 0 : k == 1 ? 5 : k == 2 ? 3 : k == 3 ? 2 : k == 4 ? 3 : k == 5 ? 2 : k == 6 ? 0 : 5; }

// One time sample of eqs. 17-18 for X, Y, Z.  raw/dif: six staged series [6][W] and first differences.
// prm.chain_sum 0: nested delays, 1: eq. 20 sums.
template <int PT, int GEN>
LR_HD void tdi_sample(const Params& prm, const double* raw, const double* dif, int W, int nl, double trel,
                      double (&xyz)[3]) {
  constexpr int NK = GEN == 1 ? 4 : 8;
  const int a_min = PT > 0 ? PT : prm.p, a_max = W - (PT > 0 ? PT : prm.p);
  auto clampi = [](int v, int lo, int hi) { return v < lo ? lo : (v > hi ? hi : v); };

  const bool sum_mode = prm.chain_sum != 0;
  double Lt[6] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0};
  if (sum_mode) {  // eq. 20: every L at t
#pragma unroll
    for (int s = 0; s < 6; ++s) Lt[s] = spline_eval(prm, 9 + s, trel);
  }
#pragma unroll
  for (int ch = 0; ch < 3; ++ch) {  // Y, Z: every index of X rotated 1->2->3->1
    int aA[NK];
    double acc = 0.0;
    {
      double d = 0.0;
#pragma unroll
      for (int k = 0; k < NK; ++k) {
        const int s = rot_slot(chain_a(k), ch);
        if (k == 0) {
          aA[k] = nl;
        } else {
          double eps, S[1];
          split_delay(d * prm.inv_dt, nl, aA[k], eps);
          aA[k] = clampi(aA[k], a_min, a_max);
          const double* ds = dif + s * W;
          interp_sbp<PT, 1>(prm, eps, aA[k], [&](int m, double (&o)[1]) { o[0] = ds[m]; }, S);
          acc -= S[0];
        }
        if (k + 1 < NK) d += sum_mode ? Lt[s] : spline_eval(prm, 9 + s, trel - d);
      }
    }
    {
      double d = 0.0;
#pragma unroll
      for (int k = 0; k < NK; ++k) {
        const int s = rot_slot(chain_b(k), ch);
        int aB = nl;
        if (k > 0) {
          double eps, S[1];
          split_delay(d * prm.inv_dt, nl, aB, eps);
          aB = clampi(aB, a_min, a_max);
          const double* ds = dif + s * W;
          interp_sbp<PT, 1>(prm, eps, aB, [&](int m, double (&o)[1]) { o[0] = ds[m]; }, S);
          acc += S[0];
        }
        // same series: + y_s at the anchor of A's term k^2, - y_s at this term's anchor
        acc += raw[s * W + aA[k ^ 2]] - raw[s * W + aB];
        if (k + 1 < NK) d += sum_mode ? Lt[s] : spline_eval(prm, 9 + s, trel - d);
      }
    }
    xyz[ch] = acc;
  }
}

// Source basis (eq. 10) with the polarisation angle applied to (u, v) (reading A4):
// out[0..2] = k, out[3..5] = u, out[6..8] = v.  Runs in source_basis_kernel (one thread per template).
LR_HD void source_basis(double beta, double lam, double psi, double* out) {
  const double cb = cos(beta), sb = sin(beta), cl = cos(lam), sl = sin(lam);
  const double k[3] = {-cb * cl, -cb * sl, -sb};
  const double u0[3] = {sl, -cl, 0.0};                 // -e_phi
  const double v0[3] = {-sb * cl, -sb * sl, cb};       // -e_theta
  const double cp = cos(psi), sp = sin(psi);
  for (int a = 0; a < 3; ++a) {
    out[a] = k[a];
    out[3 + a] = u0[a] * cp + v0[a] * sp;
    out[6 + a] = -u0[a] * sp + v0[a] * cp;
  }
}

}  // namespace lr
