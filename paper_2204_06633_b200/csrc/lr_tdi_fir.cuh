// lr_tdi_fir.cuh — TDI as a slowly time-varying FIR filter (the fast path of lr_tdi).
//
// TDI delays drift by ~1e-8..1e-6 samples per sample (armlength rates of 1-100 m/s against c), so inside
// a tile of a few hundred samples the Lagrange weights of every delayed term are, to rounding, a low-degree
// polynomial in the tile time tau in [-1,1].  Per tile the CTA therefore
//   A  walks the delay chains of eqs. 17-20 at NN nodes of the tile                      (fir_chain_nodes)
//   B  splits every term's delay into an integer shift, fixed over the tile, and eps(node); tiles where a
//      shift could change inside the tile, or where the polynomial model is not safe, are flagged and run
//      the exact per-sample code instead                                                   (fir_split_terms)
//   C  evaluates the summation-by-parts coefficients of every term at the nodes           (fir_node_coeffs)
//   D  merges all terms that act on one series, anchors included, into one coefficient array per
//      (channel, series, power of tau)                                                     (fir_merge)
//   E  applies X(n) = sum_p tau_n^p sum_series sum_m K_p[series][m] * dif_series[n + m]   (fir_apply)
// so the per-sample work drops from 36 weight sets + 36 dot products to 4 series x NN short FIR filters per
// channel.  Interpolating the coefficients through NN Chebyshev-Lobatto nodes costs a relative error
// <= 2 (de/2)^3 (NN = 3) or 1.3 (de/2)^4 (NN = 4) with de the change of eps over the tile; lr_tdi picks NN
// so that this stays below 1e-16 and falls back to the per-sample kernel otherwise.
//
// Each phase is a function of (tid, nthreads) that strides over its work items, so the kernel calls it with
// (threadIdx.x, blockDim.x) between __syncthreads() and a host harness can call it with (0, 1).
#pragma once
#include "lr_device.cuh"

namespace lr {

constexpr int kFirMinBlocks = 7;  // resident apply CTAs per SM the register budget is set for (80 registers: 8 fit)
constexpr int kFirR = 7;          // consecutive samples per thread (odd: conflict-free 64-bit smem reads; R = 5, 9,
                                  // 11 and 14 were measured slower)
constexpr int kFirKStride = 4;    // doubles per (series, m) coefficient record (NN <= 4)

// series used by channel X, in "local" order 13, 31, 12, 21; Y and Z rotate the slots
__host__ __device__ constexpr int fir_base_slot(int sl) { return sl == 0 ? 3 : sl == 1 ? 2 : sl == 2 ? 0 : 5; }
// local series of term k of chain A / chain B
__host__ __device__ constexpr int fir_sl_a(int k) { return k == 0 ? 0 : k == 1 ? 1 : k == 2 ? 2 : k == 3 ? 3 : k == 4 ? 2 : k == 5 ? 3 : k == 6 ? 0 : 1; }
__host__ __device__ constexpr int fir_sl_b(int k) { return fir_sl_a(k ^ 2); }

LR_HD int rot_slot_rt(int s, int r) {
  const int rx = (s == 0 || s == 3) ? 0 : (s == 1 || s == 5) ? 1 : 2;
  const int tx = (s == 2 || s == 5) ? 0 : (s == 0 || s == 4) ? 1 : 2;
  const int i = (rx + r) % 3, j = (tx + r) % 3;
  return (i == 0 && j == 1) ? 0 : (i == 1 && j == 2) ? 1 : (i == 2 && j == 0) ? 2
       : (i == 0 && j == 2) ? 3 : (i == 2 && j == 1) ? 4 : 5;
}

// the link slots of the four series of channel ch (X, Y, Z = rotation by ch), three bits each
__host__ __device__ constexpr int fir_slot_word(int ch) {
  return rot_slot(fir_base_slot(0), ch) | rot_slot(fir_base_slot(1), ch) << 3 | rot_slot(fir_base_slot(2), ch) << 6 |
         rot_slot(fir_base_slot(3), ch) << 9;
}

template <int NN> LR_HD double fir_node(int i);
template <> LR_HD double fir_node<3>(int i) { return i == 0 ? -1.0 : i == 1 ? 0.0 : 1.0; }
template <> LR_HD double fir_node<4>(int i) { return i == 0 ? -1.0 : i == 1 ? -0.5 : i == 2 ? 0.5 : 1.0; }

// Per-tile scratch in shared memory (the kernel carves it out of dynamic smem).
template <int GEN, int NN>
struct FirTile {
  static constexpr int NK = GEN == 1 ? 4 : 8;        // terms per chain (term 0 has no delay)
  static constexpr int NT = 6 * (NK - 1);            // delayed terms of X, Y, Z
  double dnode[6][NN][NK];                           // chain delay d_k [s] at the nodes, [ch*2+chain]
  double eps[NT][NN];                                // eps of term (ch*2+chain)*(NK-1) + k-1 at the nodes
  int shift[NT];                                     // integer part I = ceil(D), fixed over the tile
  int generic;                                       // != 0: run the per-sample code for this tile
};

// A: chain delays at the nodes.  x0 = sample index of the tile's first sample, B = tile length.
// (The nodes of the first and last partly valid tiles can lie inside the margins, i.e. up to one tile outside the
// span lr_tdi checked against the knot table; spline_interval clamps the interval index there, which extrapolates the
// end cubic by at most 224 samples.  Only the polynomial fit over the tile sees those nodes: the valid samples of the
// tile lie inside the table, and the fit of a smooth cubic is exact wherever its nodes are.)
template <int GEN, int NN>
LR_HD void fir_chain_nodes(const Params& prm, FirTile<GEN, NN>& T, int n0, int B, int tid, int nthreads) {
  constexpr int NK = FirTile<GEN, NN>::NK;
  for (int w = tid; w < 6 * NN; w += nthreads) {
    const int cc = w / NN, node = w - cc * NN;       // cc = ch*2 + chain
    const int ch = cc >> 1, chain = cc & 1;
    const double xs = 0.5 * (double)(B - 1) * (1.0 + fir_node<NN>(node));  // position inside the tile [samples]
    const double trel = fma((double)n0 + xs, prm.dt, prm.trel0);
    double d = 0.0;
    T.dnode[cc][node][0] = 0.0;
#pragma unroll
    for (int k = 0; k + 1 < NK; ++k) {
      const int s = rot_slot_rt(chain == 0 ? chain_a(k) : chain_b(k), ch);
      d += spline_eval(prm, 9 + s, prm.chain_sum ? trel : trel - d);
      T.dnode[cc][node][k + 1] = d;
    }
  }
}

// B: integer shift and eps(node) per delayed term; decide whether the tile may use the FIR path.
template <int GEN, int NN>
LR_HD void fir_split_terms(const Params& prm, FirTile<GEN, NN>& T, int tid, int nthreads) {
  constexpr int NK = FirTile<GEN, NN>::NK;
  constexpr int NT = FirTile<GEN, NN>::NT;
  for (int term = tid; term < NT; term += nthreads) {
    const int cc = term / (NK - 1), k = term - cc * (NK - 1) + 1;
    double D[NN], lo = 1e300, hi = -1e300;
#pragma unroll
    for (int i = 0; i < NN; ++i) {
      D[i] = T.dnode[cc][i][k] * prm.inv_dt;
      lo = D[i] < lo ? D[i] : lo;
      hi = D[i] > hi ? D[i] : hi;
    }
    const double I = ceil(lo);
    const double spread = hi - lo;
    // every sample of the tile must see ceil(D) == I: the nodes include both ends of the tile, an interior
    // extremum can exceed the node range by less than `spread`
    const double guard = spread + 1e-12;
    const bool safe = (spread == 0.0) || ((I - hi) >= guard && (lo - (I - 1.0)) >= guard);
    T.shift[term] = (int)I;
#pragma unroll
    for (int i = 0; i < NN; ++i) T.eps[term][i] = I - D[i];
    if (!safe) T.generic = 1;   // benign race: every writer stores 1
  }
}

// The 2P-1 summation-by-parts coefficients of one interpolation: value = raw[a] - sum_j c[j+P-1] dif[a-1+j],
// j = 1-P..P-1, with c_j = C_j (j <= 0) and -E_j (j >= 1)   (cf. interp_sbp).
template <int PT>
LR_HD void sbp_coeffs(const Params& prm, double eps, double* c) {
  const int P = PT > 0 ? PT : prm.p;
  double R[PT > 0 ? PT : kPMax];
  const double z = fma(eps, eps, -eps);
  double pre = 1.0;
#pragma unroll
  for (int k = 1; k <= P; ++k) {
    R[k - 1] = pre * prm.bk[k];
    pre *= z - (double)(k * (k - 1));
  }
  double suf = 1.0, C = 0.0, E = 0.0;
#pragma unroll
  for (int k = P; k >= 1; --k) {
    const double Rk = R[k - 1] * suf;
    suf *= z - (double)(k * (k - 1));
    C = fma(Rk, (double)k - eps, C);
    c[(1 - k) + P - 1] = C;                       // j = 1-k
    if (k >= 2) {
      E = fma(Rk, eps + (double)(k - 1), E);
      c[(k - 1) + P - 1] = -E;                    // j = k-1
    }
  }
}

// C: coefficients of every delayed term at every node: cnode[term][node][2P-1]
template <int PT, int GEN, int NN>
LR_HD void fir_node_coeffs(const Params& prm, const FirTile<GEN, NN>& T, double* cnode, int tid, int nthreads) {
  constexpr int NT = FirTile<GEN, NN>::NT;
  const int P = PT > 0 ? PT : prm.p;
  const int L = 2 * P - 1;
  for (int w = tid; w < NT * NN; w += nthreads) {
    const int term = w / NN, node = w - term * NN;
    sbp_coeffs<PT>(prm, T.eps[term][node], cnode + (size_t)w * L);
  }
}

// D: merge.  K[((ch*4 + sl)*Wc + m)*kFirKStride + p] = coefficient of tau^p of dif_series[nl + m - back]
// where back = Wc - (P - 1) is the number of staged differences behind the sample.  m_rel = m - back.
template <int PT, int GEN, int NN>
LR_HD void fir_merge(const Params& prm, const FirTile<GEN, NN>& T, const double* cnode, double* K, int Wc,
                     int tid, int nthreads) {
  constexpr int NK = FirTile<GEN, NN>::NK;
  const int P = PT > 0 ? PT : prm.p;
  const int L = 2 * P - 1;
  const int back = Wc - (P - 1);
  for (int w = tid; w < 12 * Wc; w += nthreads) {
    const int cs = w / Wc, m = w - cs * Wc;       // cs = ch*4 + sl
    const int ch = cs >> 2, sl = cs & 3;
    const int m_rel = m - back;
    double v[NN];
#pragma unroll
    for (int i = 0; i < NN; ++i) v[i] = 0.0;
#pragma unroll
    for (int chain = 0; chain < 2; ++chain) {
      const double sign = chain == 0 ? 1.0 : -1.0;
#pragma unroll
      for (int k = 0; k < NK; ++k) {
        if ((chain == 0 ? fir_sl_a(k) : fir_sl_b(k)) != sl) continue;
        const int term = (ch * 2 + chain) * (NK - 1) + (k - 1);
        const int I = k == 0 ? 0 : T.shift[term];
        const int o = k == 0 ? 0 : 1 - I;         // anchor offset of the term: value = raw[nl+o] - S
        // anchors: term k of chain B and term k^2 of chain A carry the same series with opposite signs;
        // raw[nl+oA] - raw[nl+oB] = +/- the sum of the first differences between the two anchors
        double step = 0.0;
        if (chain == 1) {
          const int ka = k ^ 2;
          const int oa = ka == 0 ? 0 : 1 - T.shift[(ch * 2) * (NK - 1) + (ka - 1)];
          step = (m_rel >= o && m_rel < oa) ? 1.0 : (m_rel >= oa && m_rel < o) ? -1.0 : 0.0;
        }
        const int j = m_rel + I;                  // dif index nl - I + j
        const bool in = k > 0 && j >= 1 - P && j <= P - 1;
#pragma unroll
        for (int i = 0; i < NN; ++i) {
          double c = step;
          if (in) c -= sign * cnode[((size_t)term * NN + i) * L + (j + P - 1)];
          v[i] += c;
        }
      }
    }
    double* out = K + (size_t)w * kFirKStride;
    if (NN == 3) {          // nodes -1, 0, 1
      out[0] = v[1];
      out[1] = 0.5 * (v[2] - v[0]);
      out[2] = 0.5 * (v[0] + v[2]) - v[1];
      out[3] = 0.0;
    } else {                // nodes -1, -1/2, 1/2, 1
      const double s1 = 0.5 * (v[NN - 1] + v[0]), d1 = 0.5 * (v[NN - 1] - v[0]);
      const double s2 = 0.5 * (v[NN - 2] + v[1]), d2 = 0.5 * (v[NN - 2] - v[1]);
      const double a2 = (s1 - s2) * (4.0 / 3.0), a3 = (d1 - 2.0 * d2) * (4.0 / 3.0);
      out[0] = s2 - 0.25 * a2;
      out[1] = d1 - a3;
      out[2] = a2;
      out[3] = a3;
    }
  }
}

// E: apply.  One work item = kFirR consecutive samples of one channel.  dif: [6][W]; res: [3][B] (tile
// staging of X, Y, Z).  nl0 = staged index of the tile's first sample; Wc is a multiple of kFirR and the
// first `pad` taps of every series are zero padding.
// X(n) = sum_p tau_n^p A_p(n) with A_p(n) = sum_m K_p[m] dif[n + m]: NN accumulators per sample, NN FMAs per
// (tap, sample), the powers of tau applied once at the end.  Every FMA of the loop is (k_p, dif, A_p): k_p is
// common to the R samples of a tap and dif to the NN accumulators of a sample, so consecutive FMAs share a
// source register.  That matters on sm_100: a DFMA with three register operands none of which the previous
// instruction used issues every third cycle instead of every second (measured: 42 against 53-54 DFMA/clk/SM),
// which is what the Horner form (coefficient evaluated at tau_n first, then one FMA into one accumulator) ran at.
// NN = 1 (constant light times): k0 alone.
// ALIAS: `res` overlays `dif`; every thread then runs the loop body exactly once (nthreads == 3 * groups) and
// the block synchronises between the last read of dif and the first write of res.
template <int NN, bool ALIAS = false>
LR_HD void fir_apply(const double* dif, int W, const double* K, int Wc, int pad, int P, int nl0, int B, double* res,
                     int tid, int nthreads) {
  constexpr int R = kFirR;
  const int groups = (B + R - 1) / R;
  const int back = Wc - (P - 1);
  const double half = 0.5 * (double)(B - 1), inv_half = 1.0 / half;
  for (int w = tid; w < 3 * groups; w += nthreads) {
    const int ch = w / groups, g = w - ch * groups;
    const int i0 = g * R;                                  // first sample of the group inside the tile
    const int slots = ch == 0 ? fir_slot_word(0) : ch == 1 ? fir_slot_word(1) : fir_slot_word(2);
    double acc[NN][R];
#pragma unroll
    for (int p = 0; p < NN; ++p)
#pragma unroll
      for (int r = 0; r < R; ++r) acc[p][r] = 0.0;
#pragma unroll 1
    for (int sl = 0; sl < 4; ++sl) {
      const double* d = dif + ((slots >> (3 * sl)) & 7) * W + (nl0 + i0 - back);
      int koff = (ch * 4 + sl) * Wc * kFirKStride;
#ifdef __CUDA_ARCH__
      asm volatile("" : "+r"(koff));   // keep the tap offset in a register (ptxas otherwise rebuilds it per tap)
#endif
      const double* kk = K + koff;
      // circular window: tap t = m0 + mm needs d[t .. t+R), kept at positions (t + r) % R; after the tap the
      // slot of d[t] takes d[t + R] (indices are compile-time constants: m0 is a multiple of R)
      double win[R];
#pragma unroll
      for (int r = 0; r < R; ++r) win[r] = d[r];
#pragma unroll 1
      for (int m0 = 0; m0 < Wc; m0 += R) {
        const int skip = m0 == 0 ? pad : 0;   // the first `pad` stored taps are padding (all zero)
#pragma unroll
        for (int mm = 0; mm < R; ++mm) {
          if (mm >= skip) {
            double kc[NN];
#pragma unroll
            for (int p = 0; p < NN; ++p) kc[p] = kk[(m0 + mm) * kFirKStride + p];
#pragma unroll
            for (int p = 0; p < NN; ++p)
#pragma unroll
              for (int r = 0; r < R; ++r) acc[p][r] = fma(kc[p], win[(mm + r) % R], acc[p][r]);
          }
          win[mm] = d[m0 + mm + R];
        }
      }
    }
#pragma unroll
    for (int r = 0; r < R; ++r) {
      const double tau = ((double)(i0 + r) - half) * inv_half;
#pragma unroll
      for (int p = NN - 2; p >= 0; --p) acc[p][r] = fma(acc[p + 1][r], tau, acc[p][r]);
    }
#ifdef __CUDA_ARCH__
    if (ALIAS) __syncthreads();
#endif
#pragma unroll
    for (int r = 0; r < R; ++r)
      if (i0 + r < B) res[ch * B + i0 + r] = acc[0][r];
  }
}

constexpr int kFirGroups = 32;                    // groups of kFirR samples per channel and tile
constexpr int kFirTile = kFirGroups * kFirR;      // 224 samples per tile
constexpr int kFirThreads = 3 * kFirGroups;       // apply kernel: one warp per channel
constexpr int kFirSetupThreads = 128;

// The plan of one tile in global memory: K[12][Wc][kFirKStride] doubles; flags[tile] != 0 marks a tile that
// must run the exact per-sample code.  The plan depends on the orbits and the time grid only (not on y), so
// one plan serves every template of a batch and every later lr_tdi call on the same grid.
LR_HD size_t fir_plan_doubles_per_tile(int Wc) { return (size_t)12 * Wc * kFirKStride; }

#ifdef __CUDACC__
// ------------------------------------------------------------------------------------------ plan kernel
// grid.x = ntiles; dynamic smem: FirTile + cnode[NT][NN][2P-1]
template <int PT, int GEN, int NN>
__global__ void __launch_bounds__(kFirSetupThreads)
tdi_fir_setup_kernel(const Params prm, double* __restrict__ plan, int* __restrict__ flags,
                     int* __restrict__ list /* [0] = count, [1..] = flagged tiles */) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  constexpr int B = kFirTile;
  FirTile<GEN, NN>& T = *reinterpret_cast<FirTile<GEN, NN>*>(smem_raw);
  double* cnode = reinterpret_cast<double*>(smem_raw + ((sizeof(FirTile<GEN, NN>) + 15) / 16) * 16);
  const int tid = threadIdx.x;
  const int slot = blockIdx.x;                      // plan slot; = the global tile unless the plan is uniform
  const int tile = prm.fir_tile0 + slot;
  const int n0 = tile * B;
  const int Wc = prm.fir_wc;
  // (the plan is always built for the whole series: prm.n_off = 0, tiles are global)
  if (n0 + B <= prm.m_front || n0 >= prm.n_glob - prm.m_back) {   // tile entirely inside a margin: never applied
    if (tid == 0) flags[slot] = 0;
    return;
  }
  if (tid == 0) T.generic = 0;
  fir_chain_nodes<GEN, NN>(prm, T, n0, B, tid, kFirSetupThreads);
  __syncthreads();
  fir_split_terms<GEN, NN>(prm, T, tid, kFirSetupThreads);
  __syncthreads();
  if (tid == 0) {
    flags[slot] = T.generic;
    if (T.generic) list[1 + atomicAdd(list, 1)] = tile;
  }
  if (T.generic) return;
  fir_node_coeffs<PT, GEN, NN>(prm, T, cnode, tid, kFirSetupThreads);
  __syncthreads();
  fir_merge<PT, GEN, NN>(prm, T, cnode, plan + (size_t)slot * fir_plan_doubles_per_tile(Wc), Wc, tid,
                         kFirSetupThreads);
}

// ----------------------------------------------------------------------------------------- apply kernel
// grid.x = ntiles * batch, template index fastest (the tiles of one time span share their plan through L2).
// Tiles flagged by the plan are left to tdi_fir_fixup_kernel.
// dynamic smem: dif[6][W] | K[12][Wc][4]; the results res[3][B] overlay dif once every read of it is done
LR_HD size_t fir_apply_smem_bytes(int W, int Wc) {
  return ((size_t)6 * W + fir_plan_doubles_per_tile(Wc)) * sizeof(double);
}

// eq. 21 and the coalesced store of one sample (shared by the apply and fix-up kernels)
__device__ __forceinline__ void fir_store(double* ob, int64_t N, int n, int channels, double X, double Y, double Z) {
  if (channels != 1) { ob[n] = X; ob[N + n] = Y; ob[2 * N + n] = Z; }
  if (channels != 0) {
    double* oa = channels == 2 ? ob + 3 * N : ob;
    oa[n] = (Z - X) * 0.70710678118654752440;
    oa[N + n] = (X - 2.0 * Y + Z) * 0.40824829046386301637;
    oa[2 * N + n] = (X + Y + Z) * 0.57735026918962576451;
  }
}

template <int NN>
__global__ void __launch_bounds__(kFirThreads, kFirMinBlocks)
tdi_fir_apply_kernel(const Params prm, const double* __restrict__ y, double* __restrict__ out, int channels,
                     const double* __restrict__ plan, const int* __restrict__ flags, int batch) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  constexpr int B = kFirTile;
  const int W = B + prm.halo_lo + prm.halo_hi;
  const int Wc = prm.fir_wc;
  double* dif = reinterpret_cast<double*>(smem_raw);
  double* K = dif + 6 * W;
  double* res = dif;
  static_assert(kFirThreads == 3 * kFirGroups && kFirGroups * kFirR == kFirTile, "one work item per thread");

  const int tid = threadIdx.x;
  const int tile = blockIdx.x / batch;                       // local tile: local samples [n0, n0 + B)
  const int64_t b = blockIdx.x - (int64_t)tile * batch;
  const int n0 = tile * B;
  const int g0 = n0 - prm.halo_lo;
  const int tile_g = tile + prm.n_off / B;                   // global tile (prm.n_off is a multiple of B)
  const int n0g = prm.n_off + n0;
  const int64_t N = prm.out_stride;
  const int nout = channels == 2 ? 6 : 3;
  double* ob = out + b * nout * N;

  const int v_lo = prm.m_front, v_hi = prm.n_glob - prm.m_back;   // valid global samples [v_lo, v_hi)
  if (n0g + B <= v_lo || n0g >= v_hi) {                      // tile entirely inside a margin
    for (int i = tid; i < B; i += kFirThreads)
      if (n0 + i < prm.n)
        for (int c = 0; c < nout; ++c) ob[(int64_t)c * N + n0 + i] = 0.0;
    return;
  }
  const int slot = prm.fir_uniform ? 0 : tile_g;             // constant light times: one plan for every tile
  if (flags[slot] != 0) return;                              // exact per-sample tile: the fix-up kernel's

  // the tile's plan: global -> shared without passing through registers, in flight under the loads of y
  {
    const double2* src = reinterpret_cast<const double2*>(plan + (size_t)slot * fir_plan_doubles_per_tile(Wc));
    const unsigned dst = (unsigned)__cvta_generic_to_shared(K);
    const int cnt = (int)(fir_plan_doubles_per_tile(Wc) / 2);
    for (int m = tid; m < cnt; m += kFirThreads)
      asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst + 16u * m), "l"(src + m) : "memory");
    asm volatile("cp.async.commit_group;" ::: "memory");
  }
  // first differences straight from global memory (the second load of each pair hits L1).  Instructions
  // count here: an FP64 instruction holds its scheduler's issue port for two cycles, so every other
  // instruction of the kernel takes time from the filter loop of the co-resident CTAs.
  {
    const double* yb = y + b * 6 * prm.in_stride + g0;
    if (g0 >= prm.rd_lo && g0 + W < prm.rd_hi) {             // (block-uniform) the whole window is readable
#pragma unroll
      for (int sr = 0; sr < 6; ++sr) {
        const double* ys = yb + sr * prm.in_stride;
        double* ds = dif + sr * W;
#pragma unroll 3
        for (int w = tid; w < W; w += kFirThreads) ds[w] = __ldg(ys + w + 1) - __ldg(ys + w);
      }
    } else {
      for (int sr = 0; sr < 6; ++sr) {
        const double* ys = yb + sr * prm.in_stride;
        for (int w = tid; w < W; w += kFirThreads) {
          const int g = g0 + w;
          const double a = (g >= prm.rd_lo && g < prm.rd_hi) ? __ldg(ys + w) : 0.0;
          const double c = (g + 1 >= prm.rd_lo && g + 1 < prm.rd_hi) ? __ldg(ys + w + 1) : 0.0;
          dif[sr * W + w] = c - a;
        }
      }
    }
  }
  asm volatile("cp.async.wait_group 0;" ::: "memory");
  __syncthreads();
  fir_apply<NN, true>(dif, W, K, Wc, Wc - prm.fir_taps, prm.p, prm.halo_lo, B, res, tid, kFirThreads);
  __syncthreads();
  if (n0 + B <= prm.n && n0g >= v_lo && n0g + B <= v_hi) {   // (block-uniform) a full tile of valid samples
    for (int i = tid; i < B; i += kFirThreads) fir_store(ob, N, n0 + i, channels, res[i], res[B + i], res[2 * B + i]);
    return;
  }
  for (int i = tid; i < B; i += kFirThreads) {
    const int n = n0 + i;
    if (n >= prm.n) break;
    const bool valid = n0g + i >= v_lo && n0g + i < v_hi;
    fir_store(ob, N, n, channels, valid ? res[i] : 0.0, valid ? res[B + i] : 0.0, valid ? res[2 * B + i] : 0.0);
  }
}

// ------------------------------------------------------------------------- apply kernel, cubic plans (NN = 4)
// The same filter through the FP64 tensor path (mma.sync.m8n8k4.f64).  A DFMA of the loop above reads two fresh
// 64-bit register operands and cannot issue every second cycle (43 per SM and clock at NN = 4); an MMA reads four
// operand registers per eight FMAs per thread and runs at the pipe's rate.  With four powers of tile time the tensor
// tile is full: every y series feeds exactly two of the three channels, so for series s
//   D[8 samples][8 columns] += A[8 samples][4 taps] * B[4 taps][8 columns],
//   A[i][k] = dif_s[n0 + i + m0 + k],  B[k][(half, p)] = K_p[channel of that half][s][m0 + k],
// columns = (left channel: p = 0..3 | right channel: p = 0..3).  Three accumulator tiles per 8 samples:
//   XY (series 12, 21: X | Y),  ZY (series 23, 32: Z | Y),  XZ (series 31, 13: X | Z),
// and X = XY.left + XZ.left, Y = XY.right + ZY.right, Z = ZY.left + XZ.right; the powers of tile time are applied to
// the sums at the end (as in fir_apply).  (With three powers the tile would be 6/8 full: no faster than the DFMA loop;
// the quadratic plans keep it.)
// One CTA = one plan tile of 224 samples = 4 warps x 7 row tiles of 8 samples.  A is a Hankel block (it depends on
// i + k only), so the A fragment of row tile j at tap step q is the fragment of row tile j+1 at step q-2: two sliding
// windows of 7 fragments (even and odd steps), one new LDS.64 per step.  dynamic smem: dif[6][W] | K[12][Wc][4] |
// raw[6][W + 1] (the y window as it arrives by cp.async); the staged sums res[3][4][224] overlay dif and K once the
// MMAs are done.
constexpr int kFirMmaThreads = 128;
LR_HD size_t fir_mma_smem_bytes(int W, int Wc) {
  const size_t a = fir_apply_smem_bytes(W, Wc) + (size_t)6 * ((W + 2) & ~1) * sizeof(double);   // dif | K | raw
  const size_t b = (size_t)12 * kFirTile * sizeof(double);
  return a > b ? a : b;
}

#ifdef __CUDACC__
__device__ __forceinline__ void dmma_8x8x4(double& d0, double& d1, double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
               : "+d"(d0), "+d"(d1) : "d"(a), "d"(b));
}

template <int NN>
__global__ void __launch_bounds__(kFirMmaThreads, 3)
tdi_fir_apply_mma_kernel(const Params prm, const double* __restrict__ y, double* __restrict__ out, int channels,
                         const double* __restrict__ plan, const int* __restrict__ flags, int batch) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  constexpr int B = kFirTile, RT = 7;                        // row tiles (of 8 samples) per warp
  static_assert(NN == 4 && NN == kFirKStride, "the MMA tile holds two channels x four powers");
  static_assert(kFirMmaThreads / 32 * RT * 8 == kFirTile, "4 warps x 7 row tiles x 8 samples");
  const int W = B + prm.halo_lo + prm.halo_hi;
  const int Wc = prm.fir_wc;
  const int Wr = (W + 2) & ~1;                               // staged y samples per series (W differences need W + 1)
  double* dif = reinterpret_cast<double*>(smem_raw);
  double* K = dif + 6 * W;
  double* raw = K + fir_plan_doubles_per_tile(Wc);           // [6][Wr]
  double* res = dif;                                         // [3 channels][4 powers][B], after the MMAs

  const int tid = threadIdx.x;
  const int tile = blockIdx.x / batch;                       // local tile: local samples [n0, n0 + B)
  const int64_t b = blockIdx.x - (int64_t)tile * batch;
  const int n0 = tile * B;
  const int g0 = n0 - prm.halo_lo;
  const int tile_g = tile + prm.n_off / B;                   // global tile (prm.n_off is a multiple of B)
  const int n0g = prm.n_off + n0;
  const int64_t N = prm.out_stride;
  const int nout = channels == 2 ? 6 : 3;
  double* ob = out + b * nout * N;

  const int v_lo = prm.m_front, v_hi = prm.n_glob - prm.m_back;   // valid global samples [v_lo, v_hi)
  if (n0g + B <= v_lo || n0g >= v_hi) {                      // tile entirely inside a margin
    for (int i = tid; i < B; i += kFirMmaThreads)
      if (n0 + i < prm.n)
        for (int c = 0; c < nout; ++c) ob[(int64_t)c * N + n0 + i] = 0.0;
    return;
  }
  if (flags[tile_g] != 0) return;                            // exact per-sample tile: the fix-up kernel's

  {   // the tile's plan: global -> shared without passing through registers, in flight under the loads of y
    const double2* src = reinterpret_cast<const double2*>(plan + (size_t)tile_g * fir_plan_doubles_per_tile(Wc));
    const unsigned dst = (unsigned)__cvta_generic_to_shared(K);
    const int cnt = (int)(fir_plan_doubles_per_tile(Wc) / 2);
    for (int m = tid; m < cnt; m += kFirMmaThreads)
      asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst + 16u * m), "l"(src + m) : "memory");
    asm volatile("cp.async.commit_group;" ::: "memory");
  }
  {   // the y window of the six series: asynchronous 8-byte copies (the rows of y need not be 16-byte aligned), all in
      // flight at once; with 12 warps per SM a staging phase of six dependent global loads would not be hidden
    const double* yb = y + b * 6 * prm.in_stride + g0;
    if (g0 >= prm.rd_lo && g0 + W < prm.rd_hi) {             // (block-uniform) the whole window is readable
      const unsigned dst = (unsigned)__cvta_generic_to_shared(raw);
#pragma unroll
      for (int sr = 0; sr < 6; ++sr) {
        const double* ys = yb + sr * prm.in_stride;
        for (int w = tid; w <= W; w += kFirMmaThreads)
          asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(dst + 8u * (unsigned)(sr * Wr + w)), "l"(ys + w)
                       : "memory");
      }
    } else {
      for (int sr = 0; sr < 6; ++sr) {
        const double* ys = yb + sr * prm.in_stride;
        for (int w = tid; w <= W; w += kFirMmaThreads) {
          const int g = g0 + w;
          raw[sr * Wr + w] = (g >= prm.rd_lo && g < prm.rd_hi) ? __ldg(ys + w) : 0.0;
        }
      }
    }
    asm volatile("cp.async.commit_group;" ::: "memory");
  }
  asm volatile("cp.async.wait_group 0;" ::: "memory");
  __syncthreads();
  for (int m = tid; m < 6 * W; m += kFirMmaThreads) {        // exact first differences, as the one-shot kernel forms them
    const int sr = m / W, w = m - sr * W;
    dif[m] = raw[sr * Wr + w + 1] - raw[sr * Wr + w];
  }
  __syncthreads();

  const int warp = tid >> 5, lane = tid & 31;
  const int row = lane >> 2, kq = lane & 3;                  // A: [row][kq]; B: [kq][column = row]; D: [row][2 kq, 2 kq + 1]
  const int half = row >> 2, pw = row & 3;                   // B column -> (left | right channel, power)
  const int back = Wc - (prm.p - 1);
  const int Q = (Wc + 3) >> 2;                               // tap steps of 4 (coefficients beyond Wc count as 0)
  const int abase = prm.halo_lo + warp * (RT * 8) - back + row + kq;   // A fragment u: dif[abase + 4 u]
  // accumulator tiles: (series slots, (channel, local series) of the left and of the right half), see above and
  // fir_base_slot: X = {13, 31, 12, 21}, Y = {21, 12, 23, 32}, Z = {32, 23, 31, 13} in local order
  double acc[3][RT][2];
#pragma unroll
  for (int t = 0; t < 3; ++t)
#pragma unroll
    for (int j = 0; j < RT; ++j) { acc[t][j][0] = 0.0; acc[t][j][1] = 0.0; }
#pragma unroll
  for (int t = 0; t < 3; ++t) {
#pragma unroll
    for (int e = 0; e < 2; ++e) {
      // XY: slot 0 = (X,2)|(Y,1), slot 5 = (X,3)|(Y,0);  ZY: slot 1 = (Z,1)|(Y,2), slot 4 = (Z,0)|(Y,3);
      // XZ: slot 2 = (X,1)|(Z,2), slot 3 = (X,0)|(Z,3)
      const int slot = t == 0 ? (e == 0 ? 0 : 5) : t == 1 ? (e == 0 ? 1 : 4) : (e == 0 ? 2 : 3);
      const int csl = t == 0 ? (e == 0 ? 0 * 4 + 2 : 0 * 4 + 3) : t == 1 ? (e == 0 ? 2 * 4 + 1 : 2 * 4 + 0)
                                                                       : (e == 0 ? 0 * 4 + 1 : 0 * 4 + 0);
      const int csr = t == 0 ? (e == 0 ? 1 * 4 + 1 : 1 * 4 + 0) : t == 1 ? (e == 0 ? 1 * 4 + 2 : 1 * 4 + 3)
                                                                       : (e == 0 ? 2 * 4 + 2 : 2 * 4 + 3);
      const double* a = dif + slot * W + abase;
      const double* kb = K + ((size_t)(half ? csr : csl) * Wc + kq) * kFirKStride + pw;   // + 4 q taps
      // A fragments of the even / odd steps as circular windows: at step q = q0 + s (q0 a multiple of 2 RT) row tile j
      // needs fragment u = q + 2 j, kept at position (j + s / 2) % RT; after the step the position of row tile 0
      // takes fragment u = q + 2 RT.  All positions are compile-time constants (no register moves).
      double we[RT], wo[RT];
#pragma unroll
      for (int j = 0; j < RT; ++j) { we[j] = a[4 * (2 * j)]; wo[j] = a[4 * (2 * j + 1)]; }
#pragma unroll 1
      for (int q0 = 0; q0 < Q; q0 += 2 * RT) {
#pragma unroll
        for (int sp = 0; sp < 2 * RT; ++sp) {
          const int q = q0 + sp;
          if (q < Q) {                                         // (warp-uniform)
            const double bf = 4 * q + kq < Wc ? kb[(size_t)4 * q * kFirKStride] : 0.0;
            if (sp % 2 == 0) {
#pragma unroll
              for (int j = 0; j < RT; ++j) dmma_8x8x4(acc[t][j][0], acc[t][j][1], we[(j + sp / 2) % RT], bf);
              we[(sp / 2) % RT] = a[4 * (q + 2 * RT)];
            } else {
#pragma unroll
              for (int j = 0; j < RT; ++j) dmma_8x8x4(acc[t][j][0], acc[t][j][1], wo[(j + sp / 2) % RT], bf);
              wo[(sp / 2) % RT] = a[4 * (q + 2 * RT)];
            }
          }
        }
      }
    }
  }
  __syncthreads();                                           // every warp is done with dif and K: res may overlay them
  // lanes with kq < 2 hold left halves (powers 2 kq, 2 kq + 1), the others right halves (powers 2 (kq - 2), ...):
  //   kq < 2 : X = XY + XZ complete, Z (ZY.left) partial;  kq >= 2 : Y = XY + ZY complete, Z (XZ.right) partial
#pragma unroll
  for (int j = 0; j < RT; ++j) {
    const int i = warp * (RT * 8) + j * 8 + row;
    const int p0 = 2 * (kq & 1);
    const bool left = kq < 2;
#pragma unroll
    for (int c = 0; c < 2; ++c) {
      const double mine = left ? acc[0][j][c] + acc[2][j][c] : acc[0][j][c] + acc[1][j][c];   // X | Y
      const double zpart = left ? acc[1][j][c] : acc[2][j][c];
      const double z = zpart + __shfl_xor_sync(0xffffffffu, zpart, 2);
      res[((left ? 0 : 1) * 4 + p0 + c) * B + i] = mine;
      if (left) res[(2 * 4 + p0 + c) * B + i] = z;
    }
  }
  __syncthreads();
  const double hf = 0.5 * (double)(B - 1), inv_hf = 1.0 / hf;
  const bool full = n0 + B <= prm.n && n0g >= v_lo && n0g + B <= v_hi;   // (block-uniform) a full tile of valid samples
  for (int i = tid; i < B; i += kFirMmaThreads) {
    const int n = n0 + i;
    if (!full && n >= prm.n) break;
    const double tau = ((double)i - hf) * inv_hf;
    double v[3];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      const double* r = res + (size_t)c * 4 * B + i;
      v[c] = fma(fma(fma(r[3 * B], tau, r[2 * B]), tau, r[B]), tau, r[0]);
    }
    const bool valid = full || (n0g + i >= v_lo && n0g + i < v_hi);
    fir_store(ob, N, n, channels, valid ? v[0] : 0.0, valid ? v[1] : 0.0, valid ? v[2] : 0.0);
  }
}
#endif

// ---------------------------------------------------------------------------------------- fix-up kernel
// The tiles the plan flagged (a delay crosses a whole number of samples inside them) with the exact
// per-sample weights of tdi_sample.  Fixed grid; work item = (flagged tile, template).
// dynamic smem: raw[6][W], dif[6][W]
template <int PT, int GEN>
__global__ void __launch_bounds__(kFirTile)
tdi_fir_fixup_kernel(const Params prm, const double* __restrict__ y, double* __restrict__ out, int channels,
                     const int* __restrict__ list, int batch) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  constexpr int B = kFirTile;
  const int W = B + prm.halo_lo + prm.halo_hi;
  double* raw = reinterpret_cast<double*>(smem_raw);
  double* dif = raw + 6 * W;
  const int tid = threadIdx.x;
  const int64_t N = prm.out_stride;
  const int nout = channels == 2 ? 6 : 3;
  const int v_lo = prm.m_front, v_hi = prm.n_glob - prm.m_back;
  const int tile_lo = prm.n_off / B, ntl = (prm.n + B - 1) / B;   // this launch covers global tiles [tile_lo, tile_lo + ntl)
  const int64_t items = (int64_t)list[0] * batch;
  for (int64_t w = blockIdx.x; w < items; w += gridDim.x) {
    const int tile = list[1 + (int)(w / batch)] - tile_lo;      // local tile
    if (tile < 0 || tile >= ntl) continue;                      // (block-uniform)
    const int64_t b = w % batch;
    const int n0 = tile * B, g0 = n0 - prm.halo_lo;
    const double* yb = y + b * 6 * prm.in_stride;
    __syncthreads();
    for (int m = tid; m < 6 * W; m += B) {
      const int s = m / W, g = g0 + (m - s * W);
      raw[m] = (g >= prm.rd_lo && g < prm.rd_hi) ? __ldg(yb + s * prm.in_stride + g) : 0.0;
    }
    __syncthreads();
    for (int m = tid; m < 6 * W; m += B) {
      const int ww = m % W;
      dif[m] = (ww < W - 1) ? raw[m + 1] - raw[m] : 0.0;
    }
    __syncthreads();
    const int n = n0 + tid, ng = prm.n_off + n;
    if (n < prm.n) {
      double xyz[3] = {0.0, 0.0, 0.0};
      if (ng >= v_lo && ng < v_hi) tdi_sample<PT, GEN>(prm, raw, dif, W, prm.halo_lo + tid, sample_trel(prm, ng), xyz);
      fir_store(out + b * nout * N, N, n, channels, xyz[0], xyz[1], xyz[2]);
    }
  }
}
#endif

}  // namespace lr
