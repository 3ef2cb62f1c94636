// bz_quad.cuh -- 4 lanes per zone ("quad") burn kernel pieces, DESIGN.md section 5.4.
//
// Why 4 lanes: a zone's integrator state is ~3 KB (n = 14: P/LU 196, Z 84, vectors ~60 doubles),
// so only ~100-130 zones fit on an SM.  One thread per zone then means 3-4 warps per SM and every
// instruction latency is exposed (measured: 1.6 % of FP64 peak).  Splitting a zone over 4 lanes
// gives 12-16 resident warps with the same state, 4 independent slots of work per lane, and short
// dependent chains -- at the price of a few shuffles and some redundant scalar arithmetic.
//
// Mapping: component i of every n-vector lives on lane c = i % 4 of the quad, slot s = i / 4;
// ROW i of the Newton matrix P lives in the same place (a[s][0..n-1], registers, static indices).
// The Nordsieck array, weights and the saved vector live in shared memory per zone.
// LU (a5): the unknowns are ordered temperature-first, so partial pivoting
// keeps the natural order almost always: step k's pivot row is the static (lane k%4, slot k/4);
// it is published through shared memory, every lane computes its own multipliers, updates its own
// rows and keeps the largest |multiplier|: below 1 it proves that dgefa would not have swapped
// (QuadLU::factor).  A zone that may need an interchange redoes the factorisation on the general
// path (lane 0 of the quad, LINPACK dgefa on a global-memory scratch copy), bit-identical to the
// oracle either way.
#pragma once
#include <cstdint>
#include "bz_coop.cuh"      // constants, BurnArgs, eta_of, factorial_, inv_small_int
#include "bz_coop_burn.cuh" // nord_predict / nord_retract / nord_rescale / build_d / sel

namespace bz {

struct QuadNet {
  const double *coef;  // device: lnA[K] n[K] B[K] Q[K] aion[N]
  double fac;
  double *gscratch;    // device: per-quad general-path scratch, NEQ*NEQ + NEQ doubles + NEQ ints each
};

// per-zone shared memory (doubles); size padded so that consecutive zones start 4 doubles apart
// modulo 32 (8 zones x 4 lanes x 8 B of a warp access then cover all banks exactly twice)
template <int NEQ, int K>
struct QuadMem {
  static constexpr int Z_OFF = 0;                       // Z[6][NEQ]
  static constexpr int W_OFF = Z_OFF + (QMAX + 1) * NEQ; // w[NEQ]
  static constexpr int S_OFF = W_OFF + NEQ;             // saved vector S[NEQ]
  static constexpr int Y_OFF = S_OFF + NEQ;             // y / f gather [NEQ]
  static constexpr int U_OFF = Y_OFF + NEQ;             // pivot row broadcast, 2 x (NEQ + 1)
  static constexpr int L_OFF = U_OFF + 2 * (NEQ + 1);   // lambda_k [K]
  static constexpr int SC_OFF = L_OFF + K;               // per-zone scalars: l[7] hs[6] rxi[6] tau[6]
  static constexpr int SC_L = 0, SC_HS = 7, SC_RXI = 13, SC_TAU = 19;
  // rarely used per-zone scalars, parked here instead of in registers (every lane of the quad
  // stores the same bits and reads them back: no intra-quad synchronisation needed)
  static constexpr int SC_T = 26, SC_ETAMAX = 27, SC_HSAV = 28, SC_ZID = 29, SC_INT = 30;
  // Newton-matrix reuse (bz_set_policy 1): gamma_P of the kept factorisation; two ints: flags (bit 0 a
  // factorisation exists, bit 1 a failure asked for a fresh one, bit 2 it lives on the general path)
  // and nst at the factorisation
  static constexpr int SC_GAMP = 31, SC_PINT = 32, SC_N = 33;
  static constexpr int CNT_OFF = SC_OFF + SC_N;         // event counters of this quad: 8 x uint64 (lane 0 only)
  static constexpr int CN_NST = 0, CN_XRHS = 1, CN_INIT = 2, CN_LU = 3, CN_SOL = 4, CN_ETF = 5, CN_CFN = 6, CN_FAIL = 7;
  static constexpr int SRC_OFF = CNT_OFF + 8;           // constant source terms s[NEQ] (burn_zones_src)
  static constexpr int RAW = SRC_OFF + NEQ;
  static constexpr int SIZE = RAW + ((4 - (RAW % 32) + 32) % 32);  // == 4 (mod 32)
  double *base;
  __device__ __forceinline__ double &Z(int j, int i) const { return base[Z_OFF + j * NEQ + i]; }
  __device__ __forceinline__ double &W(int i) const { return base[W_OFF + i]; }
  __device__ __forceinline__ double &Sv(int i) const { return base[S_OFF + i]; }
  __device__ __forceinline__ double *ysh() const { return base + Y_OFF; }
  __device__ __forceinline__ double *ub(int par) const { return base + U_OFF + par * (NEQ + 1); }  // row + its b
  __device__ __forceinline__ double *lam() const { return base + L_OFF; }
  __device__ __forceinline__ double &sc(int i) const { return base[SC_OFF + i]; }
  __device__ __forceinline__ long long &zid() const { return *reinterpret_cast<long long *>(base + SC_OFF + SC_ZID); }
  __device__ __forceinline__ int &isc(int i) const { return reinterpret_cast<int *>(base + SC_OFF + SC_INT)[i]; }  // 0: qS, 1: ntau
  __device__ __forceinline__ int &pint(int i) const { return reinterpret_cast<int *>(base + SC_OFF + SC_PINT)[i]; }  // 0: flags, 1: nslp
  __device__ __forceinline__ double &src(int i) const { return base[SRC_OFF + i]; }
  __device__ __forceinline__ unsigned long long &cnt(int i) const { return reinterpret_cast<unsigned long long *>(base + CNT_OFF)[i]; }
};

// Pascal-triangle predict / retract of one component for a compile-time order Q: no predication,
// exactly Q+1 loads and stores (the run-time-order versions cost a select per addition).
template <int Q, bool RETRACT, class Mem>
__device__ __forceinline__ double nord_shift_q(const Mem &m, int i) {
  double zc[Q + 1];
#pragma unroll
  for (int j = 0; j <= Q; j++) zc[j] = m.Z(j, i);
#pragma unroll
  for (int k = 1; k <= Q; k++)
#pragma unroll
    for (int j = Q; j >= k; j--) zc[j - 1] = RETRACT ? zc[j - 1] - zc[j] : zc[j - 1] + zc[j];
#pragma unroll
  for (int j = 0; j < Q; j++) m.Z(j, i) = zc[j];  // Z[Q] is unchanged
  return zc[0];
}
template <bool RETRACT, class Mem>
__device__ __forceinline__ double nord_shift(const Mem &m, int i, int q) {
  switch (q) {
    case 1: return nord_shift_q<1, RETRACT>(m, i);
    case 2: return nord_shift_q<2, RETRACT>(m, i);
    case 3: return nord_shift_q<3, RETRACT>(m, i);
    case 4: return nord_shift_q<4, RETRACT>(m, i);
    default: return nord_shift_q<5, RETRACT>(m, i);
  }
}

// One component's column of the Nordsieck array (z[j * STRIDE], j = 0..Q): retract the prediction
// (same loop order as the predictor, C.2-B.7) and rescale by eta^j, for a compile-time order.
template <int Q, int STRIDE>
__device__ __forceinline__ void nord_retract_rescale_q(double *z, double eta) {
  double zc[Q + 1];
#pragma unroll
  for (int j = 0; j <= Q; j++) zc[j] = z[j * STRIDE];
#pragma unroll
  for (int k = 1; k <= Q; k++)
#pragma unroll
    for (int j = Q; j >= k; j--) zc[j - 1] = zc[j - 1] - zc[j];
  double r = eta;
#pragma unroll
  for (int j = 1; j <= Q; j++) {
    zc[j] = zc[j] * r;
    r = r * eta;
  }
#pragma unroll
  for (int j = 0; j <= Q; j++) z[j * STRIDE] = zc[j];
}
template <int STRIDE>
__device__ __forceinline__ void nord_retract_rescale(double *z, int q, double eta) {
  switch (q) {
    case 1: nord_retract_rescale_q<1, STRIDE>(z, eta); break;
    case 2: nord_retract_rescale_q<2, STRIDE>(z, eta); break;
    case 3: nord_retract_rescale_q<3, STRIDE>(z, eta); break;
    case 4: nord_retract_rescale_q<4, STRIDE>(z, eta); break;
    default: nord_retract_rescale_q<5, STRIDE>(z, eta); break;
  }
}

// Z_j *= eta^j, j = 1..Q, powers by repeated multiplication (nord_rescale)
template <int Q, int STRIDE>
__device__ __forceinline__ void nord_rescale_only_q(double *z, double eta) {
  double r = eta;
#pragma unroll
  for (int j = 1; j <= Q; j++) {
    z[j * STRIDE] = z[j * STRIDE] * r;
    r = r * eta;
  }
}
template <int STRIDE>
__device__ __forceinline__ void nord_rescale_only(double *z, int q, double eta) {
  switch (q) {
    case 1: nord_rescale_only_q<1, STRIDE>(z, eta); break;
    case 2: nord_rescale_only_q<2, STRIDE>(z, eta); break;
    case 3: nord_rescale_only_q<3, STRIDE>(z, eta); break;
    case 4: nord_rescale_only_q<4, STRIDE>(z, eta); break;
    default: nord_rescale_only_q<5, STRIDE>(z, eta); break;
  }
}

template <int NEQ>
struct QuadLU {
  static constexpr int S = (NEQ + 3) / 4;
  double a[S][NEQ];  // my rows of P, then of its LU factors: l_ik below the diagonal, U above it,
                     // 1/pivot ON the diagonal (LINPACK keeps the pivot; only its reciprocal is used)

  __device__ __forceinline__ static unsigned hi_abs(double x) {
    return (unsigned)(__double_as_longlong(x) >> 32) & 0x7fffffffu;
  }

  // no-interchange factorisation.  returns bit 0: an interchange may be needed (results invalid,
  // redo on the general path), bit 1: zero / NaN pivot.  Quad-uniform result.
  // Interchange test: LINPACK swaps iff some |a_ik| > |a_kk| below the diagonal.  Then
  // |a_ik| >= |a_kk| (1 + 2^-52), and with inv = RN(1/a_kk) = (1 + e)/a_kk, |e| <= 2^-53, the exact
  // product |a_ik * inv| >= (1 + 2^-52)(1 - 2^-53) > 1, so the computed multiplier
  // l = RN(a_ik * inv) has |l| >= 1 (rounding is monotone).  Hence |l| < 1 -- high word below
  // 0x3FF00000, one AND and one unsigned max per multiplier -- PROVES that dgefa would not swap.
  // |l| >= 1 without a swap needs |a_ik| within one ulp of |a_kk| (exact ties included); those and
  // NaN multipliers take the general path, which pivots exactly.  (A bound of 1 - 2^-21 was
  // tried first: stiff steps approach |l| -> 1 from below and sent the hot zones of config 4 to the
  // general path often enough to cost 18 % of that config.)
  // b: right-hand side of the first solve; its forward elimination (dgesl, k ascending) rides along:
  // the pivot row's b_k is published with the row, so the first solve needs only back_solve().
  // wf (quad-uniform): this quad factorises.  With wf false (Newton-matrix reuse: the quad keeps its
  // factors) the quad goes through the same instruction stream but changes neither a nor b.
  template <class Mem>
  __device__ __forceinline__ unsigned factor(const Mem &m, int c, unsigned gmask, double (&b)[S], const bool wf) {
    unsigned lmax = 0u;
    bool bad = false;
#pragma unroll
    for (int k = 0; k < NEQ; k++) {
      const int ko = k & 3, ks = k >> 2;
      double *ub = m.ub(k & 1);
      if (c == ko) {
        volatile double *vb = ub;  // 64-bit stores straight from the row's registers (no tuple packing)
#pragma unroll
        for (int j = k; j < NEQ; j++) vb[j] = a[ks][j];
        vb[NEQ] = b[ks];
      }
      __syncwarp(gmask);
      const double piv = ub[k];
      const double bk = ub[NEQ];
      bad |= !(fabs(piv) > 0.0);
      const double inv = 1.0 / piv;
      if (wf && c == ko) a[ks][k] = inv;
#pragma unroll
      for (int s = 0; s < S; s++) {
        if (s < ks) continue;
        const bool mine = wf && ((s > ks) || (c > ko));  // row 4s+c is below the pivot row
        if (mine) {
          const double l = a[s][k] * inv;
          lmax = max(lmax, hi_abs(l));
          a[s][k] = l;
#pragma unroll
          for (int j = k + 1; j < NEQ; j++) a[s][j] = fma_(-l, ub[j], a[s][j]);
          b[s] = fma_(-l, bk, b[s]);
        }
      }
    }
    const unsigned f = (lmax >= 0x3FF00000u ? 1u : 0u) | (bad ? 2u : 0u);
    // make the flags quad-uniform
    unsigned r = f;
    r |= __shfl_xor_sync(gmask, r, 1, 4);
    r |= __shfl_xor_sync(gmask, r, 2, 4);
    return r;
  }

  // dgesl without interchanges: b[s] = my components of the right-hand side / solution
  __device__ __forceinline__ void solve(int c, unsigned gmask, double (&b)[S]) const {
    fwd_solve(c, gmask, b);
    back_solve(c, gmask, b);
  }
  // forward half (k ascending, axpy form)
  __device__ __forceinline__ void fwd_solve(int c, unsigned gmask, double (&b)[S]) const {
#pragma unroll
    for (int k = 0; k < NEQ; k++) {
      const int ko = k & 3, ks = k >> 2;
      const double bk = __shfl_sync(gmask, b[ks], ko, 4);
#pragma unroll
      for (int s = 0; s < S; s++) {
        if (s < ks) continue;
        if ((s > ks) || (c > ko)) b[s] = fma_(-a[s][k], bk, b[s]);
      }
    }
  }
  // backward half only (the forward half was fused into factor())
  __device__ __forceinline__ void back_solve(int c, unsigned gmask, double (&b)[S]) const {
#pragma unroll
    for (int k = NEQ - 1; k >= 0; k--) {
      const int ko = k & 3, ks = k >> 2;
      const double x = b[ks] * a[ks][k];  // lane ko: its 1/pivot (other lanes' x is unused)
      if (c == ko) b[ks] = x;
      const double xk = __shfl_sync(gmask, x, ko, 4);
#pragma unroll
      for (int s = 0; s < S; s++) {
        if (s > ks) continue;
        if ((s < ks) || (c < ko)) b[s] = fma_(-a[s][k], xk, b[s]);
      }
    }
  }
};

// ---- general path (rare): LINPACK dgefa / dgesl on a row-major n x n matrix in global memory ----
template <int NEQ>
__device__ __noinline__ bool quad_lu_general(double *P, int *ipvt) {
  bool ok = true;
  for (int k = 0; k < NEQ; k++) {
    int p = k;
    double amax = fabs(P[k * NEQ + k]);
    for (int i = k + 1; i < NEQ; i++) {
      const double v = fabs(P[i * NEQ + k]);
      if (v > amax) {
        amax = v;
        p = i;
      }
    }
    ipvt[k] = p;
    if (!(amax > 0.0)) {
      ok = false;
      P[k * NEQ + k] = 0.0;
      continue;
    }
    if (p != k)
      for (int j = k; j < NEQ; j++) {
        const double t = P[p * NEQ + j];
        P[p * NEQ + j] = P[k * NEQ + j];
        P[k * NEQ + j] = t;
      }
    const double inv = 1.0 / P[k * NEQ + k];
    for (int i = k + 1; i < NEQ; i++) P[i * NEQ + k] = P[i * NEQ + k] * inv;
    for (int i = k + 1; i < NEQ; i++) {
      const double l = P[i * NEQ + k];
      for (int j = k + 1; j < NEQ; j++) P[i * NEQ + j] = fma_(-l, P[k * NEQ + j], P[i * NEQ + j]);
    }
    P[k * NEQ + k] = inv;  // 1/pivot on the diagonal
  }
  return ok;
}
template <int NEQ>
__device__ __noinline__ void quad_solve_general(const double *P, const int *ipvt, double *b) {
  for (int k = 0; k < NEQ; k++) {
    const int p = ipvt[k];
    const double t = b[p];
    b[p] = b[k];
    b[k] = t;
    for (int i = k + 1; i < NEQ; i++) b[i] = fma_(-P[i * NEQ + k], t, b[i]);
  }
  for (int k = NEQ - 1; k >= 0; k--) {
    b[k] = b[k] * P[k * NEQ + k];
    const double t = b[k];
    for (int i = 0; i < k; i++) b[i] = fma_(-P[i * NEQ + k], t, b[i]);
  }
}

}  // namespace bz
