// bz_tpz.cuh -- thread-per-zone burn kernel for small networks (n <= 16), DESIGN.md section 5.2.
//
// One thread integrates one zone; 32 zones per warp run the same straight-line code, so every
// FP64 lane does useful work (no cross-lane shuffles, no redundant scalar work).  The network
// functions (rates, Jacobian) are generated per topology (gen/net_*.cuh): all state vectors are
// register arrays with compile-time indices.  What does not fit in registers lives in shared
// memory, one column per thread (element e of thread t at [e*BLOCK + t]: conflict-free):
//   the Newton matrix / its LU factors (n*n doubles), the Nordsieck array (6*n), the weights (n).
// LU (a5) is left-looking over register panels of W columns: a panel is loaded once (structural
// zeros of I - gamma*J as constants), updated with the previous columns' multipliers (one shared-
// memory load per W fused multiply-adds), factorised in registers and stored once.  The first
// Newton solve's forward elimination rides along as an extra column of the last panel.
// Pivoting: the unknowns are ordered temperature-first so partial pivoting keeps
// the natural order almost always; the panel code VERIFIES that (exact comparison of |a_ik| with
// |a_kk|) and a zone that does need an interchange redoes that factorisation on a slow, fully
// general path with LINPACK interchanges (bit-identical to the oracle either way).
// Zones are pulled one by one from a global atomic queue by each THREAD (a2): a lane that
// finishes its zone starts the next one while its neighbours keep stepping.
#pragma once
#include <cstdint>
#include "bz_coop.cuh"  // constants, BurnArgs, eta_of, factorial_, inv_small_int

namespace bz {

struct TpzNet {
  const double *coef;  // device: lnA[K] n[K] B[K] Q[K] aion[N]
  double fac;
};

template <int NEQ, int BLOCK>
struct TpzMem {
  // doubles per thread in shared memory
  static constexpr int P_OFF = 0;
  static constexpr int Z_OFF = NEQ * NEQ;
  static constexpr int W_OFF = Z_OFF + (QMAX + 1) * NEQ;
  static constexpr int PER_THREAD = W_OFF + NEQ;
  double *base;  // smem + tid
  __device__ __forceinline__ double &P(int i, int j) const { return base[(P_OFF + i * NEQ + j) * BLOCK]; }
  __device__ __forceinline__ double &Z(int j, int i) const { return base[(Z_OFF + j * NEQ + i) * BLOCK]; }
  __device__ __forceinline__ double &W(int i) const { return base[(W_OFF + i) * BLOCK]; }
};

// receivers of the generated Jacobian entries
template <int NEQ, int BLOCK>
struct NewtonStore {  // P_ij = fma(-gamma, J_ij, delta_ij) -> shared memory
  TpzMem<NEQ, BLOCK> m;
  double gamma;
  __device__ __forceinline__ void set(int i, int j, double Jij) { m.P(i, j) = fma_(-gamma, Jij, (i == j) ? 1.0 : 0.0); }
};
template <int NEQ>
struct JfStore {  // (J f)_i accumulated in column order (init: h0 from the exact y'')
  const double (&f)[NEQ];
  double (&s)[NEQ];
  __device__ __forceinline__ JfStore(const double (&f_)[NEQ], double (&s_)[NEQ]) : f(f_), s(s_) {}
  __device__ __forceinline__ void set(int i, int j, double Jij) { s[i] = fma_(Jij, f[j], s[i]); }
};
struct NoStore {
  __device__ __forceinline__ void set(int, int, double) {}
};

// WRMS norm with 4 interleaved partial sums combined as (p0+p2)+(p1+p3)  (norm_lanes = 4)
template <int NEQ, int BLOCK>
__device__ __forceinline__ double wrms4(const double (&v)[NEQ], const TpzMem<NEQ, BLOCK> &m, double inv_n) {
  double p[4] = {0.0, 0.0, 0.0, 0.0};
#pragma unroll
  for (int i = 0; i < NEQ; i++) {
    const double d = v[i] * m.W(i);
    p[i & 3] = fma_(d, d, p[i & 3]);
  }
  return sqrt(((p[0] + p[2]) + (p[1] + p[3])) * inv_n);
}

__device__ __forceinline__ unsigned hi_abs(double x) { return (unsigned)(__double_as_longlong(x) >> 32) & 0x7fffffffu; }

// a5 + forward half of the first a6: left-looking panel LU without interchanges.
// On return: L (below diagonal), U (above) and 1/pivot (ON the diagonal) are in shared memory,
// b is forward-eliminated.  flags: bit 0 = an interchange would have been needed (results are
// then garbage and the caller takes the general path), bit 1 = zero/NaN pivot.
template <class Net, int BLOCK, int W>
__device__ __forceinline__ unsigned lu_panels(const TpzMem<Net::NEQ, BLOCK> &m, double (&b)[Net::NEQ]) {
  constexpr int NEQ = Net::NEQ;
  bool swap_needed = false, bad = false;
#pragma unroll
  for (int j0 = 0; j0 < NEQ; j0 += W) {
    const int wp = (NEQ - j0 < W) ? NEQ - j0 : W;
    const bool lastp = (j0 + W >= NEQ);
    double c[W][NEQ];
#pragma unroll
    for (int jj = 0; jj < W; jj++)
#pragma unroll
      for (int i = 0; i < NEQ; i++)
        if (jj < wp) c[jj][i] = Net::nz(i, j0 + jj) ? m.P(i, j0 + jj) : ((i == j0 + jj) ? 1.0 : 0.0);
    // previous columns
#pragma unroll
    for (int k = 0; k < NEQ; k++) {
      if (k < j0) {
#pragma unroll
        for (int i = k + 1; i < NEQ; i++) {
          const double l = m.P(i, k);
#pragma unroll
          for (int jj = 0; jj < W; jj++)
            if (jj < wp) c[jj][i] = fma_(-l, c[jj][k], c[jj][i]);
          if (lastp) b[i] = fma_(-l, b[k], b[i]);
        }
      }
    }
    // the panel itself
#pragma unroll
    for (int jj = 0; jj < W; jj++) {
      if (jj < wp) {
        const int k = j0 + jj;
        const double piv = c[jj][k];
        const unsigned hk = hi_abs(piv);
        bool maybe = false;
#pragma unroll
        for (int i = k + 1; i < NEQ; i++) maybe |= (hi_abs(c[jj][i]) >= hk);
        if (maybe) {
#pragma unroll
          for (int i = k + 1; i < NEQ; i++) swap_needed |= (fabs(c[jj][i]) > fabs(piv));
        }
        bad |= !(fabs(piv) > 0.0);
        const double inv = 1.0 / piv;
        c[jj][k] = inv;
#pragma unroll
        for (int i = k + 1; i < NEQ; i++) c[jj][i] = c[jj][i] * inv;
#pragma unroll
        for (int j2 = 0; j2 < W; j2++)
          if (j2 > jj && j2 < wp) {
#pragma unroll
            for (int i = k + 1; i < NEQ; i++) c[j2][i] = fma_(-c[jj][i], c[j2][k], c[j2][i]);
          }
        if (lastp) {
#pragma unroll
          for (int i = k + 1; i < NEQ; i++) b[i] = fma_(-c[jj][i], b[k], b[i]);
        }
      }
    }
#pragma unroll
    for (int jj = 0; jj < W; jj++)
#pragma unroll
      for (int i = 0; i < NEQ; i++)
        if (jj < wp) m.P(i, j0 + jj) = c[jj][i];
  }
  return (swap_needed ? 1u : 0u) | (bad ? 2u : 0u);
}

// backward half of a6 (dgesl order, k descending), no interchanges
template <int NEQ, int BLOCK>
__device__ __forceinline__ void back_subst(const TpzMem<NEQ, BLOCK> &m, double (&b)[NEQ]) {
#pragma unroll
  for (int k = NEQ - 1; k >= 0; k--) {
    b[k] = b[k] * m.P(k, k);  // the diagonal holds 1/pivot
#pragma unroll
    for (int i = 0; i < k; i++) b[i] = fma_(-m.P(i, k), b[k], b[i]);
  }
}
template <int NEQ, int BLOCK>
__device__ __forceinline__ void fwd_subst(const TpzMem<NEQ, BLOCK> &m, double (&b)[NEQ]) {
#pragma unroll
  for (int k = 0; k < NEQ; k++)
#pragma unroll
    for (int i = k + 1; i < NEQ; i++) b[i] = fma_(-m.P(i, k), b[k], b[i]);
}

// General path (rare): LINPACK dgefa/dgesl with interchanges on the shared-memory matrix.
// Dynamic indices are fine here (shared / local memory); speed is irrelevant.
template <int NEQ, int BLOCK>
__device__ __noinline__ bool lu_general(const TpzMem<NEQ, BLOCK> &m, int *ipvt) {
  bool ok = true;
  for (int k = 0; k < NEQ; k++) {
    int p = k;
    double amax = fabs(m.P(k, k));
    for (int i = k + 1; i < NEQ; i++) {
      const double v = fabs(m.P(i, k));
      if (v > amax) {
        amax = v;
        p = i;
      }
    }
    ipvt[k] = p;
    if (!(amax > 0.0)) {
      ok = false;
      m.P(k, k) = 0.0;
      continue;
    }
    if (p != k)
      for (int j = k; j < NEQ; j++) {
        const double t = m.P(p, j);
        m.P(p, j) = m.P(k, j);
        m.P(k, j) = t;
      }
    const double inv = 1.0 / m.P(k, k);
    for (int i = k + 1; i < NEQ; i++) m.P(i, k) = m.P(i, k) * inv;
    for (int i = k + 1; i < NEQ; i++) {
      const double l = m.P(i, k);
      for (int j = k + 1; j < NEQ; j++) m.P(i, j) = fma_(-l, m.P(k, j), m.P(i, j));
    }
    m.P(k, k) = inv;  // same convention as the panel path: 1/pivot on the diagonal
  }
  return ok;
}
template <int NEQ, int BLOCK>
__device__ __noinline__ void solve_general(const TpzMem<NEQ, BLOCK> &m, const int *ipvt, double *b) {
  for (int k = 0; k < NEQ; k++) {
    const int p = ipvt[k];
    const double t = b[p];
    b[p] = b[k];
    b[k] = t;
    for (int i = k + 1; i < NEQ; i++) b[i] = fma_(-m.P(i, k), t, b[i]);
  }
  for (int k = NEQ - 1; k >= 0; k--) {
    b[k] = b[k] * m.P(k, k);
    const double t = b[k];
    for (int i = 0; i < k; i++) b[i] = fma_(-m.P(i, k), t, b[i]);
  }
}

}  // namespace bz
