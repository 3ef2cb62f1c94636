// bz_coop_burn.cuh -- the persistent cooperative burn kernel: LU, solves and the BDF driver.
#pragma once
#include "bz_coop_kernel.cuh"

namespace bz {

// Per-lane view of the factorised Newton matrix.
template <int NEQ, int LANES>
struct LuRow {
  double a[NEQ];  // my row: multipliers l_ik (k < pos), then U (k >= pos)
  double myinv;   // 1/pivot of the step at which my row was the pivot row
  int pos;        // LINPACK position of my row (= step at which it became the pivot row)
  unsigned plpack[(NEQ + 3) / 4];  // pivot lane of every step, 8 bits each

  __device__ __forceinline__ int pivot_lane(int k) const { return (plpack[k >> 2] >> ((k & 3) * 8)) & 0xff; }

  // my row of P = I - gamma*J, from the row of J that the rates left in the group's matrix M
  template <class G>
  __device__ __forceinline__ void form(const G &g, double gamma, bool act, int n) {
#pragma unroll
    for (int j = 0; j < NEQ; j++) {
      const double Jij = (act && j < n) ? g.M[g.lig * CoopSmem<NEQ, LANES>::LD + j] : 0.0;
      a[j] = fma_(-gamma, Jij, (j == g.lig) ? 1.0 : 0.0);
    }
  }

  // a5: in-place LU with partial pivoting, LINPACK tie-break (first maximal |a_ik| in the
  // current row order), rows never move.  Returns false if a pivot column is all zero.
  template <class G>
  __device__ __forceinline__ bool factor(const G &g) {
    const int lig = g.lig;
    pos = lig;
    myinv = 0.0;
    bool ok = true;
#pragma unroll
    for (int w = 0; w < (NEQ + 3) / 4; w++) plpack[w] = 0u;
#pragma unroll
    for (int k = 0; k < NEQ; k++) {
      const bool cand0 = (pos >= k) && (lig < NEQ);
      const unsigned long long key =
          cand0 ? (unsigned long long)(__double_as_longlong(a[k]) & 0x7fffffffffffffffLL) : 0ull;
      const unsigned long long kmax = g.gmax(key);
      if (kmax == 0ull || kmax > 0x7ff0000000000000ull) ok = false;  // zero or NaN pivot column
      const bool cand = cand0 && (key == kmax);
      unsigned ball = g.gballot(cand);
      if (__popc(ball) > 1) {  // exact tie: smallest LINPACK position wins
        const int mp = g.gmin(cand ? pos : 0x7fffffff);
        ball = g.gballot(cand && pos == mp);
      }
      const int pl = __ffs(ball) - 1;
      plpack[k >> 2] |= (unsigned)(pl & 0xff) << ((k & 3) * 8);
      const int ppos = __shfl_sync(g.gmask, pos, pl & (LANES - 1), LANES);
      const bool isp = (lig == pl);
      if (pos == k) pos = ppos;
      if (isp) pos = k;
      double *ub = g.urow + (k & 1) * LANES;
      if (isp) {
#pragma unroll
        for (int j = k; j < NEQ; j++) ub[j] = a[j];
      }
      g.sync();
      const double inv = 1.0 / ub[k];
      if (isp) myinv = inv;
      if (pos > k) {
        const double l = a[k] * inv;
        a[k] = l;
#pragma unroll
        for (int j = k + 1; j < NEQ; j++) a[j] = fma_(-l, ub[j], a[j]);
      }
    }
    return ok;
  }

  // a6: solve P x = b (dgesl order).  b = my component on entry, x_lig on return.
  template <class G>
  __device__ __forceinline__ double solve(const G &g, double b) const {
#pragma unroll
    for (int k = 0; k < NEQ; k++) {
      const double bk = g.bcast(b, pivot_lane(k));
      if (pos > k) b = fma_(-a[k], bk, b);
    }
#pragma unroll
    for (int k = NEQ - 1; k >= 0; k--) {
      const double x = b * myinv;
      if (pos == k) b = x;
      const double xk = g.bcast(x, pivot_lane(k));
      if (pos < k) b = fma_(-a[k], xk, b);
    }
    // x_j sits on the lane whose row has position j: route it to lane j
    g.sync();
    if (g.lig < NEQ) g.xs[pos] = b;
    g.sync();
    return (g.lig < NEQ) ? g.xs[g.lig] : 0.0;
  }
};

// The same factorisation with the rows left where the rates put them: in the group's shared-memory
// matrix M (lane i owns row i at M + i*LD, LD = LANES + 1: lanes i and i + 16 share a bank, the minimum
// for 64-bit accesses).  A warp-per-zone lane then carries no row in registers (62 of them for n = 31),
// the pivot row is read where it lies instead of being published to a broadcast buffer, and the loops
// over k and j are rolled: the factorisation is 2 KB of code instead of 54 KB.  Operations and their
// order are those of LuRow: same bits.  The pivot lanes of the steps are kept in the group's old
// broadcast buffer (urow) as ints.
template <int NEQ, int LANES>
struct LuSmem {
  static constexpr int LD = CoopSmem<NEQ, LANES>::LD;
  double myinv;  // 1/pivot of the step at which my row was the pivot row
  int pos;       // LINPACK position of my row

  template <class G>
  __device__ __forceinline__ void form(const G &g, double gamma, bool act, int n) {
    if (g.lig < NEQ) {
      double *row = g.M + g.lig * LD;
#pragma unroll 4
      for (int j = 0; j < NEQ; j++) {
        const double Jij = (act && j < n) ? row[j] : 0.0;
        row[j] = fma_(-gamma, Jij, (j == g.lig) ? 1.0 : 0.0);
      }
    }
  }

  template <class G>
  __device__ __forceinline__ bool factor(const G &g) {
    const int lig = g.lig;
    pos = lig;
    myinv = 0.0;
    bool ok = true;
    double *row = g.M + (lig < NEQ ? lig : 0) * LD;
    int *pls = reinterpret_cast<int *>(g.urow);
#pragma unroll 1
    for (int k = 0; k < NEQ; k++) {
      g.sync();  // the rows as updated in step k - 1 (or formed) are visible to every lane
      const double my = row[k];
      const bool cand0 = (pos >= k) && (lig < NEQ);
      const unsigned long long key =
          cand0 ? (unsigned long long)(__double_as_longlong(my) & 0x7fffffffffffffffLL) : 0ull;
      const unsigned long long kmax = g.gmax(key);
      if (kmax == 0ull || kmax > 0x7ff0000000000000ull) ok = false;  // zero or NaN pivot column
      const bool cand = cand0 && (key == kmax);
      unsigned ball = g.gballot(cand);
      if (__popc(ball) > 1) {  // exact tie: smallest LINPACK position wins
        const int mp = g.gmin(cand ? pos : 0x7fffffff);
        ball = g.gballot(cand && pos == mp);
      }
      const int pl = __ffs(ball) - 1;
      if (lig == 0) pls[k] = pl;
      const int ppos = __shfl_sync(g.gmask, pos, pl & (LANES - 1), LANES);
      const bool isp = (lig == pl);
      if (pos == k) pos = ppos;
      if (isp) pos = k;
      const double *prow = g.M + (pl & (LANES - 1)) * LD;  // the pivot row, where it lies (its owner does not touch it now)
      const double inv = 1.0 / prow[k];
      if (isp) myinv = inv;
      if (pos > k && lig < NEQ) {
        const double l = my * inv;
        row[k] = l;
        // Loads staged by hand, four columns at a time, then two: written as row[j] = fma(-l, prow[j], row[j])
        // the compiler must assume that row and prow overlap and chains load -> FMA -> store -> load, ~45
        // cycles per column.  An odd number of columns takes the next one along -- index NEQ, padding of the
        // row (NEQ < LD), updated and never read -- so that no column is left for a serial tail.
        static_assert(NEQ < LD, "padding column");
        int j = k + 1;
        const int end = j + ((NEQ - j + 1) & ~1);
#pragma unroll 1
        for (; j + 4 <= end; j += 4) {
          double p[4], r[4];
#pragma unroll
          for (int u = 0; u < 4; u++) p[u] = prow[j + u], r[u] = row[j + u];
#pragma unroll
          for (int u = 0; u < 4; u++) row[j + u] = fma_(-l, p[u], r[u]);
        }
        if (j < end) {
          const double p0 = prow[j], p1 = prow[j + 1], r0 = row[j], r1 = row[j + 1];
          row[j] = fma_(-l, p0, r0);
          row[j + 1] = fma_(-l, p1, r1);
        }
      }
    }
    g.sync();
    return ok;
  }

  template <class G>
  __device__ __forceinline__ double solve(const G &g, double b) const {
    const double *row = g.M + (g.lig < NEQ ? g.lig : 0) * LD;
    const int *pls = reinterpret_cast<const int *>(g.urow);
#pragma unroll
    for (int k = 0; k < NEQ; k++) {
      const double bk = g.bcast(b, pls[k]);
      if (pos > k) b = fma_(-row[k], bk, b);
    }
#pragma unroll
    for (int k = NEQ - 1; k >= 0; k--) {
      const double x = b * myinv;
      if (pos == k) b = x;
      const double xk = g.bcast(x, pls[k]);
      if (pos < k) b = fma_(-row[k], xk, b);
    }
    g.sync();
    if (g.lig < NEQ) g.xs[pos] = b;
    g.sync();
    return (g.lig < NEQ) ? g.xs[g.lig] : 0.0;
  }
};

template <int NEQ, int LANES, bool SMEM = (LANES == 32)>
struct LuPick {
  typedef LuRow<NEQ, LANES> type;
};
template <int NEQ, int LANES>
struct LuPick<NEQ, LANES, true> {
  typedef LuSmem<NEQ, LANES> type;
};

// Nordsieck helpers on my component.  Arrays are indexed with compile-time indices only.
__device__ __forceinline__ void nord_predict(double (&Z)[QMAX + 1], int q) {
#pragma unroll
  for (int k = 1; k <= QMAX; k++)
#pragma unroll
    for (int j = QMAX; j >= k; j--)
      if (j <= q && k <= q) Z[j - 1] = Z[j - 1] + Z[j];
}
__device__ __forceinline__ void nord_retract(double (&Z)[QMAX + 1], int q) {
#pragma unroll
  for (int k = 1; k <= QMAX; k++)
#pragma unroll
    for (int j = QMAX; j >= k; j--)
      if (j <= q && k <= q) Z[j - 1] = Z[j - 1] - Z[j];
}
__device__ __forceinline__ void nord_rescale(double (&Z)[QMAX + 1], int q, double eta) {
  double r = eta;
#pragma unroll
  for (int j = 1; j <= QMAX; j++) {
    if (j <= q) {
      Z[j] = Z[j] * r;
      r = r * eta;
    }
  }
}
// d(x) = x^2 prod_{i=1..cnt} (x + xi[i]);  d[0..7]
__device__ __forceinline__ void build_d(int cnt, const double (&xi)[QMAX + 1], double (&d)[8]) {
#pragma unroll
  for (int j = 0; j < 8; j++) d[j] = 0.0;
  d[2] = 1.0;
#pragma unroll
  for (int i = 1; i <= QMAX - 1; i++) {
    if (i <= cnt) {
      // degree before this factor is i + 1
#pragma unroll
      for (int j = QMAX + 1; j >= 1; j--)
        if (j <= i + 2) d[j] = fma_(xi[i], d[j], d[j - 1]);
      d[0] = xi[i] * d[0];
    }
  }
}
template <int J>
__device__ __forceinline__ double sel(const double (&v)[J], int i) {  // v[i] without local memory
  double r = v[0];
#pragma unroll
  for (int j = 1; j < J; j++) r = (i == j) ? v[j] : r;
  return r;
}

}  // namespace bz
