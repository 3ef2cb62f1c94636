// bz_coop_burn.cuh -- the persistent cooperative burn kernel: LU, solves and the BDF driver.
#pragma once
#include "bz_coop_kernel.cuh"

namespace bz {

// The factorised Newton matrix of a group's zone, in place in the group's shared-memory matrix M, where the
// rates left the rows of J: lane i owns row i at M + i*LD (LD = LANES + 1: the lanes of a group walk their rows
// in step, or read one column, without bank conflicts beyond the two wavefronts of a 64-bit access).
// a5: LU with partial pivoting, LINPACK tie-break (first maximal |a_ik| in the current row order); rows never
// move: each lane carries the LINPACK position of its row (= the step at which it became the pivot row) and
// the pivot lanes of the steps are kept as ints in the group's buffer urow; the pivot row is read where it
// lies.  The loops over k and j are rolled: 2 KB of code.
// Round 1 and most of round 2 kept each lane's row in REGISTERS instead (static indices, everything unrolled:
// 54 KB of code for n = 31, 62 registers for the row, the pivot row published through a double-buffered
// broadcast buffer).  Same operations in the same order, same bits, and slower on every instance, because the
// row's registers and the size of the code cost more than the shared-memory traffic of this form:
// burn_coop<31,32> 3 447 -> 3 258 ms (twice the warps at 128 registers), <14,16> 747 -> 555 ms, <8,8> 471 -> 387
// ms, <3,4> 415 -> 372 ms (configs 5, 3, 2 and 1's networks on the generic kernel).
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
