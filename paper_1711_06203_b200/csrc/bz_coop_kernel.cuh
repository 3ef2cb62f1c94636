// bz_coop_kernel.cuh -- body of the cooperative burn kernel (see bz_coop.cuh for the mapping).
#pragma once
#include "bz_coop.cuh"

namespace bz {

// EXT: the optional model extensions -- density exponents of weak rates and c_v from the
// analytic EOS -- are compiled into a separate instantiation, so that networks without
// them run the kernel without a trace of either (they cost 3.4 % of config 5 when compiled in).
template <int NEQ, int LANES, bool EXT = false>
struct Group {
  static constexpr int LD = CoopSmem<NEQ, LANES>::LD;
  // identity of this lane
  unsigned gmask;  // lanes of my group within the warp
  int lig;         // lane in group = component index
  // tables in shared memory (per block)
  int N, n, K;
  double fac, inv_n;
  const double *lnA, *en, *B, *Q, *invsym, *aion, *sp_dy;
  const double *rexp;  // density exponents of weak rates, or nullptr
  const double *zp1;   // 1 + Z_i: c_v from the analytic EOS, or nullptr (constant c_v in fac)
  double eos_extra;
  const int *rp, *sp_off, *sp_k, *cl_off, *cl_ks;
  // per-group scratch in shared memory
  double *ysh, *R, *dRdT, *dRdY, *M, *urow, *xs;
  // constant source of my component (burn_zones_src); added to f after the network's own sums
  bool has_src;
  double src;

  __device__ __forceinline__ void sync() const { __syncwarp(gmask); }

  __device__ __forceinline__ double gsum(double v) const {
#pragma unroll
    for (int s = LANES / 2; s >= 1; s >>= 1) v = v + __shfl_xor_sync(gmask, v, s, LANES);
    return v;
  }
  // 64-bit maximum over the group.  A full warp (LANES == 32) takes it in two hardware reductions
  // (redux.sync): the largest high word, then the largest low word among the lanes that hold it -- exact,
  // and 9.5 % of config 5's time less than the 5-round butterfly of 64-bit shuffles and compares it
  // replaces.  Sub-warp groups keep the butterfly: redux with a partial member mask measured 5 % slower.
  __device__ __forceinline__ unsigned long long gmax(unsigned long long v) const {
    if constexpr (LANES == 32) {
      const unsigned hi = (unsigned)(v >> 32), lo = (unsigned)v;
      const unsigned mh = __reduce_max_sync(0xffffffffu, hi);
      const unsigned ml = __reduce_max_sync(0xffffffffu, hi == mh ? lo : 0u);
      return ((unsigned long long)mh << 32) | (unsigned long long)ml;
    } else {
#pragma unroll
      for (int s = LANES / 2; s >= 1; s >>= 1) {
        unsigned long long o = __shfl_xor_sync(gmask, v, s, LANES);
        v = o > v ? o : v;
      }
      return v;
    }
  }
  __device__ __forceinline__ int gmin(int v) const {
#pragma unroll
    for (int s = LANES / 2; s >= 1; s >>= 1) {
      int o = __shfl_xor_sync(gmask, v, s, LANES);
      v = o < v ? o : v;
    }
    return v;
  }
  // group-relative ballot
  __device__ __forceinline__ unsigned gballot(bool p) const {
    unsigned b = __ballot_sync(gmask, p);
    if (LANES == 32) return b;
    return (b >> ((threadIdx.x & 31) & ~(LANES - 1))) & ((1u << (LANES & 31)) - 1u);
  }
  __device__ __forceinline__ bool gany(bool p) const { return gballot(p) != 0u; }
  __device__ __forceinline__ double bcast(double v, int src) const { return __shfl_sync(gmask, v, src, LANES); }

  // WRMS norm, association = LANES interleaved partial sums + xor butterfly
  __device__ __forceinline__ double wrms(double v, double w) const {
    const double d = v * w;
    const double s = gsum(d * d);
    return sqrt(s * inv_n);
  }

  // a3 (+a4): f (own component) and, if WITH_J, row `lig` of J left in M (shared memory).
  template <bool WITH_J>
  __device__ __forceinline__ double rates(double rho, double y) {
    sync();  // previous readers of the scratch are done
    if (lig < n) ysh[lig] = y;
    sync();
    const double T = ysh[0];  // internal order: T first, species i at i + 1
    const double T9 = T * 1e-9;
    const double lnT9 = log_(T9);
    const double t13 = exp_(lnT9 * (-1.0 / 3.0));
    const double t13third = t13 * (1.0 / 3.0);
    const double invT = 1.0 / T;
    const double rho2 = rho * rho;
    const double lnrho = (EXT && rexp) ? log_(rho) : 0.0;  // lambda_k *= rho^e_k inside the exponent
    for (int k = lig; k < K; k += LANES) {
      const int4 rpk = reinterpret_cast<const int4 *>(rp)[k];
      const int m = rpk.x & 0xff;
      const int r0 = rpk.y & 0xff, r1 = (rpk.y >> 8) & 0xff, r2 = (rpk.y >> 16) & 0xff;
      double arg = fma_(-B[k], t13, fma_(en[k], lnT9, lnA[k]));
      if (EXT && rexp) arg = fma_(rexp[k], lnrho, arg);
      const double lam = exp_(arg);
      const double pref = (lam * (m == 1 ? 1.0 : (m == 2 ? rho : rho2))) * invsym[k];
      const double y0 = ysh[r0 + 1];
      const double v0 = fabs(y0);
      double Rk, d0, d1 = 0.0, d2 = 0.0;
      bool neg0 = y0 < 0.0, neg1 = false, neg2 = false;
      if (m == 1) {
        Rk = pref * v0;
        d0 = pref;
      } else if (m == 2) {
        const double y1 = ysh[r1 + 1];
        const double v1 = fabs(y1);
        neg1 = y1 < 0.0;
        Rk = (pref * v0) * v1;
        if (r1 == r0) {
          d0 = pref * (v1 + v0);
        } else {
          d0 = pref * v1;
          d1 = pref * v0;
        }
      } else {
        const double y1 = ysh[r1 + 1], y2 = ysh[r2 + 1];
        const double v1 = fabs(y1), v2 = fabs(y2);
        neg1 = y1 < 0.0;
        neg2 = y2 < 0.0;
        Rk = ((pref * v0) * v1) * v2;
        const double P0 = v1 * v2, P1 = v0 * v2, P2 = v0 * v1;
        // slots = distinct species in order of first appearance
        double s0 = P0;
        if (r1 == r0) s0 = s0 + P1;
        if (r2 == r0) s0 = s0 + P2;
        d0 = pref * s0;
        if (r1 != r0) {
          double s1 = P1;
          if (r2 == r1) s1 = s1 + P2;
          d1 = pref * s1;
          if (r2 != r0 && r2 != r1) d2 = pref * P2;
        } else if (r2 != r0) {
          d1 = pref * P2;
        }
      }
      const bool anyneg = neg0 | neg1 | neg2;
      if (anyneg) Rk = -Rk;  // reading s19: odd, monotone extension to Y < 0
      R[k] = Rk;
      if (WITH_J) {
        // sign of the partial w.r.t. a slot's species: flipped unless that species is negative
        const int c0 = rpk.z & 0xff, c1 = (rpk.z >> 8) & 0xff, c2 = (rpk.z >> 16) & 0xff;
        const int nslot = (rpk.x >> 8) & 0xff;
        if (anyneg) {
          if (!(ysh[c0 + 1] < 0.0)) d0 = -d0;
          if (nslot > 1 && !(ysh[c1 + 1] < 0.0)) d1 = -d1;
          if (nslot > 2 && !(ysh[c2 + 1] < 0.0)) d2 = -d2;
        }
        dRdY[3 * k + 0] = d0;
        dRdY[3 * k + 1] = d1;
        dRdY[3 * k + 2] = d2;
        const double g = fma_(B[k], t13third, en[k]);
        dRdT[k] = (Rk * g) * invT;
      }
    }
    sync();
    // analytic EOS: c_v = 1.5 R (extra + sum_i (1+Z_i) Y_i) + 4 a T^3 / rho, raw Y, i ascending; every lane
    // computes it (uniform code, identical bits); facv replaces the constant fac
    double facv = fac, invcv = 0.0, T2 = 0.0, invrho = 0.0;
    if (EXT && zp1) {
      double ysum = eos_extra;
      for (int i = 0; i < N; i++) ysum = fma_(zp1[i], ysh[i + 1], ysum);
      T2 = T * T;
      invrho = 1.0 / rho;
      const double cv = fma_(1.5 * RGAS, ysum, ((4.0 * ARAD) * (T2 * T)) * invrho);
      invcv = 1.0 / cv;
      facv = NA_MEV * invcv;
    }
    double f = 0.0, jt0 = 0.0;
    const int sp = lig - 1;  // my species (lanes 1..N); lane 0 owns T
    if (lig >= 1 && lig <= N) {
      const int e = sp_off[sp + 1];
      for (int t = sp_off[sp]; t < e; t++) f = fma_(sp_dy[t], R[sp_k[t]], f);
    } else if (lig == 0) {
      // the temperature lane sums over ALL reactions: its two K-term chains (energy rate and
      // d/dT of it) share one loop, so the single active lane has two independent FMAs in flight
      double s = 0.0;
      if (WITH_J) {
        for (int k = 0; k < K; k++) {
          s = fma_(Q[k], R[k], s);
          jt0 = fma_(Q[k], dRdT[k], jt0);
        }
      } else {
        for (int k = 0; k < K; k++) s = fma_(Q[k], R[k], s);
      }
      f = facv * s;
    }
    if (WITH_J) {
      double *row = M + lig * LD;
      if (lig < n)
        for (int j = 0; j < n; j++) row[j] = 0.0;
      double jt = 0.0;
      if (lig >= 1 && lig <= N) {
        const int e = sp_off[sp + 1];
        for (int t = sp_off[sp]; t < e; t++) {
          const int k = sp_k[t];
          const double dy = sp_dy[t];
          const int4 rpk = reinterpret_cast<const int4 *>(rp)[k];
          const int nslot = (rpk.x >> 8) & 0xff;
          const int c0 = rpk.z & 0xff, c1 = (rpk.z >> 8) & 0xff, c2 = (rpk.z >> 16) & 0xff;
          row[c0 + 1] = fma_(dy, dRdY[3 * k], row[c0 + 1]);
          if (nslot > 1) row[c1 + 1] = fma_(dy, dRdY[3 * k + 1], row[c1 + 1]);
          if (nslot > 2) row[c2 + 1] = fma_(dy, dRdY[3 * k + 2], row[c2 + 1]);
          row[0] = fma_(dy, dRdT[k], row[0]);
        }
        // my column of the temperature row: sum_k Q_k dR_k/dY_lig, k ascending
        const int ce = cl_off[sp + 1];
        for (int c = cl_off[sp]; c < ce; c++) {
          const int ks = cl_ks[c];
          jt = fma_(Q[ks & 0xffff], dRdY[3 * (ks & 0xffff) + (ks >> 16)], jt);
        }
      } else if (lig == 0) {
        jt = jt0;  // summed alongside f above (same k-ascending fma chain)
      }
      sync();  // rows of the species are complete before the T row is written
      if (EXT && zp1) {
        // dT/dt = facv s: the row gains -f_T (dc_v/dy_j) / c_v, dc_v/dT = 12 a T^2/rho, dc_v/dY_j = 1.5 R (1+Z_j)
        const double gq = bcast(f, 0) * invcv;
        const double dcv = (lig == 0) ? ((12.0 * ARAD) * T2) * invrho : ((lig <= N) ? (1.5 * RGAS) * zp1[sp] : 0.0);
        if (lig < n) M[lig] = fma_(-gq, dcv, facv * jt);
      } else if (lig < n) {
        M[lig] = fac * jt;  // row 0 = temperature equation
      }
      sync();
    }
    if (has_src) f = f + src;
    return f;
  }
};

}  // namespace bz
