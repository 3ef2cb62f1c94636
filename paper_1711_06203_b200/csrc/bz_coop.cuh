// bz_coop.cuh -- cooperative burn kernel: LANES threads of a warp integrate one zone.
//
// Mapping: lane i of a group owns component i of every n-vector
// (Nordsieck rows, weights, corrections) in registers and ROW i of the Newton matrix P = I - gamma*J
// in the group's shared-memory matrix.  A warp holds 32/LANES zones.  Groups pull zones from a global atomic work queue
// (step a2: compaction against step-count divergence -- a group that finishes its zone fetches
// the next one, so co-resident zones never wait for the slowest of a fixed batch).
//   a3/a4 rates + Jacobian: reactions are dealt round-robin to lanes (one exp each), the
//         per-reaction rate and partials go through shared memory, then lane i gathers row i.
//   a5    LU: in place in shared memory, implicit row pivoting (rows never move; each lane carries its
//         LINPACK position `pos`), pivot search by a 64-bit maximum over the group, the pivot row read
//         where it lies, rank-1 update of the lane's own row with fma.
//   a6    solves: dgesl order; the pivot component is broadcast by shuffle.
//   a7/a8 BDF bookkeeping: per lane on its own component; step/order control is computed
//         redundantly by every lane of the group (identical bits, no communication).
// The floating-point operation sequence per component is the one fixed in DESIGN.md 3.6, so the
// results are bit-identical to the CPU oracle run with norm_lanes = LANES.
#pragma once
#include <cstdint>
#include "bz_math.cuh"

namespace bz {

// ---- constants of BZ-BDF v1 ---------------------------------------------------
constexpr int QMAX = 5, MAXCOR = 3, MXNCF = 10, MXNEF = 7, MXSTEP = 20000;
constexpr double NTOL = 0.1, CRDOWN = 0.3, RDIV = 2.0, ETACF = 0.25;
constexpr double BIAS1 = 4.0, BIAS2 = 6.0, BIAS3 = 10.0, ADDON = 1e-6, THRESH = 1.5;
constexpr double ETAMIN = 0.1, ETAMXF = 0.2, ETAMX1 = 1e4, ETAMAX = 2.0, SLIVER = 1e-6;
// Newton-matrix reuse (bz_set_policy 1, "BZ-BDF v2"): refactor when |gamma/gamma_P - 1|
// exceeds CCMAX or MSBP steps were accepted since the last factorisation
// analytic EOS for c_v: N_A k_B [erg/mol/K], radiation constant a [erg/cm^3/K^4], N_A MeV
constexpr double RGAS = 8.31446261815324e7, ARAD = 7.565733250e-15, NA_MEV = 9.648533212331e17;
constexpr double CCMAX = 0.3;
constexpr int MSBP = 20;

// flat network tables in device memory (built by net_create)
struct DevNet {
  int N, n, K, nterm, ncl;
  double fac;             // N_A MeV / cv
  const double *dbl;      // lnA[K] en[K] B[K] Q[K] invsym[K] aion[N] sp_dy[nterm] (+ rexp[K] if has_rexp)
  const int *itab;        // rp[4K] sp_off[N+1] sp_k[nterm] cl_off[N+1] cl_ks[ncl]
  int ndbl, nint;
  int has_rexp;           // density exponents of weak rates present (bz_net_desc.rate_rho_exp)
  int eos;                // c_v from the analytic EOS (bz_net_desc.zion): zp1[N] follows rexp in dbl; fac unused
  double eos_extra;
};

struct BurnArgs {
  long long nz;   // zones of this launch
  long long ld;   // row stride of X, X_out, src_X in doubles (= nz, except for the chunks of burn_zones_host)
  const double *rho, *T, *X;
  double dt, rtol, atol;
  double *T_out, *X_out;
  int *nsteps;
  unsigned long long *queue;     // work-queue head
  unsigned long long *counters;  // [8]
  const double *src_T, *src_X;   // constant source terms (burn_zones_src), both nullptr = none
  int mxstep, mxnef, mxncf;      // limits behind the failure codes -3 / -2 / -1 (bz_set_limits)
  int static_sched;              // 1: static round-robin zone assignment instead of the work queue (bz_set_schedule)
  const long long *order;        // nullptr, or the order in which the queue hands the zones out (bz_set_zone_order)
};

__device__ __forceinline__ double inv_small_int(int p) {  // 1.0/p, p = 1..7, correctly rounded
  switch (p) {
    case 1: return 1.0;
    case 2: return 1.0 / 2.0;
    case 3: return 1.0 / 3.0;
    case 4: return 1.0 / 4.0;
    case 5: return 1.0 / 5.0;
    case 6: return 1.0 / 6.0;
    default: return 1.0 / 7.0;
  }
}
__device__ __forceinline__ double factorial_(int p) {  // p = 0..7
  switch (p) {
    case 0: case 1: return 1.0;
    case 2: return 2.0;
    case 3: return 6.0;
    case 4: return 24.0;
    case 5: return 120.0;
    case 6: return 720.0;
    default: return 5040.0;
  }
}
// eta = 1 / ((bias*E)^(1/p) + ADDON), root through the own exp/log
__device__ __forceinline__ double eta_of(double E, double bias, int p) {
  const double v = bias * E;
  const double root = (v > 1e-300) ? exp_(log_(v) * inv_small_int(p)) : 0.0;
  return 1.0 / (root + ADDON);
}

// C.2-D, the decision proper, shared by both kernels: the next step-size ratio eta and the order action
// (-1 lower, 0 keep, +1 raise) from the three candidate etas.  order_due: the order may change at this
// step (nqwait reached 0); otherwise only eta_q counts.  Then THRESH and the growth cap.
__device__ __forceinline__ void select_eta(bool order_due, double etaq, double etaqm1, double etaqp1, double etamax,
                                           double &eta, int &action) {
  eta = etaq;
  action = 0;
  if (order_due) {
    if (etaq >= etaqp1) {
      if (!(etaq >= etaqm1)) {
        eta = etaqm1;
        action = -1;
      }
    } else if (etaqp1 > etaqm1) {
      eta = etaqp1;
      action = +1;
    } else {
      eta = etaqm1;
      action = -1;
    }
  }
  if (eta < THRESH) {
    eta = 1.0;
    action = 0;
  } else if (eta > etamax) {
    eta = etamax;
  }
}

// Row stride of a group's matrix M, in doubles: LANES + 1 (odd), so that the lanes of a group read one column,
// or walk their own rows in step, without bank conflicts beyond the two wavefronts of a 64-bit access.
// (Measured on config 5 and dropped: stride 34 with the rows walked by 128-bit accesses -- 3 instead of 6
// instructions per FMA of the LU update, same bits, 2 904 ms instead of 2 787 ms: what is read by columns,
// the pivot searches and the solves, then takes twice the wavefronts.)
__host__ __device__ constexpr int coop_ld(int lanes) { return lanes + 1; }
// per-group scratch, in doubles: M (LANES rows), urow (2 LANES), ysh, xs (LANES each), R, dRdT (K each), dRdY
// (3 K); M on a 16-byte boundary wherever it is placed (burn_coop_kernel places it)
__host__ __device__ constexpr int coop_per_group(int lanes, int K) { return lanes * coop_ld(lanes) + ((4 * lanes + 5 * K + 1) & ~1); }

template <int NEQ, int LANES>
struct CoopSmem {
  static constexpr int LD = coop_ld(LANES);
  __host__ __device__ static constexpr int per_group(int K) { return coop_per_group(LANES, K); }
};

}  // namespace bz
