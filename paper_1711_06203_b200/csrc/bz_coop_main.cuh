// bz_coop_main.cuh -- kernel entry: persistent blocks, work queue, BZ-BDF v1 driver as a flat
// state machine: one loop trip = one step attempt of the group's zone.  In the sub-warp instances ONE
// block barrier per trip keeps all warps of the block in the same part of the (large) loop body so that
// they share instruction-cache lines (profiles/README.md: unsynchronised warps stalled 8 cycles per issue
// on instruction fetch; still 713 against 555 ms for burn_coop<14,16> with the rolled LU); the
// warp-per-zone instances run without (see the loop).
#pragma once
#include "bz_coop_burn.cuh"

namespace bz {

constexpr int COOP_THREADS = 256;
// Threads per block of an instance.  The LU lives in the group's shared-memory matrix (LuSmem,
// bz_coop_burn.cuh), so a warp-per-zone lane carries no 31-entry row: 128 registers instead of 255, and one
// block holds 16 zones (16 warps) instead of 8.  Measured on config 5 (131 072-zone sample): rows in
// registers, 256 threads 3 447 ms; rows in shared memory, 256 threads 4 290 ms, 384 threads 3 415 ms, 512
// threads 3 258 ms.  net_create launches fewer threads when the tables of a large network leave no room for
// 16 groups.
template <int LANES>
struct CoopShape {
  static constexpr int THREADS = (LANES == 32) ? 512 : COOP_THREADS;
  static constexpr int MINB = (LANES == 32) ? 1 : 2;
};
// Blocks per SM: the warp-per-zone instances take one block of 16 warps (registers and shared memory both
// full).  The sub-warp instances fit 128 registers, and two blocks per SM (16 warps instead of 8) ran 9 %
// faster (config 3 on burn_coop<14,16>) -- when shared memory allows two blocks, which net_create asks the
// occupancy calculator.
// REUSE: the Newton-matrix policy of bz_set_policy(net, 1), a separate instantiation.  A
// group owns its zone's factors (in its matrix M, which only a fresh Jacobian overwrites) and nothing of them
// is shared across groups, so a group that keeps its matrix simply skips Jacobian and LU: no warp-level
// sharing as in the quad kernel.
template <int NEQ, int LANES, bool EXT, bool REUSE>
__global__ void __launch_bounds__(CoopShape<LANES>::THREADS, CoopShape<LANES>::MINB) burn_coop_kernel(DevNet net, BurnArgs A) {
  extern __shared__ __align__(16) double smem[];
  constexpr int LD = CoopSmem<NEQ, LANES>::LD;
  const int N = net.N, n = net.n, K = net.K;

  // ---- block prologue: network tables -> shared memory ---------------------------------------
  double *s_dbl = smem;
  int *s_int = reinterpret_cast<int *>(smem + ((net.ndbl + 1) & ~1));
  for (int i = threadIdx.x; i < net.ndbl; i += blockDim.x) s_dbl[i] = net.dbl[i];
  for (int i = threadIdx.x; i < net.nint; i += blockDim.x) s_int[i] = net.itab[i];
  __syncthreads();

  Group<NEQ, LANES, EXT> g;
  g.lig = threadIdx.x & (LANES - 1);
  g.gmask = (LANES == 32) ? 0xffffffffu : (((1u << (LANES & 31)) - 1u) << ((threadIdx.x & 31) & ~(LANES - 1)));
  g.N = N; g.n = n; g.K = K; g.fac = net.fac;
  g.inv_n = 1.0 / (double)n;
  g.lnA = s_dbl; g.en = s_dbl + K; g.B = s_dbl + 2 * K; g.Q = s_dbl + 3 * K; g.invsym = s_dbl + 4 * K;
  g.aion = s_dbl + 5 * K; g.sp_dy = s_dbl + 5 * K + N;
  g.rexp = (EXT && net.has_rexp) ? s_dbl + 5 * K + N + net.nterm : nullptr;
  g.zp1 = (EXT && net.eos) ? s_dbl + 5 * K + N + net.nterm + (net.has_rexp ? K : 0) : nullptr;
  g.eos_extra = net.eos_extra;
  g.rp = s_int; g.sp_off = s_int + 4 * K; g.sp_k = g.sp_off + (N + 1);
  g.cl_off = g.sp_k + net.nterm; g.cl_ks = g.cl_off + (N + 1);
  {
    const int tab = ((net.ndbl + 1) & ~1) + ((net.nint + 3) & ~3) / 2;  // doubles, 16-byte aligned
    const int pg = CoopSmem<NEQ, LANES>::per_group(K);
    const int pga = (pg + 1) & ~1;
    double *base = smem + tab + (threadIdx.x / LANES) * pga;
    // M first for the sub-warp instances, last for the warp-per-zone ones: measured, the same kernel apart from
    // address arithmetic (burn_coop<14,16> on config 3: 765 ms with M last, 741 ms with M first;
    // burn_coop<31,32> on config 5: 2 777 ms with M last, 2 945 ms with M first)
    constexpr int MSIZE = LANES * LD;  // even
    const int rest = (4 * LANES + 5 * K + 1) & ~1;
    g.M = (LANES == 32) ? base + rest : base;
    g.urow = (LANES == 32) ? base : base + MSIZE;  // 2*LANES, 16-byte aligned
    g.ysh = g.urow + 2 * LANES;
    g.xs = g.ysh + LANES;
    g.R = g.xs + LANES;
    g.dRdT = g.R + K;
    g.dRdY = g.dRdT + K;
  }
  g.has_src = (A.src_T != nullptr);
  g.src = 0.0;
  const int lig = g.lig;
  const bool act = lig < n;      // lanes that own a component
  const double dt = A.dt, rtol = A.rtol, atol = A.atol;
  unsigned long long c_nst = 0, c_rhs = 0, c_jac = 0, c_lu = 0, c_sol = 0, c_etf = 0, c_cfn = 0, c_fail = 0;

  LuSmem<NEQ, LANES> lu;  // the factors live in g.M; the lane keeps its row's position and 1/pivot

  // per-zone integrator state, persistent across loop trips (registers; uniform within the group
  // except the per-component Z, w, S)
  int phase = 0;  // 0 need a zone, 1 stepping, 2 queue empty
  long long z = 0;
  double rho = 0.0, ai = 1.0;
  double Z[QMAX + 1], w = 0.0, S = 0.0;
  double h = 0.0, t = 0.0, etamax = ETAMX1, hS = 0.0;
  int q = 1, nqwait = 2, qS = 0, nst = 0, ntau = 0, ncf = 0, nef = 0;
  bool newstep = true, last = false;
  // REUSE: gamma_P and the step count of the kept factorisation; a factorisation exists; a failure asked for a fresh one
  double gamP = 0.0;
  int nslp = 0;
  bool haveP = false, forceP = false;
  double tau[QMAX + 1];
#pragma unroll
  for (int i = 0; i <= QMAX; i++) tau[i] = 0.0, Z[i] = 0.0;

  bool started = false;
  for (;;) {
    if (phase == 0) {
      // ---- a2: fetch the next zone from the work queue -------------------------------------------
      // (bz_set_schedule(1) switches a2 off for the before/after measurement: group g then burns zones
      // g, g + G, g + 2G, ... with G = groups of the grid; results are the same, only the balance differs)
      if (A.static_sched) {
        const long long G = (long long)gridDim.x * (blockDim.x / LANES);
        z = started ? z + G : (long long)blockIdx.x * (blockDim.x / LANES) + threadIdx.x / LANES;
        started = true;
      } else {
        if (lig == 0) {
          z = (long long)atomicAdd(A.queue, 1ull);
          if (A.order != nullptr && z < A.nz) {  // bz_set_zone_order: the q-th zone handed out is order[q]
            z = A.order[z];
            if ((unsigned long long)z >= (unsigned long long)A.nz) z = -1;  // not a zone: ignored
          }
        }
        z = __shfl_sync(g.gmask, z, 0, LANES);
      }
      if (z >= A.nz) {
        phase = 2;
      } else if (z >= 0) {
        // ---- a1: load zone state -----------------------------------------------------------------
        rho = A.rho[z];
        double xin = 0.0;
        ai = 1.0;
        if (lig >= 1 && lig <= N) {  // internal order: lane 0 = T, lane i + 1 = species i
          xin = A.X[(long long)(lig - 1) * A.ld + z];
          ai = g.aion[lig - 1];
        } else if (lig == 0) {
          xin = A.T[z];
        }
        const double y0 = (lig >= 1 && lig <= N) ? xin / ai : xin;
        if (g.has_src) {
          g.src = 0.0;
          if (lig >= 1 && lig <= N) g.src = A.src_X[(long long)(lig - 1) * A.ld + z] / ai;
          else if (lig == 0) g.src = A.src_T[z];
        }
        const bool bad = !(rho > 0.0) || !finite_(rho) || (act && !finite_(y0)) || (lig == 0 && !(y0 > 0.0)) ||
                         (g.has_src && !finite_(g.src));
        if (g.gany(bad)) {  // invalid input zone: outputs = inputs; stay in phase 0
          if (lig >= 1 && lig <= N) {
            A.X_out[(long long)(lig - 1) * A.ld + z] = xin;
          } else if (lig == 0) {
            A.T_out[z] = xin;
            A.nsteps[z] = -4;
          }
          c_fail++;
        } else {
          // ---- Init ---------------------------------------------------------------------------------
#pragma unroll
          for (int j = 0; j <= QMAX; j++) Z[j] = 0.0;
          const double f = g.template rates<true>(rho, y0);
          c_rhs++, c_jac++;
          w = act ? 1.0 / fma_(rtol, fabs(y0), atol) : 0.0;
          {
            g.sync();
            if (act) g.ysh[lig] = f;
            g.sync();
            double s = 0.0;
            if (act)
              for (int j = 0; j < n; j++) s = fma_(g.M[lig * LD + j], g.ysh[j], s);
            const double d2 = g.wrms(s, w);
            h = dt;
            if (d2 > 0.0) {
              const double hh = 0.5 * sqrt(2.0 / d2);
              if (hh < dt) h = hh;
            }
          }
          Z[0] = y0;
          Z[1] = h * f;
          q = 1, nqwait = 2, qS = 0, nst = 0, ntau = 0;
          t = 0.0, etamax = ETAMX1, hS = 0.0, S = 0.0;
          if (REUSE) gamP = 0.0, nslp = 0, haveP = false, forceP = false;
#pragma unroll
          for (int i = 0; i <= QMAX; i++) tau[i] = 0.0;
          newstep = true;
          phase = 1;
        }
      }
    }
    // Sub-warp instances: one block barrier per trip (instruction cache, see the head of this file).  The
    // warp-per-zone instances run free of each other: with the rolled in-place LU the hot part of a trip is
    // ~70 KB of code and lockstep costs more than it saves (config 5 sample: 3 258 -> 2 883 ms; instruction-fetch
    // stalls 10 % of the samples), and a warp leaves when the queue is empty (phase is warp-uniform there, and
    // nothing else in the loop is block-wide).
    if (LANES == 32) {
      if (phase == 2) break;
    } else if (__syncthreads_and(phase == 2)) break;
    if (phase == 1) {
#include "bz_coop_attempt.inc"
    }
  }
  // ---- counters: one atomic per group and counter --------------------------------------------
  if (lig == 0) {
    atomicAdd(A.counters + 0, c_nst);
    atomicAdd(A.counters + 1, c_rhs);
    atomicAdd(A.counters + 2, c_jac);
    atomicAdd(A.counters + 3, c_lu);
    atomicAdd(A.counters + 4, c_sol);
    atomicAdd(A.counters + 5, c_etf);
    atomicAdd(A.counters + 6, c_cfn);
    atomicAdd(A.counters + 7, c_fail);
  }
}

}  // namespace bz
