// bz_quad_main.cuh -- quad kernel entry: work queue + BZ-BDF v1 driver, one loop trip = one
// step attempt of the quad's zone (flat state machine, see bz_quad.cuh for the mapping).
#pragma once
#include "bz_quad.cuh"

namespace bz {

// BLOCK threads = BLOCK/4 zones per block; MINB blocks per SM (register budget 65536/(BLOCK*MINB)).
// All warps of a block meet at ONE barrier per loop trip (= per step attempt): that keeps them in
// the same part of the ~100 KB loop body, so instruction-cache lines fetched by one warp are reused
// by the others (unsynchronised warps thrashed the instruction cache: profiles/README.md).
// REUSE: the Newton-matrix policy of bz_set_policy(net, 1) (a separate instantiation: the default kernel
// is compiled without any of it).
template <class Net, int BLOCK, int MINB, bool REUSE>
__global__ void __launch_bounds__(BLOCK, MINB) burn_quad_kernel(QuadNet qn, BurnArgs A) {
  constexpr int QUAD_THREADS = BLOCK;  // (a run-time block size was tried for small batches: it perturbed the
                                       // register allocation of the alpha13 instance, config 3 +3 %)
  constexpr int NEQ = Net::NEQ, N = Net::N, K = Net::K, S = Net::S;
  typedef QuadMem<NEQ, K> Mem;
  extern __shared__ __align__(16) double smem[];
  double *coef = smem;  // lnA n B Q [4K] + aion [N]
  for (int i = threadIdx.x; i < 4 * K + N; i += QUAD_THREADS) coef[i] = qn.coef[i];
  __syncthreads();
  const double *aion = coef + 4 * K;
  const int c = threadIdx.x & 3;
  const unsigned gmask = 0xfu << ((threadIdx.x & 31) & ~3);
  Mem m;
  m.base = smem + ((4 * K + N + 1) & ~1) + (threadIdx.x >> 2) * Mem::SIZE;
  const long long gquad = (long long)blockIdx.x * (QUAD_THREADS / 4) + (threadIdx.x >> 2);
  double *gP = qn.gscratch + gquad * (NEQ * NEQ + 2 * NEQ);  // general path: P, b, ipvt
  const double dt = A.dt, rtol = A.rtol, atol = A.atol, fac = qn.fac;
  const double inv_n = 1.0 / (double)NEQ;
  const bool has_src = (A.src_T != nullptr);  // burn_zones_src: f <- f + s after every rate evaluation
  // (each lane adds the sources of its own components; they sit in the zone's shared memory)
#define BZQ_ADD_SRC(fv)                                         \
  do {                                                          \
    if (has_src) {                                              \
      _Pragma("unroll") for (int s_ = 0; s_ < S; s_++)          \
        if (BZQ_OK(s_)) fv[s_] = fv[s_] + m.src(BZQ_I(s_));     \
    }                                                           \
  } while (0)
  // event counters live in the quad's shared memory (lane 0 counts): registers are the scarce
  // resource of this kernel.  nrhs = nlu + ninit + xrhs and njac = nlu + ninit are derived at the end.
#define BZQ_COUNT(k) do { if (c == 0) m.cnt(Mem::k) += 1ull; } while (0)
  if (c == 0) {
#pragma unroll
    for (int k = 0; k < 8; k++) m.cnt(k) = 0ull;
    m.zid() = gquad - (long long)gridDim.x * (QUAD_THREADS / 4);  // static schedule: first zone = gquad
  }

  // component index of my slot s and its validity
#define BZQ_I(s) (4 * (s) + c)
#define BZQ_OK(s) (4 * (s) + c < NEQ)

  auto qsum = [&](double v) {  // quad butterfly, strides 2 then 1 (norm_lanes = 4)
    v = v + __shfl_xor_sync(gmask, v, 2, 4);
    v = v + __shfl_xor_sync(gmask, v, 1, 4);
    return v;
  };
  auto wrms = [&](const double (&v)[S]) {
    double p = 0.0;
#pragma unroll
    for (int s = 0; s < S; s++)
      if (BZQ_OK(s)) {
        const double d = v[s] * m.W(BZQ_I(s));
        p = fma_(d, d, p);
      }
    return sqrt(qsum(p) * inv_n);
  };
  auto qany = [&](bool p) { return (__ballot_sync(gmask, p) & gmask) != 0u; };
  // full-warp versions for the warp-uniform part of an attempt (constant mask: no mask matching)
  constexpr unsigned FULLMASK = 0xffffffffu;
  auto qanyw = [&](bool p) { return (__ballot_sync(FULLMASK, p) & gmask) != 0u; };
  auto wrmsw = [&](const double (&v)[S]) {
    double p = 0.0;
#pragma unroll
    for (int s = 0; s < S; s++)
      if (BZQ_OK(s)) {
        const double d = v[s] * m.W(BZQ_I(s));
        p = fma_(d, d, p);
      }
    p = p + __shfl_xor_sync(FULLMASK, p, 2, 4);
    p = p + __shfl_xor_sync(FULLMASK, p, 1, 4);
    return sqrt(p * inv_n);
  };

  int phase = 0;  // 0 need a zone, 1 stepping, 2 queue empty, 3 zone loaded: initial rates pending
  double rho = 0.0, h = 0.0;
  int q = 1, nqwait = 2, nst = 0, ncf = 0, nef = 0;
  // t, etamax, h_S, q_S, ntau and the zone index live in the zone's shared memory (bz_quad.cuh)
#define BZQ_T m.sc(Mem::SC_T)
#define BZQ_ETAMAX m.sc(Mem::SC_ETAMAX)
#define BZQ_HSAV m.sc(Mem::SC_HSAV)
#define BZQ_QS m.isc(0)
#define BZQ_NTAU m.isc(1)
  bool newstep = true, last = false;
  QuadLU<NEQ> lu;

  for (unsigned trip = 0;; trip++) {
    // zone starts: few per warp and trip while zones take hundreds of steps (config 3), all eight
    // quads every trip where zones take one step (config 4).  Every thread votes here.
    const bool bulk = __popc(__ballot_sync(0xffffffffu, phase == 0)) >= 8;  // two quads or more
    if (phase == 0) {
      // ---- a2 + a1: next zone, load, validate, initialise ------------------------------------------
      // (bz_set_schedule(1) switches the queue off for the before/after measurement of a2: quad g then
      // burns zones g, g + G, g + 2G, ... with G = quads of the grid; same results, different balance)
      long long z = 0;
      if (c == 0) {
        z = A.static_sched ? m.zid() + (long long)gridDim.x * (QUAD_THREADS / 4) : (long long)atomicAdd(A.queue, 1ull);
        if (A.order != nullptr && z < A.nz) {  // bz_set_zone_order: the q-th zone handed out is order[q]
          z = A.order[z];
          if ((unsigned long long)z >= (unsigned long long)A.nz) z = -1;  // not a zone: ignored
        }
      }
      z = __shfl_sync(gmask, z, 0, 4);
      m.zid() = z;
      if (z >= A.nz) {
        phase = 2;
      } else if (z >= 0) {
        rho = A.rho[z];
        double xin[S], y[S];
        bool bad = !(rho > 0.0) || !finite_(rho);
#pragma unroll
        for (int s = 0; s < S; s++) {
          const int i = BZQ_I(s);
          xin[s] = 0.0;
          y[s] = 0.0;
          if (i == 0) {
            xin[s] = A.T[z];
            y[s] = xin[s];
            bad |= !(y[s] > 0.0) || !finite_(y[s]);
          } else if (i < NEQ) {
            xin[s] = A.X[(long long)(i - 1) * A.ld + z];
            y[s] = xin[s] / aion[i - 1];
            bad |= !finite_(y[s]);
          }
          if (has_src && i < NEQ) {
            const double sv = (i == 0) ? A.src_T[z] : A.src_X[(long long)(i - 1) * A.ld + z] / aion[i - 1];
            m.src(i) = sv;  // own component only: no intra-quad hazard
            bad |= !finite_(sv);
          }
        }
        if (qany(bad)) {  // invalid input zone: outputs = inputs, stay in phase 0
#pragma unroll
          for (int s = 0; s < S; s++) {
            const int i = BZQ_I(s);
            if (i == 0) {
              A.T_out[z] = xin[s];
              A.nsteps[z] = -4;
            } else if (i < NEQ)
              A.X_out[(long long)(i - 1) * A.ld + z] = xin[s];
          }
          BZQ_COUNT(CN_FAIL);
        } else {
          if (bulk) {
            // several quads of the warp start a zone in this trip: initialise here and now, so that a
            // one-step zone (the cold regions of config 4) costs one trip
            double f[S], v[S];
            __syncwarp(gmask);
#pragma unroll
            for (int s = 0; s < S; s++)
              if (BZQ_OK(s)) {
                m.ysh()[BZQ_I(s)] = y[s];
                m.W(BZQ_I(s)) = 1.0 / fma_(rtol, fabs(y[s]), atol);
                m.Z(0, BZQ_I(s)) = y[s];
              }
            __syncwarp(gmask);
            Net::template eval_quad<true, true>(coef, fac, rho, m.ysh(), m.lam(), c, gmask, 0.0, 0.0, true, f, lu.a);
            BZQ_ADD_SRC(f);
            BZQ_COUNT(CN_INIT);
            // exact second derivative y'' = J f for the first step size
            __syncwarp(gmask);
#pragma unroll
            for (int s = 0; s < S; s++)
              if (BZQ_OK(s)) m.ysh()[BZQ_I(s)] = f[s];
            __syncwarp(gmask);
#pragma unroll
            for (int s = 0; s < S; s++) {
              double acc = 0.0;
#pragma unroll
              for (int j = 0; j < NEQ; j++) acc = fma_(lu.a[s][j], m.ysh()[j], acc);
              v[s] = acc;
            }
            const double d2 = wrms(v);
            h = dt;
            if (d2 > 0.0) {
              const double hh = 0.5 * sqrt(2.0 / d2);
              if (hh < dt) h = hh;
            }
#pragma unroll
            for (int s = 0; s < S; s++)
              if (BZQ_OK(s)) m.Z(1, BZQ_I(s)) = h * f[s];
            q = 1, nqwait = 2, nst = 0;
            BZQ_QS = 0, BZQ_NTAU = 0;
            BZQ_T = 0.0, BZQ_ETAMAX = ETAMX1, BZQ_HSAV = 0.0;
            if (REUSE) m.pint(0) = 0, m.pint(1) = 0, m.sc(Mem::SC_GAMP) = 0.0;
            if (c == 0) {
#pragma unroll
              for (int i = 0; i <= QMAX; i++) m.sc(Mem::SC_TAU + i) = 0.0;
            }
            newstep = true;
            phase = 1;
          } else {
            // publish y0; the first rate evaluation (f0, J0) rides along with the warp-uniform attempt
            // of this trip (phase 3, bz_quad_attempt.inc), stepping starts with the next trip
            __syncwarp(gmask);
#pragma unroll
            for (int s = 0; s < S; s++)
              if (BZQ_OK(s)) {
                m.ysh()[BZQ_I(s)] = y[s];
                m.W(BZQ_I(s)) = 1.0 / fma_(rtol, fabs(y[s]), atol);
                m.Z(0, BZQ_I(s)) = y[s];
              }
            q = 1, nqwait = 2, nst = 0;
            BZQ_QS = 0, BZQ_NTAU = 0;
            BZQ_T = 0.0, BZQ_ETAMAX = ETAMX1, BZQ_HSAV = 0.0;
            if (REUSE) m.pint(0) = 0, m.pint(1) = 0, m.sc(Mem::SC_GAMP) = 0.0;
            if (c == 0) {
#pragma unroll
              for (int i = 0; i <= QMAX; i++) m.sc(Mem::SC_TAU + i) = 0.0;
            }
            phase = 3;
          }
        }
      }
    }
    if (__syncthreads_and(phase == 2)) break;
#include "bz_quad_attempt.inc"
  }
#undef BZQ_I
#undef BZQ_OK
  // ---- counters (lane 0 of each quad holds the zone's counts) ------------------------------------
#undef BZQ_COUNT
#undef BZQ_ADD_SRC
#undef BZQ_T
#undef BZQ_ETAMAX
#undef BZQ_HSAV
#undef BZQ_QS
#undef BZQ_NTAU
  unsigned long long cs[8];
  {
    const unsigned long long lu_ = m.cnt(Mem::CN_LU), in_ = m.cnt(Mem::CN_INIT);
    cs[0] = m.cnt(Mem::CN_NST), cs[1] = lu_ + in_ + m.cnt(Mem::CN_XRHS), cs[2] = lu_ + in_, cs[3] = lu_;
    cs[4] = m.cnt(Mem::CN_SOL), cs[5] = m.cnt(Mem::CN_ETF), cs[6] = m.cnt(Mem::CN_CFN), cs[7] = m.cnt(Mem::CN_FAIL);
  }
#pragma unroll
  for (int k = 0; k < 8; k++) {
    unsigned long long v = (c == 0) ? cs[k] : 0ull;
#pragma unroll
    for (int s = 16; s >= 1; s >>= 1) v += __shfl_xor_sync(0xffffffffu, v, s);
    if ((threadIdx.x & 31) == 0) atomicAdd(A.counters + k, v);
  }
}

}  // namespace bz
