// bz_tpz_main.cuh -- thread-per-zone kernel entry: work queue + BZ-BDF v1 driver as a flat
// per-lane state machine (one loop trip = one step ATTEMPT, so lanes never wait for a
// neighbour's zone to finish; see bz_tpz.cuh for the data layout).
#pragma once
#include "bz_tpz.cuh"

namespace bz {

template <class Net, int BLOCK, int W>
__global__ void __launch_bounds__(BLOCK) burn_tpz_kernel(TpzNet tn, BurnArgs A, double *__restrict__ Sg) {
  constexpr int NEQ = Net::NEQ, N = Net::N, K = Net::K;
  extern __shared__ __align__(16) double smem[];
  double *coef = smem;  // lnA n B Q [4K] + aion [N]
  for (int i = threadIdx.x; i < 4 * K + N; i += BLOCK) coef[i] = tn.coef[i];
  __syncthreads();
  const double *aion = coef + 4 * K;
  TpzMem<NEQ, BLOCK> m;
  m.base = smem + ((4 * K + N + 1) & ~1) + threadIdx.x;
  const long long nthreads = (long long)gridDim.x * BLOCK;
  double *Sme = Sg + (long long)blockIdx.x * BLOCK + threadIdx.x;  // S_i at Sme[i * nthreads]
  const double dt = A.dt, rtol = A.rtol, atol = A.atol, fac = tn.fac;
  const double inv_n = 1.0 / (double)NEQ;
  unsigned long long c_nst = 0, c_rhs = 0, c_jac = 0, c_lu = 0, c_sol = 0, c_etf = 0, c_cfn = 0, c_fail = 0;

  // per-zone integrator state
  int phase = 0;  // 0 need a zone, 1 stepping, 2 queue empty
  long long z = 0;
  double rho = 0.0, h = 0.0, t = 0.0, etamax = ETAMX1, hS = 0.0;
  int q = 1, nqwait = 2, qS = 0, nst = 0, ntau = 0, ncf = 0, nef = 0;
  bool newstep = true, last = false;
  double tau[QMAX + 1];
#pragma unroll
  for (int i = 0; i <= QMAX; i++) tau[i] = 0.0;

  for (;;) {
    if (phase == 0) {
      // ---- a2 + a1: next zone from the queue, load, validate, initialise --------------------
      z = (long long)atomicAdd(A.queue, 1ull);
      if (z >= A.nz) {
        phase = 2;
      } else {
        rho = A.rho[z];
        double y[NEQ], f[NEQ], s2[NEQ];
        y[0] = A.T[z];
        bool bad = !(rho > 0.0) || !finite_(rho) || !(y[0] > 0.0) || !finite_(y[0]);
#pragma unroll
        for (int i = 0; i < N; i++) {
          y[i + 1] = A.X[(long long)i * A.nz + z] / aion[i];
          bad |= !finite_(y[i + 1]);
        }
        if (bad) {  // invalid input zone: outputs = inputs, stay in phase 0
          A.T_out[z] = A.T[z];
#pragma unroll
          for (int i = 0; i < N; i++) A.X_out[(long long)i * A.nz + z] = A.X[(long long)i * A.nz + z];
          A.nsteps[z] = -4;
          c_fail++;
        } else {
#pragma unroll
          for (int i = 0; i < NEQ; i++) s2[i] = 0.0;
          JfStore<NEQ> js(f, s2);
          Net::template eval<true>(coef, fac, rho, y, f, js);
          c_rhs++, c_jac++;
#pragma unroll
          for (int i = 0; i < NEQ; i++) m.W(i) = 1.0 / fma_(rtol, fabs(y[i]), atol);
          const double d2 = wrms4<NEQ, BLOCK>(s2, m, inv_n);
          h = dt;
          if (d2 > 0.0) {
            const double hh = 0.5 * sqrt(2.0 / d2);
            if (hh < dt) h = hh;
          }
#pragma unroll
          for (int i = 0; i < NEQ; i++) {
            m.Z(0, i) = y[i];
            m.Z(1, i) = h * f[i];
          }
          q = 1, nqwait = 2, qS = 0, nst = 0, ntau = 0;
          t = 0.0, etamax = ETAMX1, hS = 0.0;
#pragma unroll
          for (int i = 0; i <= QMAX; i++) tau[i] = 0.0;
          newstep = true;
          phase = 1;
        }
      }
    }
    // one block barrier per trip keeps the block's warps in the same part of the (large) loop body,
    // so they share instruction-cache lines (profiles/README.md)
    if (__syncthreads_and(phase == 2)) break;
    if (phase != 1) continue;

    // ================= one step attempt (C.2-A/B) =============================================
    if (newstep) {
      const double rem = dt - t;
      if (h >= rem || rem - h < SLIVER * h) {
        const double eta = rem / h;
        double r = eta;
        for (int j = 1; j <= q; j++) {
#pragma unroll
          for (int i = 0; i < NEQ; i++) m.Z(j, i) = m.Z(j, i) * r;
          r = r * eta;
        }
        h = rem;
        last = true;
      } else
        last = false;
      ncf = nef = 0;
      newstep = false;
    }
    // B.1 coefficients
    double l[QMAX + 2], hs[QMAX + 1], rxi[QMAX + 1];
    l[0] = 1.0;
#pragma unroll
    for (int j = 1; j <= QMAX + 1; j++) l[j] = 0.0;
#pragma unroll
    for (int i = 0; i <= QMAX; i++) hs[i] = 0.0, rxi[i] = 0.0;
    {
      double s = h;
#pragma unroll
      for (int i = 1; i <= QMAX; i++) {
        if (i <= q) {
          if (i > 1) s = s + tau[i - 1];
          hs[i] = s;
          const double r = h / s;
          rxi[i] = r;
#pragma unroll
          for (int j = QMAX; j >= 1; j--)
            if (j <= i) l[j] = fma_(l[j - 1], r, l[j]);
        }
      }
    }
    const double l1 = l[1];
    const double gamma = h / l1;
    const double rl1 = 1.0 / l1;
    const double cerr = (double)(q + 1) * l1;
    // B.2 predict (Pascal triangle in place), component by component
    double acor[NEQ];
    bool inval = false;
#pragma unroll
    for (int i = 0; i < NEQ; i++) {
      double zc[QMAX + 1];
#pragma unroll
      for (int j = 0; j <= QMAX; j++) zc[j] = (j <= q) ? m.Z(j, i) : 0.0;
      nord_predict(zc, q);
#pragma unroll
      for (int j = 0; j <= QMAX; j++)
        if (j <= q) m.Z(j, i) = zc[j];
      inval |= !finite_(zc[0]);
      if (i == 0) inval |= !(zc[0] > 0.0);
      acor[i] = 0.0;
    }
    bool ok = false, slow = false;
    int ipvt[NEQ];
    double dsm = 0.0;
    if (!inval) {
      // B.3 rates + Jacobian + LU (general path only if an interchange is needed)
      double b[NEQ];
      bool fok = true;
#pragma unroll 1
      for (int pass = 0; pass < 2; pass++) {
        double y[NEQ], f[NEQ];
#pragma unroll
        for (int i = 0; i < NEQ; i++) y[i] = m.Z(0, i);
        if (pass == 1) {
          for (int i = 0; i < NEQ; i++)
            for (int j = 0; j < NEQ; j++) m.P(i, j) = (i == j) ? 1.0 : 0.0;
        }
        NewtonStore<NEQ, BLOCK> ps{m, gamma};
        Net::template eval<true>(coef, fac, rho, y, f, ps);
#pragma unroll
        for (int i = 0; i < NEQ; i++) b[i] = fma_(gamma, f[i], -fma_(m.Z(1, i), rl1, 0.0));
        if (pass == 0) {
          c_rhs++, c_jac++, c_lu++;
          const unsigned fl = lu_panels<Net, BLOCK, W>(m, b);
          if (!(fl & 1u)) {
            fok = !(fl & 2u);
            if (fok) back_subst<NEQ, BLOCK>(m, b);
            break;
          }
        } else {
          slow = true;
          fok = lu_general<NEQ, BLOCK>(m, ipvt);
          if (fok) {
            double bl[NEQ];
            for (int i = 0; i < NEQ; i++) bl[i] = b[i];
            solve_general<NEQ, BLOCK>(m, ipvt, bl);
            for (int i = 0; i < NEQ; i++) b[i] = bl[i];
          }
        }
      }
      if (fok) {  // B.4 Newton (b holds the first correction)
        double crate = 1.0, delp = 0.0;
        const double tq = NTOL * cerr;
#pragma unroll 1
        for (int mi = 0; mi < MAXCOR; mi++) {
          if (mi > 0) {
            double y[NEQ], f[NEQ];
            bool iv = false;
#pragma unroll
            for (int i = 0; i < NEQ; i++) {
              y[i] = m.Z(0, i) + acor[i];
              iv |= !finite_(y[i]);
            }
            iv |= !(y[0] > 0.0);
            if (iv) break;
            NoStore ns;
            Net::template eval<false>(coef, fac, rho, y, f, ns);
            c_rhs++;
#pragma unroll
            for (int i = 0; i < NEQ; i++) b[i] = fma_(gamma, f[i], -fma_(m.Z(1, i), rl1, acor[i]));
            if (!slow) {
              fwd_subst<NEQ, BLOCK>(m, b);
              back_subst<NEQ, BLOCK>(m, b);
            } else {
              double bl[NEQ];
              for (int i = 0; i < NEQ; i++) bl[i] = b[i];
              solve_general<NEQ, BLOCK>(m, ipvt, bl);
              for (int i = 0; i < NEQ; i++) b[i] = bl[i];
            }
          }
          c_sol++;
#pragma unroll
          for (int i = 0; i < NEQ; i++) acor[i] = acor[i] + b[i];
          const double del = wrms4<NEQ, BLOCK>(b, m, inv_n);
          if (!finite_(del)) break;
          if (mi > 0) {
            const double rr = del / delp;
            crate = CRDOWN * crate;
            if (rr > crate) crate = rr;
          }
          const double dcon = (del * (crate < 1.0 ? crate : 1.0)) / tq;
          if (dcon <= 1.0) {
            ok = true;
            break;
          }
          if (mi > 0 && del > RDIV * delp) break;
          delp = del;
        }
      }
    }
    int code = 0;  // set when the zone ends (nsteps value)
    bool accepted = false;
    if (!ok) {
      // B.6 Newton failure: retract, quarter the step
      ncf++, c_cfn++;
      etamax = 1.0;
      last = false;
      const bool give_up = ncf > MXNCF;
      double r = ETACF;
#pragma unroll
      for (int i = 0; i < NEQ; i++) {
        double zc[QMAX + 1];
#pragma unroll
        for (int j = 0; j <= QMAX; j++) zc[j] = (j <= q) ? m.Z(j, i) : 0.0;
        nord_retract(zc, q);
        if (!give_up) nord_rescale(zc, q, ETACF);
#pragma unroll
        for (int j = 0; j <= QMAX; j++)
          if (j <= q) m.Z(j, i) = zc[j];
      }
      (void)r;
      if (give_up) code = -1;
      else h = h * ETACF;
    } else {
      dsm = wrms4<NEQ, BLOCK>(acor, m, inv_n) / cerr;
      if (dsm <= 1.0) {
        accepted = true;
      } else {
        // B.5 error-test failure
        nef++, c_etf++;
        etamax = 1.0;
        last = false;
#pragma unroll
        for (int i = 0; i < NEQ; i++) {
          double zc[QMAX + 1];
#pragma unroll
          for (int j = 0; j <= QMAX; j++) zc[j] = (j <= q) ? m.Z(j, i) : 0.0;
          nord_retract(zc, q);
#pragma unroll
          for (int j = 0; j <= QMAX; j++)
            if (j <= q) m.Z(j, i) = zc[j];
        }
        if (nef == MXNEF) {
          code = -2;
        } else if (nef <= 2) {
          double eta = eta_of(dsm, BIAS2, q + 1);
          if (eta < ETAMIN) eta = ETAMIN;
          if (nef == 2 && eta > ETAMXF) eta = ETAMXF;
          double r = eta;
          for (int j = 1; j <= q; j++) {
#pragma unroll
            for (int i = 0; i < NEQ; i++) m.Z(j, i) = m.Z(j, i) * r;
            r = r * eta;
          }
          h = h * eta;
        } else if (q > 1) {
          double xi[QMAX + 1], d[8];
#pragma unroll
          for (int i = 0; i <= QMAX; i++) xi[i] = 0.0;
          double s = 0.0;
#pragma unroll
          for (int i = 1; i <= QMAX - 2; i++) {
            if (i <= q - 2) {
              s = (i == 1) ? tau[1] : s + tau[i];
              xi[i] = s / h;
            }
          }
          build_d(q - 2, xi, d);
#pragma unroll
          for (int i = 0; i < NEQ; i++) {
            const double zq = m.Z(q, i);
#pragma unroll
            for (int j = 2; j <= QMAX - 1; j++)
              if (j <= q - 1) m.Z(j, i) = fma_(-d[j], zq, m.Z(j, i));
          }
          q = q - 1;
          nqwait = q + 1;
          double r = ETAMIN;
          for (int j = 1; j <= q; j++) {
#pragma unroll
            for (int i = 0; i < NEQ; i++) m.Z(j, i) = m.Z(j, i) * r;
            r = r * ETAMIN;
          }
          h = h * ETAMIN;
        } else {
          h = h * ETAMIN;
          double y[NEQ], f[NEQ];
#pragma unroll
          for (int i = 0; i < NEQ; i++) y[i] = m.Z(0, i);
          NoStore ns;
          Net::template eval<false>(coef, fac, rho, y, f, ns);
          c_rhs++;
#pragma unroll
          for (int i = 0; i < NEQ; i++) m.Z(1, i) = h * f[i];
          nqwait = 10;
        }
      }
    }
#include "bz_tpz_accept.inc"
  }
  // ---- counters: warp-reduce, one atomic per warp and counter ------------------------------------
  unsigned long long cs[8] = {c_nst, c_rhs, c_jac, c_lu, c_sol, c_etf, c_cfn, c_fail};
#pragma unroll
  for (int c = 0; c < 8; c++) {
    unsigned long long v = cs[c];
#pragma unroll
    for (int s = 16; s >= 1; s >>= 1) v += __shfl_xor_sync(0xffffffffu, v, s);
    if ((threadIdx.x & 31) == 0) atomicAdd(A.counters + c, v);
  }
}

}  // namespace bz
