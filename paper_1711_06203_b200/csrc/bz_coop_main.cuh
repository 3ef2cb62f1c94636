// bz_coop_main.cuh -- kernel entry: persistent blocks, work queue, BZ-BDF v1 driver.
#pragma once
#include "bz_coop_burn.cuh"

namespace bz {

constexpr int COOP_THREADS = 128;

template <int NEQ, int LANES>
__global__ void __launch_bounds__(COOP_THREADS) burn_coop_kernel(DevNet net, BurnArgs A) {
  extern __shared__ __align__(16) double smem[];
  constexpr int LD = LANES + 1;
  const int N = net.N, n = net.n, K = net.K;

  // ---- block prologue: network tables -> shared memory ---------------------------------------
  double *s_dbl = smem;
  int *s_int = reinterpret_cast<int *>(smem + ((net.ndbl + 1) & ~1));
  for (int i = threadIdx.x; i < net.ndbl; i += blockDim.x) s_dbl[i] = net.dbl[i];
  for (int i = threadIdx.x; i < net.nint; i += blockDim.x) s_int[i] = net.itab[i];
  __syncthreads();

  Group<NEQ, LANES> g;
  g.lig = threadIdx.x & (LANES - 1);
  g.gmask = (LANES == 32) ? 0xffffffffu : (((1u << (LANES & 31)) - 1u) << ((threadIdx.x & 31) & ~(LANES - 1)));
  g.N = N; g.n = n; g.K = K; g.fac = net.fac;
  g.inv_n = 1.0 / (double)n;
  g.lnA = s_dbl; g.en = s_dbl + K; g.B = s_dbl + 2 * K; g.Q = s_dbl + 3 * K; g.invsym = s_dbl + 4 * K;
  g.aion = s_dbl + 5 * K; g.sp_dy = s_dbl + 5 * K + N;
  g.rp = s_int; g.sp_off = s_int + 4 * K; g.sp_k = g.sp_off + (N + 1);
  g.cl_off = g.sp_k + net.nterm; g.cl_ks = g.cl_off + (N + 1);
  {
    const int tab = ((net.ndbl + 1) & ~1) + ((net.nint + 3) & ~3) / 2;  // doubles, 16-byte aligned
    const int pg = CoopSmem<NEQ, LANES>::per_group(K);
    const int pga = (pg + 1) & ~1;
    double *base = smem + tab + (threadIdx.x / LANES) * pga;
    g.urow = base;                 // 2*LANES, 16-byte aligned
    g.ysh = g.urow + 2 * LANES;
    g.xs = g.ysh + LANES;
    g.R = g.xs + LANES;
    g.dRdT = g.R + K;
    g.dRdY = g.dRdT + K;
    g.M = g.dRdY + 3 * K;
  }
  const int lig = g.lig;
  const bool act = lig < n;      // lanes that own a component
  const double dt = A.dt, rtol = A.rtol, atol = A.atol;
  unsigned long long c_nst = 0, c_rhs = 0, c_jac = 0, c_lu = 0, c_sol = 0, c_etf = 0, c_cfn = 0, c_fail = 0;

  LuRow<NEQ, LANES> lu;

  for (;;) {
    // ---- a2: fetch the next zone from the work queue -------------------------------------------
    long long z = 0;
    if (lig == 0) z = (long long)atomicAdd(A.queue, 1ull);
    z = __shfl_sync(g.gmask, z, 0, LANES);
    if (z >= A.nz) break;

    // ---- a1: load zone state -------------------------------------------------------------------
    const double rho = A.rho[z];
    double xin = 0.0, ai = 1.0;
    if (lig >= 1 && lig <= N) {  // internal order: lane 0 = T, lane i + 1 = species i
      xin = A.X[(long long)(lig - 1) * A.nz + z];
      ai = g.aion[lig - 1];
    } else if (lig == 0) {
      xin = A.T[z];
    }
    const double y0 = (lig >= 1 && lig <= N) ? xin / ai : xin;
    bool bad = !(rho > 0.0) || !finite_(rho) || (act && !finite_(y0)) || (lig == 0 && !(y0 > 0.0));
    int code = 0;
    double yfin = y0;
    if (g.gany(bad)) {
      code = -4;
    } else {
      // ---- Init -------------------------------------------------------------------------------
      double Z[QMAX + 1];
#pragma unroll
      for (int j = 0; j <= QMAX; j++) Z[j] = 0.0;
      double f = g.template rates<true>(rho, y0);
      c_rhs++, c_jac++;
      double w = act ? 1.0 / fma_(rtol, fabs(y0), atol) : 0.0;
      double h;
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
      int q = 1, nqwait = 2, qS = 0, nst = 0, ntau = 0;
      double t = 0.0, etamax = ETAMX1, hS = 0.0, dsm = 0.0, S = 0.0, acor = 0.0;
      double tau[QMAX + 1], l[QMAX + 2], hs[QMAX + 1], rxi[QMAX + 1], xi[QMAX + 1], d[8];
#pragma unroll
      for (int i = 0; i <= QMAX; i++) tau[i] = 0.0, hs[i] = 0.0, rxi[i] = 0.0, xi[i] = 0.0;

      for (;;) {  // steps
        // A. end clip
        bool last;
        {
          const double rem = dt - t;
          if (h >= rem || rem - h < SLIVER * h) {
            nord_rescale(Z, q, rem / h);
            h = rem;
            last = true;
          } else
            last = false;
        }
        int ncf = 0, nef = 0;
        for (;;) {  // B. attempts
          // B.1 coefficients
          l[0] = 1.0;
#pragma unroll
          for (int j = 1; j <= QMAX + 1; j++) l[j] = 0.0;
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
          nord_predict(Z, q);  // B.2
          bool ok = false;
          double y = Z[0];
          bool inval = (act && !finite_(y)) || (lig == 0 && !(y > 0.0));
          if (!g.gany(inval)) {  // B.3
            f = g.template rates<true>(rho, y);
            c_rhs++, c_jac++;
#pragma unroll
            for (int j = 0; j < NEQ; j++) {
              const double Jij = (act && j < n) ? g.M[lig * LD + j] : 0.0;
              lu.a[j] = fma_(-gamma, Jij, (j == lig) ? 1.0 : 0.0);
            }
            const bool fok = lu.factor(g);
            c_lu++;
            if (fok) {  // B.4 Newton
              acor = 0.0;
              double crate = 1.0, delp = 0.0;
              const double tq = NTOL * cerr;
              for (int m = 0; m < MAXCOR; m++) {
                if (m > 0) {
                  y = Z[0] + acor;
                  inval = (act && !finite_(y)) || (lig == 0 && !(y > 0.0));
                  if (g.gany(inval)) break;
                  f = g.template rates<false>(rho, y);
                  c_rhs++;
                }
                double b = fma_(gamma, f, -fma_(Z[1], rl1, acor));
                b = lu.solve(g, b);
                c_sol++;
                acor = acor + b;
                const double del = g.wrms(b, w);
                if (!finite_(del)) break;
                if (m > 0) {
                  const double rr = del / delp;
                  crate = CRDOWN * crate;
                  if (rr > crate) crate = rr;
                }
                const double dcon = (del * (crate < 1.0 ? crate : 1.0)) / tq;
                if (dcon <= 1.0) {
                  ok = true;
                  break;
                }
                if (m > 0 && del > RDIV * delp) break;
                delp = del;
              }
            }
          }
          if (!ok) {  // B.6 Newton failure
            nord_retract(Z, q);
            ncf++, c_cfn++;
            etamax = 1.0;
            last = false;
            if (ncf > MXNCF) {
              code = -1;
              break;
            }
            nord_rescale(Z, q, ETACF);
            h = h * ETACF;
            continue;
          }
          // B.5 error test
          dsm = g.wrms(acor, w) / cerr;
          if (dsm <= 1.0) break;  // accept
          nord_retract(Z, q);
          nef++, c_etf++;
          etamax = 1.0;
          last = false;
          if (nef == MXNEF) {
            code = -2;
            break;
          }
          if (nef <= 2) {
            double eta = eta_of(dsm, BIAS2, q + 1);
            if (eta < ETAMIN) eta = ETAMIN;
            if (nef == 2 && eta > ETAMXF) eta = ETAMXF;
            nord_rescale(Z, q, eta);
            h = h * eta;
          } else if (q > 1) {
            double s = 0.0;
#pragma unroll
            for (int i = 1; i <= QMAX - 2; i++) {
              if (i <= q - 2) {
                s = (i == 1) ? tau[1] : s + tau[i];
                xi[i] = s / h;
              }
            }
            build_d(q - 2, xi, d);
            const double zq = sel(Z, q);
#pragma unroll
            for (int j = 2; j <= QMAX - 1; j++)
              if (j <= q - 1) Z[j] = fma_(-d[j], zq, Z[j]);
            q = q - 1;
            nqwait = q + 1;
            nord_rescale(Z, q, ETAMIN);
            h = h * ETAMIN;
          } else {
            h = h * ETAMIN;
            f = g.template rates<false>(rho, Z[0]);
            c_rhs++;
            Z[1] = h * f;
            nqwait = 10;
          }
        }
        if (code < 0) break;
        // C. accept
#pragma unroll
        for (int j = 0; j <= QMAX; j++)
          if (j <= q) Z[j] = fma_(l[j], acor, Z[j]);
        t = last ? dt : t + h;
        nst++;
        c_nst++;
        w = act ? 1.0 / fma_(rtol, fabs(Z[0]), atol) : 0.0;
        if (last) break;
        if (nst == MXSTEP) {
          code = -3;
          break;
        }
        // D. select next step and order
        double eta = 1.0;
        int action = 0;
        nqwait--;
        const double lq = sel(l, q);
        if (etamax == 1.0) {
          if (nqwait < 2) nqwait = 2;
        } else {
          const double etaq = eta_of(dsm, BIAS2, q + 1);
          if (nqwait != 0) {
            eta = etaq;
          } else {
            nqwait = 2;
            double etaqm1 = 0.0, etaqp1 = 0.0;
            if (q > 1) {
              double pm = rxi[1], sm = rxi[1];
#pragma unroll
              for (int i = 2; i <= QMAX - 1; i++)
                if (i <= q - 1) {
                  pm = pm * rxi[i];
                  sm = sm + rxi[i];
                }
              const double Em = g.wrms(sel(Z, q), w) / (pm * sm);
              etaqm1 = eta_of(Em, BIAS1, q);
            }
            if (q < QMAX && qS == q && ntau >= q) {
              const double rq1 = h / (sel(hs, q) + sel(tau, q));
              double pp = rxi[1], sp = rxi[1];
#pragma unroll
              for (int i = 2; i <= QMAX; i++)
                if (i <= q) {
                  pp = pp * rxi[i];
                  sp = sp + rxi[i];
                }
              pp = pp * rq1;
              sp = sp + rq1;
              const double cq = factorial_(q) * lq;
              const double rh = h / hS;
              double rs = rh;
#pragma unroll
              for (int j = 1; j <= QMAX; j++)
                if (j <= q) rs = rs * rh;
              const double v = fma_(cq, acor, -(rs * S));
              const double Ep = g.wrms(v, w) / ((pp * sp) * factorial_(q + 2));
              etaqp1 = eta_of(Ep, BIAS3, q + 2);
            }
            if (etaq >= etaqp1) {
              if (etaq >= etaqm1) {
                eta = etaq;
              } else {
                eta = etaqm1;
                action = -1;
              }
            } else {
              if (etaqp1 > etaqm1) {
                eta = etaqp1;
                action = +1;
              } else {
                eta = etaqm1;
                action = -1;
              }
            }
          }
          if (eta < THRESH) {
            eta = 1.0;
            action = 0;
          } else if (eta > etamax)
            eta = etamax;
        }
        if (nqwait == 1 && q < QMAX) {
          S = (factorial_(q) * lq) * acor;
          hS = h;
          qS = q;
        }
        // E. apply
        if (action == -1) {
#pragma unroll
          for (int i = 1; i <= QMAX - 2; i++)
            if (i <= q - 2) xi[i] = hs[i] / h;
          build_d(q - 2, xi, d);
          const double zq = sel(Z, q);
#pragma unroll
          for (int j = 2; j <= QMAX - 1; j++)
            if (j <= q - 1) Z[j] = fma_(-d[j], zq, Z[j]);
          q = q - 1;
          nqwait = q + 1;
        } else if (action == +1) {
#pragma unroll
          for (int i = 1; i <= QMAX - 1; i++)
            if (i <= q - 1) xi[i] = hs[i] / h;
          build_d(q - 1, xi, d);
          const double c = (lq * inv_small_int(q + 1)) * acor;
#pragma unroll
          for (int j = 2; j <= QMAX; j++) {
            if (j == q + 1) Z[j] = 0.0;
            if (j <= q + 1) Z[j] = fma_(d[j], c, Z[j]);
          }
          q = q + 1;
          nqwait = q + 1;
        }
#pragma unroll
        for (int i = QMAX; i >= 2; i--) tau[i] = tau[i - 1];
        tau[1] = h;
        if (ntau < 5) ntau++;
        etamax = ETAMAX;
        if (eta != 1.0) {
          nord_rescale(Z, q, eta);
          h = h * eta;
        }
      }
      yfin = Z[0];
      if (code == 0) code = nst;
    }
    // ---- a9: store ---------------------------------------------------------------------------
    if (code < 0) c_fail++;
    if (lig >= 1 && lig <= N) {
      A.X_out[(long long)(lig - 1) * A.nz + z] = (code == -4) ? xin : ai * yfin;
    } else if (lig == 0) {
      A.T_out[z] = (code == -4) ? xin : yfin;
      A.nsteps[z] = code;
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
