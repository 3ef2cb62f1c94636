// bz_cost_key.cuh -- step a2, second half: an a-priori cost key per zone, so that the work queue can hand
// the zones out dearest first (bz_set_schedule(net, 2); SURVEY.md 8(a) a2 names "a cost key" for the
// compaction).  Key = |sum_k Q_k R_k(rho, T, Y0)| / T, the relative heating rate at the initial state up to
// factors common to all zones (dt, N_A MeV / c_v): zones that will run away, and take hundreds of steps, have
// the largest.  One thread per zone, one right-hand side per zone (~1/1000 of a burn on config 3).  The key
// only ORDERS the queue: it never enters a result, so it has no counterpart in the oracle, and every zone's
// result is bit-identical whatever the order (tests/test_zone_order_gpu.py).
#pragma once
#include "bz_coop.cuh"

namespace bz {

// key[z] = high word of the double |s| / T (non-negative doubles order like their bit patterns; 11 exponent
// and 20 mantissa bits are far more than a schedule needs), idx[z] = z
__global__ void __launch_bounds__(256) cost_key_kernel(DevNet net, long long nz, long long ld, const double *__restrict__ rho,
                                                       const double *__restrict__ T, const double *__restrict__ X,
                                                       unsigned *__restrict__ key, long long *__restrict__ idx) {
  const long long z = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (z >= nz) return;
  const int N = net.N, K = net.K;
  const double *lnA = net.dbl, *en = net.dbl + K, *B = net.dbl + 2 * K, *Q = net.dbl + 3 * K, *invsym = net.dbl + 4 * K;
  const double *aion = net.dbl + 5 * K;
  const double *rexp = net.has_rexp ? net.dbl + 5 * K + N + net.nterm : nullptr;
  const int4 *rp = reinterpret_cast<const int4 *>(net.itab);
  double Y[32];
  for (int i = 0; i < N; i++) Y[i] = fabs(X[(long long)i * ld + z]) / aion[i];
  const double r = rho[z], Tz = T[z];
  const double T9 = Tz * 1e-9;
  const double lnT9 = log_(T9);
  const double t13 = exp_(lnT9 * (-1.0 / 3.0));
  const double lnrho = rexp ? log_(r) : 0.0;
  double s = 0.0;
  for (int k = 0; k < K; k++) {
    const int4 rpk = rp[k];
    const int m = rpk.x & 0xff;
    double arg = fma_(-B[k], t13, fma_(en[k], lnT9, lnA[k]));
    if (rexp) arg = fma_(rexp[k], lnrho, arg);
    double R = exp_(arg) * (m == 1 ? 1.0 : (m == 2 ? r : r * r)) * invsym[k] * Y[rpk.y & 0xff];
    if (m >= 2) R = R * Y[(rpk.y >> 8) & 0xff];
    if (m >= 3) R = R * Y[(rpk.y >> 16) & 0xff];
    s = fma_(Q[k], R, s);
  }
  const double c = fabs(s) / Tz;
  key[z] = (c == c && c > 0.0) ? (unsigned)(__double_as_longlong(c) >> 32) : 0u;  // NaN, zero -> cheapest
  idx[z] = z;
}

}  // namespace bz
