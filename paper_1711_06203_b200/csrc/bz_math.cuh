// bz_math.cuh -- device-side exp/log with a fixed IEEE operation sequence (DESIGN.md 3.6,
// item 3).  Compiled with -fmad=false: every fused operation is an explicit fma().
// libdevice exp/log are NOT used on the burn path: their results differ from any host libm by
// an ulp in a few per cent of calls, which the BDF controller amplifies.
#pragma once
#include <cuda_runtime.h>

namespace bz {

// Polynomial coefficients live in constant memory so that each Horner step is ONE DFMA with a
// constant-bank operand (as 64-bit immediates they cost two extra UMOV per step).
__constant__ double EXP_C[14] = {1.0, 1.0, 1.0 / 2.0, 1.0 / 6.0, 1.0 / 24.0, 1.0 / 120.0, 1.0 / 720.0,
                                 1.0 / 5040.0, 1.0 / 40320.0, 1.0 / 362880.0, 1.0 / 3628800.0,
                                 1.0 / 39916800.0, 1.0 / 479001600.0, 1.0 / 6227020800.0};
__constant__ double LOG_C[12] = {1.0, 1.0 / 3.0, 1.0 / 5.0, 1.0 / 7.0, 1.0 / 9.0, 1.0 / 11.0, 1.0 / 13.0,
                                 1.0 / 15.0, 1.0 / 17.0, 1.0 / 19.0, 1.0 / 21.0, 1.0 / 23.0};

__device__ __forceinline__ double fma_(double a, double b, double c) { return __fma_rn(a, b, c); }

// exp(x) = 2^k exp(r), r = x - k ln2 (two-piece ln2), exp(r) = sum_{j<=13} r^j/j! by Horner.
// x < -700 -> 0, x > 700 -> +inf, so the scaling by 2^k is exact (no subnormal results).
__device__ __forceinline__ double exp_(double x) {
  constexpr double LOG2E = 1.4426950408889634;
  constexpr double LN2_HI = 0x1.62e42fee00000p-1;
  constexpr double LN2_LO = 0x1.a39ef35793c76p-33;
  if (!(x >= -700.0)) return (x != x) ? x : 0.0;
  if (x > 700.0) return __longlong_as_double(0x7ff0000000000000LL);
  const double kd = rint(x * LOG2E);
  double r = fma_(-kd, LN2_HI, x);
  r = fma_(-kd, LN2_LO, r);
  double p = EXP_C[13];
#pragma unroll
  for (int j = 12; j >= 0; j--) p = fma_(p, r, EXP_C[j]);
  const int k = (int)kd;  // |k| <= 1010
  const double scale = __longlong_as_double((long long)(k + 1023) << 52);
  return p * scale;  // exact: p in [0.7, 1.42], result normal
}

// log(x), x > 0 normal: x = m 2^e with m in [sqrt(1/2), sqrt(2)); log m = 2 atanh((m-1)/(m+1)).
__device__ __forceinline__ double log_(double x) {
  constexpr double LN2_HI = 0x1.62e42fee00000p-1;
  constexpr double LN2_LO = 0x1.a39ef35793c76p-33;
  const long long bits = __double_as_longlong(x);
  int e = (int)((bits >> 52) & 0x7ff) - 1022;  // frexp exponent: x = m 2^e, m in [0.5, 1)
  double m = __longlong_as_double((bits & 0x800fffffffffffffLL) | 0x3fe0000000000000LL);
  if (m < 0.70710678118654752) {
    m = 2.0 * m;
    e -= 1;
  }
  const double s = (m - 1.0) / (m + 1.0);
  const double z = s * s;
  double p = LOG_C[11];
#pragma unroll
  for (int j = 10; j >= 0; j--) p = fma_(p, z, LOG_C[j]);
  const double t = (2.0 * s) * p;
  const double ed = (double)e;
  return fma_(ed, LN2_HI, fma_(ed, LN2_LO, t));
}

// x with its sign bit xor-ed by `mask` (0 or 0x80000000): a conditional negation that costs one
// integer LOP3 on the high word instead of DADD + 2 FSEL.  Bit-identical to `cond ? -x : x`.
__device__ __forceinline__ double flip_(double x, unsigned mask) {
  return __hiloint2double(__double2hiint(x) ^ (int)mask, __double2loint(x));
}

__device__ __forceinline__ bool finite_(double x) {
  return (__double_as_longlong(x) & 0x7ff0000000000000LL) != 0x7ff0000000000000LL;
}

}  // namespace bz
