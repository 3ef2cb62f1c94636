/* bz_oracle.c -- plain, slow, scalar CPU oracle of the per-zone burn (see bz_oracle.h).
 * TEST INFRASTRUCTURE ONLY; independent of the CUDA path; generic-n loops on stack arrays.
 *
 * Build: gcc -O2 -std=c11 -ffp-contract=off -mfma -fopenmp -shared -fPIC  (oracle/build.py)
 * -ffp-contract=off: every fused multiply-add below is an explicit fma(); nothing else is
 * fused, so the IEEE operation sequence is exactly what is written.
 *
 * Section numbers in comments (C.1, C.2-A..E, C.5) are SURVEY.md section 8(c), restated in
 * DESIGN.md section 3; "L119" etc. are PAPER.md lines.
 */
#include "bz_oracle.h"
#include <math.h>
#include <string.h>
#include <stdlib.h>
#ifdef _OPENMP
#include <omp.h>
#endif

/* ---- constants of C.1 / C.2 ------------------------------------------------------- */
#define NA_MEV 9.648533212331e17 /* N_A * 1 MeV in erg/mol */
#define RGAS 8.31446261815324e7  /* N_A k_B, erg/mol/K (analytic EOS) */
#define ARAD 7.565733250e-15     /* radiation constant a, erg/cm^3/K^4 */
#define QMAX 5
#define MAXCOR 3
#define NTOL 0.1
#define CRDOWN 0.3
#define RDIV 2.0
#define ETACF 0.25
#define MXNCF 10
#define MXNEF 7
#define BIAS1 4.0
#define BIAS2 6.0
#define BIAS3 10.0
#define ADDON 1e-6
#define THRESH 1.5
#define ETAMIN 0.1
#define ETAMXF 0.2
#define ETAMX1 1e4
#define ETAMAX 2.0
#define MXSTEP 20000
#define SLIVER 1e-6
/* policy 1 ("BZ-BDF v2": VODE's Newton-matrix reuse, ref. [33] PAPER.md:L184) */
#define CCMAX 0.3 /* refactor when |gamma/gamma_P - 1| exceeds this */
#define MSBP 20   /* ... or when this many steps were accepted since the last factorisation */

static const double FACT[8] = {1.0, 1.0, 2.0, 6.0, 24.0, 120.0, 720.0, 5040.0};
static const double INVP[8] = {0.0, 1.0, 1.0 / 2.0, 1.0 / 3.0, 1.0 / 4.0, 1.0 / 5.0, 1.0 / 6.0, 1.0 / 7.0};

/* ---- C.5 item 3: own exp / log (no libm transcendentals) -------------------------- */
#define LOG2E 1.4426950408889634
#define LN2_HI 0x1.62e42fee00000p-1
#define LN2_LO 0x1.a39ef35793c76p-33

double orc_exp(double x) {
  /* exp(x) = 2^kd * exp(r), r = x - kd ln2 in two pieces, exp(r) = sum_{k<=13} r^k/k!.
   * Arguments below -700 flush to 0 and above 700 give +inf (no subnormal results, so the
   * final scaling is an exact multiplication by a normal power of two). */
  static const double C[14] = {1.0, 1.0, 1.0 / 2.0, 1.0 / 6.0, 1.0 / 24.0, 1.0 / 120.0,
                               1.0 / 720.0, 1.0 / 5040.0, 1.0 / 40320.0, 1.0 / 362880.0,
                               1.0 / 3628800.0, 1.0 / 39916800.0, 1.0 / 479001600.0,
                               1.0 / 6227020800.0};
  if (!(x >= -700.0)) return (x != x) ? x : 0.0;
  if (x > 700.0) return INFINITY;
  double kd = rint(x * LOG2E);
  double r = fma(-kd, LN2_HI, x);
  r = fma(-kd, LN2_LO, r);
  double p = C[13];
  for (int k = 12; k >= 0; k--) p = fma(p, r, C[k]);
  return ldexp(p, (int)kd);
}

double orc_log(double x) {
  /* x > 0 normal.  x = m 2^e, m in [sqrt(1/2), sqrt(2)); log m = 2 atanh(s), s=(m-1)/(m+1) */
  static const double C[12] = {1.0, 1.0 / 3.0, 1.0 / 5.0, 1.0 / 7.0, 1.0 / 9.0, 1.0 / 11.0,
                               1.0 / 13.0, 1.0 / 15.0, 1.0 / 17.0, 1.0 / 19.0, 1.0 / 21.0,
                               1.0 / 23.0};
  int e;
  double m = frexp(x, &e); /* m in [0.5, 1) */
  if (m < 0.70710678118654752) {
    m = 2.0 * m;
    e -= 1;
  }
  double s = (m - 1.0) / (m + 1.0);
  double z = s * s;
  double p = C[11];
  for (int k = 10; k >= 0; k--) p = fma(p, z, C[k]);
  double t = (2.0 * s) * p;
  double ed = (double)e;
  return fma(ed, LN2_HI, fma(ed, LN2_LO, t));
}

/* ---- the network (C.1) -------------------------------------------------------------- */
typedef struct {
  int N, n, K;
  double aion[ORC_NMAX];
  int m[ORC_KMAX];         /* number of reactant particles 1..3      */
  int r[ORC_KMAX][3];
  int ns[ORC_KMAX];        /* number of stoichiometry entries 1..4   */
  int sid[ORC_KMAX][4];
  double sdy[ORC_KMAX][4];
  double lnA[ORC_KMAX], en[ORC_KMAX], B[ORC_KMAX], Q[ORC_KMAX], invsym[ORC_KMAX];
  int has_rexp;            /* the descriptor carries density exponents */
  double rexp[ORC_KMAX];
  int eos;                 /* 1: c_v from the analytic EOS, evaluated with every right-hand side */
  double zp1[ORC_NMAX];    /* 1 + Z_i */
  double eos_extra;
  double fac;              /* N_A MeV / c_v                          */
} Net;

static int net_init(Net *nt, const orc_net_desc *d) {
  if (!d || d->nspec < 1 || d->nspec > ORC_NMAX - 1 || d->nreac < 1 || d->nreac > ORC_KMAX) return -2;
  nt->N = d->nspec;
  nt->n = d->nspec + 1;
  nt->K = d->nreac;
  nt->eos = (d->zion != NULL);
  if (!nt->eos && !(d->cv > 0.0)) return -3;
  nt->fac = nt->eos ? 0.0 : NA_MEV / d->cv;
  nt->eos_extra = nt->eos ? d->eos_extra : 0.0;
  if (nt->eos && (!isfinite(d->eos_extra) || d->eos_extra < 0.0)) return -3;
  for (int i = 0; i < d->nspec && nt->eos; i++) {
    if (!isfinite(d->zion[i]) || d->zion[i] < 0.0) return -3;
    nt->zp1[i] = 1.0 + d->zion[i];
  }
  nt->has_rexp = (d->rate_rho_exp != NULL);
  for (int i = 0; i < nt->N; i++) {
    if (!(d->aion[i] > 0.0)) return -3;
    nt->aion[i] = d->aion[i];
  }
  for (int k = 0; k < nt->K; k++) {
    int m = 0;
    for (int a = 0; a < 3; a++) {
      int id = d->reactant[3 * k + a];
      if (id < 0) continue;
      if (id >= nt->N) return -3;
      nt->r[k][m++] = id;
    }
    if (m == 0) return -3;
    nt->m[k] = m;
    int ns = 0;
    for (int a = 0; a < 4; a++) {
      int id = d->stoich_id[4 * k + a];
      if (id < 0) continue;
      if (id >= nt->N) return -3;
      nt->sid[k][ns] = id;
      nt->sdy[k][ns] = d->stoich_dy[4 * k + a];
      ns++;
    }
    nt->ns[k] = ns;
    if (!(d->rate_A[k] > 0.0) || !isfinite(d->rate_A[k]) || !isfinite(d->rate_n[k]) ||
        !isfinite(d->rate_B[k]) || !isfinite(d->q_mev[k]))
      return -3;
    nt->lnA[k] = orc_log(d->rate_A[k]);
    nt->en[k] = d->rate_n[k];
    nt->B[k] = d->rate_B[k];
    nt->Q[k] = d->q_mev[k];
    nt->rexp[k] = 0.0;
    if (d->rate_rho_exp) {
      if (!isfinite(d->rate_rho_exp[k])) return -3;
      nt->rexp[k] = d->rate_rho_exp[k];
    }
    /* 1 / prod_i nu_ik!  (reading s2): 1, 1/2 (one pair), 1/6 (triple) */
    int r0 = nt->r[k][0], r1 = m > 1 ? nt->r[k][1] : -1, r2 = m > 2 ? nt->r[k][2] : -2;
    int same = (r0 == r1) + (r0 == r2) + (r1 == r2);
    nt->invsym[k] = same == 0 ? 1.0 : (same == 1 ? 0.5 : 1.0 / 6.0);
  }
  return 0;
}

/* f (and J, row-major n x n, if J != NULL) at (rho, y).  C.1.
 *   lambda_k = exp(lnA_k + n_k ln T9 - B_k t13),  t13 = T9^(-1/3) = exp(-ln(T9)/3)
 *   R_k = ((lambda_k rho^(m-1)) invsym_k) * Y_r0 * Y_r1 * Y_r2
 *   dR_k/dY_j = pref_k * sum_{positions a: r[a]=j} prod_{b != a} Y_r[b]   (never R/Y)
 *   dR_k/dT   = R_k (n_k + B_k t13/3) / T
 * Negative abundances (the integrator lets trace species dip to ~ -atol), reading s19: the ODD,
 * MONOTONE EXTENSION.  Products are formed from |Y|; if ANY reactant of reaction k is negative the
 * rate is R_k = -pref_k prod|Y_r| (else +pref_k prod Y_r); dR_k/dY_j = pref_k d(prod|Y|)/d|Y_j|,
 * negated when some reactant is negative UNLESS species j itself is (then d|Y_j|/dY_j = -1 cancels
 * the sign of the rate).  Equal to the raw product law whenever at most one factor is negative.
 * Accumulation order: reactions k ascending; per reaction the stoichiometry entries in table
 * order; the temperature row accumulates sum_k Q_k (.) and is scaled by fac at the end. */
/* Internal ordering of the unknowns (reading s25): y = (T, Y_0, ..., Y_{N-1}),
 * temperature FIRST.  The temperature equation carries the largest Jacobian entries
 * (N_A MeV/c_v ~ 1e10), so with T first partial pivoting keeps the natural order. */
#define SP(i) ((i) + 1)
#define TI 0
static void rates(const Net *nt, double rho, const double *y, double *f, double *J) {
  const int N = nt->N, n = nt->n;
  double sT = 0.0, JT[ORC_NMAX], ya[ORC_NMAX];
  for (int i = 0; i < n; i++) f[i] = 0.0;
  if (J) {
    for (int i = 0; i < n * n; i++) J[i] = 0.0;
    for (int j = 0; j < n; j++) JT[j] = 0.0;
  }
  for (int i = 0; i < N; i++) ya[i] = fabs(y[SP(i)]);
  const double T = y[TI];
  const double T9 = T * 1e-9;
  const double lnT9 = orc_log(T9);
  const double t13 = orc_exp(lnT9 * (-1.0 / 3.0));
  const double t13third = t13 * (1.0 / 3.0);
  const double invT = 1.0 / T;
  const double rhopow[4] = {0.0, 1.0, rho, rho * rho};
  /* density exponents (optional): lambda_k *= rho^e_k, taken into the exponent with the own log */
  const double lnrho = nt->has_rexp ? orc_log(rho) : 0.0;
  for (int k = 0; k < nt->K; k++) {
    const int m = nt->m[k];
    const int *r = nt->r[k];
    double arg = fma(-nt->B[k], t13, fma(nt->en[k], lnT9, nt->lnA[k]));
    if (nt->has_rexp) arg = fma(nt->rexp[k], lnrho, arg);
    double lam = orc_exp(arg);
    double pref = (lam * rhopow[m]) * nt->invsym[k];
    int anyneg = 0;
    for (int a = 0; a < m; a++) anyneg |= (y[SP(r[a])] < 0.0);
    double R = pref;
    for (int a = 0; a < m; a++) R = R * ya[r[a]];
    if (anyneg) R = -R; /* reading s19: odd, monotone extension to Y < 0 */
    for (int s = 0; s < nt->ns[k]; s++) f[SP(nt->sid[k][s])] = fma(nt->sdy[k][s], R, f[SP(nt->sid[k][s])]);
    sT = fma(nt->Q[k], R, sT);
    if (!J) continue;
    /* species columns: distinct reactant species in order of first appearance */
    for (int a = 0; a < m; a++) {
      int j = r[a], seen = 0;
      for (int b = 0; b < a; b++) seen |= (r[b] == j);
      if (seen) continue;
      double d = 0.0;
      int first = 1;
      for (int p = 0; p < m; p++) {
        if (r[p] != j) continue;
        double prod = 1.0;
        int pf = 1;
        for (int b = 0; b < m; b++) {
          if (b == p) continue;
          prod = pf ? ya[r[b]] : prod * ya[r[b]];
          pf = 0;
        }
        d = first ? prod : d + prod;
        first = 0;
      }
      double dRdY = (m == 1) ? pref : pref * d;
      if (anyneg && !(y[SP(j)] < 0.0)) dRdY = -dRdY;
      for (int s = 0; s < nt->ns[k]; s++) {
        int i = SP(nt->sid[k][s]);
        J[i * n + SP(j)] = fma(nt->sdy[k][s], dRdY, J[i * n + SP(j)]);
      }
      JT[SP(j)] = fma(nt->Q[k], dRdY, JT[SP(j)]);
    }
    /* temperature column */
    double g = fma(nt->B[k], t13third, nt->en[k]);
    double dRdT = (R * g) * invT;
    for (int s = 0; s < nt->ns[k]; s++) {
      int i = SP(nt->sid[k][s]);
      J[i * n + TI] = fma(nt->sdy[k][s], dRdT, J[i * n + TI]);
    }
    JT[TI] = fma(nt->Q[k], dRdT, JT[TI]);
  }
  if (!nt->eos) {
    f[TI] = nt->fac * sT;
    if (J)
      for (int j = 0; j < n; j++) J[TI * n + j] = nt->fac * JT[j];
    return;
  }
  /* analytic EOS: c_v = 1.5 R (extra + sum_i (1+Z_i) Y_i) + 4 a T^3 / rho, raw Y, i ascending;
   * dT/dt = (N_A MeV / c_v) sum_k Q_k R_k; the temperature row of J gains -f_T (dc_v/dy_j) / c_v */
  double ysum = nt->eos_extra;
  for (int i = 0; i < N; i++) ysum = fma(nt->zp1[i], y[SP(i)], ysum);
  const double T2 = T * T;
  const double invrho = 1.0 / rho;
  const double cv = fma(1.5 * RGAS, ysum, ((4.0 * ARAD) * (T2 * T)) * invrho);
  const double invcv = 1.0 / cv;
  const double facv = NA_MEV * invcv;
  f[TI] = facv * sT;
  if (J) {
    const double g = f[TI] * invcv;
    J[TI * n + TI] = fma(-g, ((12.0 * ARAD) * T2) * invrho, facv * JT[TI]);
    for (int i = 0; i < N; i++) J[TI * n + SP(i)] = fma(-g, (1.5 * RGAS) * nt->zp1[i], facv * JT[SP(i)]);
  }
}

/* ---- dense LU, LINPACK dgefa/dgesl order (step a5/a6; C.5 item 4) ------------------- */
/* test aids: how often rarely taken paths ran since the last reset --
 * [0] row interchanges in orc_lu_factor, [1] third error-test failure lowering the order
 * (C.2-B.5, q > 1), [2] third error-test failure restarting at order 1 (q = 1). */
static unsigned long long g_events[3] = {0, 0, 0};
#define ORC_EVENT(i) __atomic_fetch_add(&g_events[i], 1ull, __ATOMIC_RELAXED)
void orc_event_counts(int reset, unsigned long long out[3]) {
  for (int i = 0; i < 3; i++) {
    out[i] = __atomic_load_n(&g_events[i], __ATOMIC_RELAXED);
    if (reset) __atomic_store_n(&g_events[i], 0ull, __ATOMIC_RELAXED);
  }
}
unsigned long long orc_interchanges(int reset) {
  unsigned long long v = __atomic_load_n(&g_events[0], __ATOMIC_RELAXED);
  if (reset) __atomic_store_n(&g_events[0], 0ull, __ATOMIC_RELAXED);
  return v;
}

int orc_lu_factor(int n, double *a, int32_t *ipvt, double *inv) {
  int info = 0;
  for (int k = 0; k < n; k++) {
    /* pivot: first maximal |a_ik|, i = k..n-1, in the current (swapped) row order */
    int p = k;
    double amax = fabs(a[k * n + k]);
    for (int i = k + 1; i < n; i++) {
      double v = fabs(a[i * n + k]);
      if (v > amax) {
        amax = v;
        p = i;
      }
    }
    ipvt[k] = p;
    if (!(amax > 0.0)) { /* zero or NaN pivot column */
      if (!info) info = k + 1;
      inv[k] = 0.0;
      continue;
    }
    /* LINPACK: interchange rows k and p in columns k..n-1 only (earlier multipliers stay) */
    if (p != k) ORC_EVENT(0);
    if (p != k)
      for (int j = k; j < n; j++) {
        double t = a[p * n + j];
        a[p * n + j] = a[k * n + j];
        a[k * n + j] = t;
      }
    inv[k] = 1.0 / a[k * n + k];
    for (int i = k + 1; i < n; i++) a[i * n + k] = a[i * n + k] * inv[k];
    for (int i = k + 1; i < n; i++) {
      double l = a[i * n + k];
      for (int j = k + 1; j < n; j++) a[i * n + j] = fma(-l, a[k * n + j], a[i * n + j]);
    }
  }
  return info;
}

void orc_lu_solve(int n, const double *a, const int32_t *ipvt, const double *inv, double *b) {
  /* forward: interchanges interleaved (dgesl job 0), k ascending, axpy form */
  for (int k = 0; k < n; k++) {
    int p = ipvt[k];
    double t = b[p];
    b[p] = b[k];
    b[k] = t;
    for (int i = k + 1; i < n; i++) b[i] = fma(-a[i * n + k], t, b[i]);
  }
  /* backward: k descending, x_k = b_k * (1/u_kk), then axpy into rows above */
  for (int k = n - 1; k >= 0; k--) {
    b[k] = b[k] * inv[k];
    double t = b[k];
    for (int i = 0; i < k; i++) b[i] = fma(-a[i * n + k], t, b[i]);
  }
}

/* ---- WRMS norm ||v|| = sqrt((1/n) sum (v_i w_i)^2)  (C.2; association: C.5 item 5) ---- */
double orc_wrms(int n, const double *v, const double *w, int lanes) {
  double part[32], nxt[32];
  if (lanes < 1) lanes = 1;
  for (int q = 0; q < lanes; q++) part[q] = 0.0;
  for (int i = 0; i < n; i++) {
    double d = v[i] * w[i];
    part[i % lanes] = fma(d, d, part[i % lanes]);
  }
  for (int s = lanes / 2; s >= 1; s /= 2) { /* xor butterfly, strides L/2 .. 1 */
    for (int q = 0; q < lanes; q++) nxt[q] = part[q] + part[q ^ s];
    for (int q = 0; q < lanes; q++) part[q] = nxt[q];
  }
  return sqrt(part[0] * (1.0 / (double)n));
}

/* ---- C.2-B.1: l(x) = prod_{i=1..q} (1 + x/xi_i) ------------------------------------- */
/* hs[i] = h + tau_1 + ... + tau_{i-1} (hs[1] = h), rxi[i] = h/hs[i] = 1/xi_i */
static void bdf_coeffs(int q, double h, const double *tau, double *l, double *hs, double *rxi) {
  l[0] = 1.0;
  for (int j = 1; j <= q + 1; j++) l[j] = 0.0;
  double s = h;
  for (int i = 1; i <= q; i++) {
    if (i > 1) s = s + tau[i - 1];
    hs[i] = s;
    double r = h / s;
    rxi[i] = r;
    for (int j = i; j >= 1; j--) l[j] = fma(l[j - 1], r, l[j]);
  }
}

void orc_bdf_coeffs(int q, double h, const double *tau, double *l) {
  double hs[8], rxi[8], ll[8];
  bdf_coeffs(q, h, tau, ll, hs, rxi);
  for (int j = 0; j <= q; j++) l[j] = ll[j];
}

/* d(x) = x^2 prod_{i=1..cnt} (x + xi[i]) = sum_j d_j x^j, one linear factor at a time */
static void build_d(int cnt, const double *xi, double *d) {
  for (int j = 0; j < 8; j++) d[j] = 0.0;
  d[2] = 1.0;
  int deg = 2;
  for (int i = 1; i <= cnt; i++) {
    for (int j = deg + 1; j >= 1; j--) d[j] = fma(xi[i], d[j], d[j - 1]);
    d[0] = xi[i] * d[0];
    deg++;
  }
}

void orc_build_d(int cnt, const double *xi, double *d) { build_d(cnt, xi, d); }

/* eta = 1 / ((bias*E)^(1/p) + ADDON), the root through the own exp/log */
static double eta_of(double E, double bias, int p) {
  double v = bias * E;
  double root = (v > 1e-300) ? orc_exp(orc_log(v) * INVP[p]) : 0.0;
  return 1.0 / (root + ADDON);
}

/* ---- the integrator, C.2 ("BZ-BDF v1") ------------------------------------------------ */
static int invalid_state(int n, const double *y) {
  for (int i = 0; i < n; i++)
    if (!isfinite(y[i])) return 1;
  (void)n;
  return !(y[TI] > 0.0);
}
static void set_weights(int n, const double *y, double rtol, double atol, double *w) {
  for (int i = 0; i < n; i++) w[i] = 1.0 / fma(rtol, fabs(y[i]), atol);
}
static void predict(int n, int q, double Z[][ORC_NMAX]) { /* B.2, Pascal triangle in place */
  for (int k = 1; k <= q; k++)
    for (int j = q; j >= k; j--)
      for (int i = 0; i < n; i++) Z[j - 1][i] = Z[j - 1][i] + Z[j][i];
}
static void retract(int n, int q, double Z[][ORC_NMAX]) { /* B.7, same loop order */
  for (int k = 1; k <= q; k++)
    for (int j = q; j >= k; j--)
      for (int i = 0; i < n; i++) Z[j - 1][i] = Z[j - 1][i] - Z[j][i];
}
static void rescale(int n, int q, double Z[][ORC_NMAX], double eta) { /* Z_j *= eta^j */
  double r = eta;
  for (int j = 1; j <= q; j++) {
    for (int i = 0; i < n; i++) Z[j][i] = Z[j][i] * r;
    r = r * eta;
  }
}

/* constant source terms: f <- f + s, one rounded addition per component after the network's own
 * sums are complete (the Jacobian is unchanged: s does not depend on y).  src == NULL: f untouched. */
static void add_source(int n, const double *src, double *f) {
  if (!src) return;
  for (int i = 0; i < n; i++) f[i] = f[i] + src[i];
}

/* test hook (orc_opts.trace): copy one event record out; no arithmetic of the method here */
typedef struct {
  double *buf;
  int cap, n_unk, count;
} Trace;
static void trace_put(Trace *tr, const double head[ORC_TRACE_HEAD], double Zacc[][ORC_NMAX],
                      double Zend[][ORC_NMAX]) {
  if (!tr || !tr->buf) return;
  const int n = tr->n_unk;
  if (tr->count < tr->cap) {
    double *r = tr->buf + (size_t)tr->count * (ORC_TRACE_HEAD + 12 * n);
    for (int i = 0; i < ORC_TRACE_HEAD; i++) r[i] = head[i];
    for (int j = 0; j <= QMAX; j++)
      for (int i = 0; i < n; i++) { /* API order: T last */
        const int e = (i == TI) ? n - 1 : i - 1;
        r[ORC_TRACE_HEAD + j * n + e] = Zacc ? Zacc[j][i] : 0.0;
        r[ORC_TRACE_HEAD + (6 + j) * n + e] = Zend[j][i];
      }
  }
  tr->count++;
}

/* one zone.  returns nst (>0) or a negative failure code; yout = last accepted state */
static int burn_zone(const Net *nt, double rho, const double *y0, double dt, double rtol,
                     double atol, const orc_opts *o, const double *src, double *yout, uint64_t *cnt,
                     Trace *tr) {
  const int n = nt->n;
  const int L = (o && o->norm_lanes > 0) ? o->norm_lanes : 1;
  const int fixed = (o && o->fixed_q > 0);
  const int mxstep = (o && o->mxstep > 0) ? o->mxstep : MXSTEP;
  const int mxnef = (o && o->mxnef > 0) ? o->mxnef : MXNEF;
  const int mxncf = (o && o->mxncf > 0) ? o->mxncf : MXNCF;
  /* policy 1: the LU of P = I - gamma_P J is KEPT across steps (P, inv, ipvt below persist) */
  const int reuse = (o && o->policy == 1);
  double gamP = 0.0;
  int nslp = 0, haveP = 0, forceP = 0;
  double Z[QMAX + 2][ORC_NMAX], S[ORC_NMAX], w[ORC_NMAX], acor[ORC_NMAX], y[ORC_NMAX];
  double f[ORC_NMAX], b[ORC_NMAX], vtmp[ORC_NMAX];
  double P[ORC_NMAX * ORC_NMAX], inv[ORC_NMAX];
  int32_t ipvt[ORC_NMAX];
  double tau[8] = {0}, l[8], hs[8], rxi[8], xi[8], d[8];
  int ntau = 0;
  double Zacc[QMAX + 2][ORC_NMAX], thead[ORC_TRACE_HEAD]; /* trace hook only */
  for (int j = 0; j < QMAX + 2; j++)
    for (int i = 0; i < ORC_NMAX; i++) Z[j][i] = 0.0, Zacc[j][i] = 0.0;

  for (int i = 0; i < n; i++) yout[i] = y0[i];
  if (!(rho > 0.0) || !isfinite(rho) || invalid_state(n, y0)) return -4;
  if (src)
    for (int i = 0; i < n; i++)
      if (!isfinite(src[i])) return -4;

  /* Init */
  rates(nt, rho, y0, f, P);
  add_source(nt->n, src, f);
  cnt[1]++, cnt[2]++;
  set_weights(n, y0, rtol, atol, w);
  double h;
  int q = 1;
  if (!fixed) {
    for (int i = 0; i < n; i++) { /* exact second derivative y'' = J f */
      double s = 0.0;
      for (int j = 0; j < n; j++) s = fma(P[i * n + j], f[j], s);
      vtmp[i] = s;
    }
    double d2 = orc_wrms(n, vtmp, w, L);
    h = dt;
    if (d2 > 0.0) {
      double hh = 0.5 * sqrt(2.0 / d2);
      if (hh < dt) h = hh;
    }
    for (int i = 0; i < n; i++) {
      Z[0][i] = y0[i];
      Z[1][i] = h * f[i];
    }
  } else {
    h = o->fixed_h;
    q = o->fixed_q;
    for (int j = 0; j <= q; j++)
      for (int i = 0; i < n; i++) Z[j][i] = o->z_init[j * n + (i == TI ? n - 1 : i - 1)]; /* API order: T last */
    for (int i = 1; i <= 5; i++) tau[i] = h;
    ntau = 5;
  }
  double t = 0.0, etamax = ETAMX1, hS = 0.0, dsm = 0.0;
  int nqwait = 2, qS = 0, nst = 0;

  for (;;) {
    /* A. end clip */
    int last;
    {
      double rem = dt - t;
      if (h >= rem || rem - h < SLIVER * h) {
        double eta = rem / h;
        rescale(n, q, Z, eta);
        h = rem;
        last = 1;
      } else
        last = 0;
    }
    /* B. attempt, repeated until accepted */
    int ncf = 0, nef = 0;
    double cerr;
    for (;;) {
      int predicted = 0, ok = 0;
      bdf_coeffs(q, h, tau, l, hs, rxi); /* B.1 */
      const double l1 = l[1];
      const double gamma = h / l1;
      const double rl1 = 1.0 / l1;
      cerr = (double)(q + 1) * l1;
      predict(n, q, Z); /* B.2 */
      predicted = 1;
      for (int i = 0; i < n; i++) y[i] = Z[0][i];
      int jcur = 1, tried = 0; /* jcur: P was factorised in THIS attempt (always, under policy 0) */
      if (!invalid_state(n, y)) { /* B.3 */
        tried = 1;
        int needP = 1;
        if (reuse) {
          /* policy 1, B.3': factorise only if there is no P yet, a failure asked for it, gamma has
           * drifted more than CCMAX from gamma_P, or MSBP steps were accepted since */
          /* |gamma/gamma_P - 1| > CCMAX written without a division: gl = gamma_P l_1 ( = h_P l_1/l_1P ) */
          const double gl = gamP * l1;
          needP = !haveP || forceP || fabs(h - gl) > CCMAX * gl || (nst - nslp >= MSBP);
        }
        int info = 0;
        if (needP) {
          rates(nt, rho, y, f, P);
          add_source(n, src, f);
          cnt[1]++, cnt[2]++;
          for (int i = 0; i < n; i++)
            for (int j = 0; j < n; j++) P[i * n + j] = fma(-gamma, P[i * n + j], (i == j) ? 1.0 : 0.0);
          info = orc_lu_factor(n, P, ipvt, inv);
          cnt[3]++;
          gamP = gamma, nslp = nst, haveP = !info, forceP = 0;
        } else {
          rates(nt, rho, y, f, NULL);
          add_source(n, src, f);
          cnt[1]++;
          jcur = 0;
        }
        /* policy 1: every correction solved with a STALE matrix is scaled by 2/(1 + gamma/gamma_P), written
         * as 2 gl/(gl + h) with gl = gamma_P l_1 (one division that does not wait for gamma = h/l_1) */
        double cscale = 1.0;
        if (reuse && !jcur) {
          const double gl = gamP * l1;
          cscale = (2.0 * gl) / (gl + h);
        }
        if (!info) { /* B.4 Newton */
          for (int i = 0; i < n; i++) acor[i] = 0.0;
          double crate = 1.0, delp = 0.0;
          const double tq = NTOL * cerr;
          for (int m = 0; m < MAXCOR; m++) {
            if (m > 0) {
              for (int i = 0; i < n; i++) y[i] = Z[0][i] + acor[i];
              if (invalid_state(n, y)) break;
              rates(nt, rho, y, f, NULL);
              add_source(n, src, f);
              cnt[1]++;
            }
            for (int i = 0; i < n; i++) b[i] = fma(gamma, f[i], -fma(Z[1][i], rl1, acor[i]));
            orc_lu_solve(n, P, ipvt, inv, b);
            cnt[4]++;
            if (reuse && !jcur)
              for (int i = 0; i < n; i++) b[i] = b[i] * cscale;
            for (int i = 0; i < n; i++) acor[i] = acor[i] + b[i];
            double del = orc_wrms(n, b, w, L);
            if (!isfinite(del)) break;
            if (m > 0) {
              double rr = del / delp;
              crate = CRDOWN * crate;
              if (rr > crate) crate = rr;
            }
            double dcon = (del * (crate < 1.0 ? crate : 1.0)) / tq;
            if (dcon <= 1.0) {
              ok = 1;
              break;
            }
            if (m > 0 && del > RDIV * delp) break;
            delp = del;
          }
        }
      }
      if (!ok && reuse && tried && !jcur) {
        /* policy 1, B.6': Newton failed with a STALE matrix: same step, same h, fresh J and LU */
        retract(n, q, Z);
        forceP = 1;
        if (o->nstale) __atomic_fetch_add(o->nstale, 1ull, __ATOMIC_RELAXED);
        continue;
      }
      if (!ok) { /* B.6 Newton failure */
        forceP = 1;
        if (predicted) retract(n, q, Z);
        ncf++, cnt[6]++;
        etamax = 1.0;
        last = 0;
        if (ncf > mxncf) {
          for (int i = 0; i < n; i++) yout[i] = Z[0][i];
          return -1;
        }
        rescale(n, q, Z, ETACF);
        h = h * ETACF;
        continue;
      }
      /* B.5 error test */
      dsm = orc_wrms(n, acor, w, L) / cerr;
      const int injected = (o && o->inject_nef > 0 && nst + 1 == o->inject_step && nef < o->inject_nef);
      if (fixed || (dsm <= 1.0 && !injected)) break; /* accept (test hook: see orc_opts.inject_step) */
      retract(n, q, Z);
      nef++, cnt[5]++;
      etamax = 1.0;
      last = 0;
      forceP = 1; /* policy 1: the retry after an error-test failure uses a fresh matrix */
      if (nef == mxnef) {
        for (int i = 0; i < n; i++) yout[i] = Z[0][i];
        return -2;
      }
      if (nef <= 2) {
        double eta = eta_of(dsm, BIAS2, q + 1);
        if (eta < ETAMIN) eta = ETAMIN;
        if (nef == 2 && eta > ETAMXF) eta = ETAMXF;
        rescale(n, q, Z, eta);
        h = h * eta;
      } else if (q > 1) {
        ORC_EVENT(1);
        /* lower the order at t_{n-1}: xi_i = (tau_1 + ... + tau_i)/h */
        double s = 0.0;
        for (int i = 1; i <= q - 2; i++) {
          s = (i == 1) ? tau[1] : s + tau[i];
          xi[i] = s / h;
        }
        build_d(q - 2, xi, d);
        for (int j = 2; j <= q - 1; j++)
          for (int i = 0; i < n; i++) Z[j][i] = fma(-d[j], Z[q][i], Z[j][i]);
        q = q - 1;
        nqwait = q + 1;
        double Zpre[QMAX + 2][ORC_NMAX]; /* trace hook only: the lowered array on the scale h_used */
        if (tr)
          for (int j = 0; j <= QMAX; j++)
            for (int i = 0; i < n; i++) Zpre[j][i] = (j <= q) ? Z[j][i] : 0.0;
        rescale(n, q, Z, ETAMIN);
        if (tr) {
          double hd[ORC_TRACE_HEAD] = {1.0, t, h, (double)(q + 1), dsm, 0, 0, 0, 0, 0, -1.0, ETAMIN,
                                       h * ETAMIN, (double)q, (double)nef, (double)ncf};
          for (int j = q + 1; j <= QMAX; j++)
            for (int i = 0; i < n; i++) Zacc[j][i] = 0.0;
          for (int j = 0; j <= q; j++)
            for (int i = 0; i < n; i++) Zacc[j][i] = Z[j][i];
          trace_put(tr, hd, Zpre, Zacc);
        }
        h = h * ETAMIN;
      } else {
        ORC_EVENT(2);
        h = h * ETAMIN;
        for (int i = 0; i < n; i++) y[i] = Z[0][i];
        rates(nt, rho, y, f, NULL);
              add_source(n, src, f);
        cnt[1]++;
        for (int i = 0; i < n; i++) Z[1][i] = h * f[i];
        nqwait = 10;
        if (tr) {
          double hd[ORC_TRACE_HEAD] = {2.0, t, h / ETAMIN, 1.0, dsm, 0, 0, 0, 0, 0, 0.0, ETAMIN,
                                       h, 1.0, (double)nef, (double)ncf};
          for (int j = 2; j <= QMAX; j++)
            for (int i = 0; i < n; i++) Zacc[j][i] = 0.0;
          for (int j = 0; j <= 1; j++)
            for (int i = 0; i < n; i++) Zacc[j][i] = Z[j][i];
          trace_put(tr, hd, NULL, Zacc);
        }
      }
    }
    /* C. accept */
    for (int j = 0; j <= q; j++)
      for (int i = 0; i < n; i++) Z[j][i] = fma(l[j], acor[i], Z[j][i]);
    t = last ? dt : t + h;
    nst++;
    cnt[0]++;
    set_weights(n, Z[0], rtol, atol, w);
    if (tr) {
      for (int j = 0; j <= QMAX; j++)
        for (int i = 0; i < n; i++) Zacc[j][i] = (j <= q) ? Z[j][i] : 0.0;
      const double hd[ORC_TRACE_HEAD] = {0.0, t, h, (double)q, dsm, 0, 0, 0, 0, 0, 0.0, 1.0,
                                         h, (double)q, (double)nef, (double)ncf};
      for (int i = 0; i < ORC_TRACE_HEAD; i++) thead[i] = hd[i];
      if (last || nst == mxstep) trace_put(tr, thead, Zacc, Zacc);
    }
    if (last) break;
    if (nst == mxstep) {
      for (int i = 0; i < n; i++) yout[i] = Z[0][i];
      return -3;
    }
    /* D. select next step and order */
    double eta = 1.0;
    int action = 0; /* -1 lower, 0 keep, +1 raise */
    if (!fixed || tr) { /* (fixed-q hook: evaluated for the trace only, never applied -- see below) */
      nqwait--;
      if (etamax == 1.0) {
        if (nqwait < 2) nqwait = 2;
      } else {
        double etaq = eta_of(dsm, BIAS2, q + 1);
        if (nqwait != 0) {
          eta = etaq;
        } else {
          nqwait = 2;
          double etaqm1 = 0.0, etaqp1 = 0.0;
          if (q > 1) {
            double pm = rxi[1], sm = rxi[1];
            for (int i = 2; i <= q - 1; i++) {
              pm = pm * rxi[i];
              sm = sm + rxi[i];
            }
            double Em = orc_wrms(n, Z[q], w, L) / (pm * sm);
            etaqm1 = eta_of(Em, BIAS1, q);
            if (tr) thead[8] = Em;
          }
          if (q < QMAX && qS == q && ntau >= q) {
            double rq1 = h / (hs[q] + tau[q]); /* 1/xi_{q+1} */
            double pp = rxi[1], sp = rxi[1];
            for (int i = 2; i <= q; i++) {
              pp = pp * rxi[i];
              sp = sp + rxi[i];
            }
            pp = pp * rq1;
            sp = sp + rq1;
            double cq = FACT[q] * l[q];
            double rh = h / hS, rs = rh;
            for (int j = 1; j <= q; j++) rs = rs * rh; /* (h/h_S)^(q+1) */
            for (int i = 0; i < n; i++) vtmp[i] = fma(cq, acor[i], -(rs * S[i]));
            double Ep = orc_wrms(n, vtmp, w, L) / ((pp * sp) * FACT[q + 2]);
            etaqp1 = eta_of(Ep, BIAS3, q + 2);
            if (tr) thead[9] = Ep;
          }
          if (tr) thead[5] = etaq, thead[6] = etaqm1, thead[7] = etaqp1;
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
        double cq = FACT[q] * l[q];
        for (int i = 0; i < n; i++) S[i] = cq * acor[i];
        hS = h;
        qS = q;
      }
      if (fixed) { /* fixed-q, fixed-h hook: the selection above is reported, not applied */
        eta = 1.0;
        action = 0;
      }
    }
    /* E. apply (xi_i = hs[i]/h of B.1) */
    if (action == -1) {
      for (int i = 1; i <= q - 2; i++) xi[i] = hs[i] / h;
      build_d(q - 2, xi, d);
      for (int j = 2; j <= q - 1; j++)
        for (int i = 0; i < n; i++) Z[j][i] = fma(-d[j], Z[q][i], Z[j][i]);
      q = q - 1;
      nqwait = q + 1;
    } else if (action == +1) {
      for (int i = 1; i <= q - 1; i++) xi[i] = hs[i] / h;
      build_d(q - 1, xi, d);
      double cfac = l[q] * INVP[q + 1];
      for (int i = 0; i < n; i++) {
        double c = cfac * acor[i];
        Z[q + 1][i] = 0.0;
        for (int j = 2; j <= q + 1; j++) Z[j][i] = fma(d[j], c, Z[j][i]);
      }
      q = q + 1;
      nqwait = q + 1;
    }
    for (int i = 5; i >= 2; i--) tau[i] = tau[i - 1];
    tau[1] = h;
    if (ntau < 5) ntau++;
    etamax = ETAMAX;
    if (eta != 1.0) {
      rescale(n, q, Z, eta);
      h = h * eta;
    }
    if (tr) {
      thead[10] = (double)action, thead[11] = eta, thead[12] = h, thead[13] = (double)q;
      double Zend[QMAX + 2][ORC_NMAX];
      for (int j = 0; j <= QMAX; j++)
        for (int i = 0; i < n; i++) Zend[j][i] = (j <= q) ? Z[j][i] : 0.0;
      trace_put(tr, thead, Zacc, Zend);
    }
  }
  for (int i = 0; i < n; i++) yout[i] = Z[0][i];
  return nst;
}

/* ---- public entry points --------------------------------------------------------------- */
int orc_max_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

int orc_rates(const orc_net_desc *d, double rho, const double *y, double *f, double *J) {
  Net nt;
  int rc = net_init(&nt, d);
  if (rc) return rc;
  /* API order is (Y_0..Y_{N-1}, T); permute to the internal T-first order and back */
  const int n = nt.n, N = nt.N;
  double yi[ORC_NMAX] = {0}, fi[ORC_NMAX], Ji[ORC_NMAX * ORC_NMAX];
  int ext[ORC_NMAX]; /* internal index -> external index */
  ext[TI] = N;
  for (int i = 0; i < N; i++) ext[SP(i)] = i;
  for (int a = 0; a < n; a++) yi[a] = y[ext[a]];
  rates(&nt, rho, yi, fi, J ? Ji : NULL);
  for (int a = 0; a < n; a++) f[ext[a]] = fi[a];
  if (J)
    for (int a = 0; a < n; a++)
      for (int b = 0; b < n; b++) J[ext[a] * n + ext[b]] = Ji[a * n + b];
  return 0;
}

/* Same argument list as the library's burn_zones minus the stream (include/burnzones.h);
 * all pointers are host pointers.  nsteps[z] = accepted steps, or -1 (Newton failures),
 * -2 (error-test failures), -3 (MXSTEP), -4 (invalid input zone). */
int orc_burn(const orc_net_desc *d, int64_t nz, const double *rho, const double *T,
             const double *X, double dt, double rtol, double atol, double *T_out, double *X_out,
             int32_t *nsteps, const orc_opts *opts, uint64_t counters[8]) {
  Net nt;
  int rc = net_init(&nt, d);
  if (rc) return rc;
  if (nz < 0) return -2;
  if (!(dt > 0.0) || !(rtol > 0.0) || !(atol >= 0.0) || !isfinite(dt) || !isfinite(rtol) ||
      !isfinite(atol))
    return -4;
  if (nz > 0 && (!rho || !T || !X || !T_out || !X_out || !nsteps)) return -1;
  const int N = nt.N, n = nt.n;
  uint64_t tot[8] = {0};
  int nthreads = (opts && opts->nthreads > 0) ? opts->nthreads : orc_max_threads();
  (void)nthreads;
#pragma omp parallel num_threads(nthreads)
  {
    uint64_t cnt[8] = {0};
#pragma omp for schedule(dynamic, 64)
    for (int64_t z = 0; z < nz; z++) {
      double y0[ORC_NMAX], yout[ORC_NMAX];
      for (int i = 0; i < N; i++) y0[SP(i)] = X[(int64_t)i * nz + z] / nt.aion[i];
      y0[TI] = T[z];
      double srcv[ORC_NMAX];
      const int has_src = opts && opts->src_T && opts->src_X;
      if (has_src) {
        for (int i = 0; i < N; i++) srcv[SP(i)] = opts->src_X[(int64_t)i * nz + z] / nt.aion[i];
        srcv[TI] = opts->src_T[z];
      }
      Trace trc = {NULL, 0, n, 0};
      const int traced = (z == 0 && opts && opts->trace);
      if (traced) trc.buf = opts->trace, trc.cap = opts->trace_cap;
      int code = burn_zone(&nt, rho[z], y0, dt, rtol, atol, opts, has_src ? srcv : NULL, yout, cnt,
                           traced ? &trc : NULL);
      if (traced && opts->trace_n) *opts->trace_n = trc.count;
      if (code == -4) { /* invalid input: outputs = inputs */
        for (int i = 0; i < N; i++) X_out[(int64_t)i * nz + z] = X[(int64_t)i * nz + z];
        T_out[z] = T[z];
      } else {
        for (int i = 0; i < N; i++) X_out[(int64_t)i * nz + z] = nt.aion[i] * yout[SP(i)];
        T_out[z] = yout[TI];
      }
      nsteps[z] = code;
      if (code < 0) cnt[7]++;
    }
#pragma omp critical
    for (int c = 0; c < 8; c++) tot[c] += cnt[c];
  }
  (void)n;
  if (counters)
    for (int c = 0; c < 8; c++) counters[c] = tot[c];
  return 0;
}
