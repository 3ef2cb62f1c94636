/* bz_oracle.h -- CPU oracle for the per-zone nuclear burn.  TEST INFRASTRUCTURE ONLY.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
 * legs may call this.  It shares no code with the CUDA path (paper_1711_06203_b200/).
 *
 * What it computes (section 4: "do the entire ODE integration ... all
 * righthand side and Jacobian evaluations and the timestepping itself"; ref [33] VODE,
 * PAPER.md L184): for every zone independently, integrate
 *     dY_i/dt = sum_k D_ik R_k ,   dT/dt = (N_A MeV / c_v) sum_k Q_k R_k
 * over one hydro step dt with a variable-coefficient, variable-order (1..5) BDF in
 * Nordsieck form, Newton iteration on I - gamma*J with an analytic dense Jacobian and a
 * LINPACK-style dense LU (dgefa/dgesl).  The paper prints none of the formulas; the
 * algorithm ("BZ-BDF v1") is the reading recorded in DESIGN.md section 3, taken from
 * SURVEY.md section 8(c) C.1-C.2, and is followed here step by step in that notation.
 *
 * Parity status of the parts (pins live in tests/test_oracle_*.py, all -m "not gpu"):
 *   rate law, RHS, Jacobian (incl. every sign of the Y < 0 extension), LU/solve, exp/log, BDF
 *   coefficients, order of accuracy, the integrator as a whole (closed forms, invariants,
 *   brute-force implicit Euler, scipy Radau): pinned.
 *   Step/order machinery (tests/test_oracle_nordsieck.py): build_d against numpy's polyfromroots;
 *   the Nordsieck array after every accepted step, after both order changes of C.2-E, after the
 *   order reduction and the order-1 restart of C.2-B.5 = the array of the polynomial that
 *   interpolates the accepted values, rebuilt in exact rational arithmetic from the trace hook;
 *   E-, E+ and dsm against analytic derivatives (constant step) and against divided differences
 *   of the accepted values (variable steps); failure codes -1 (real inputs), -2, -3 (limits as
 *   parameters).  Each of these pins was checked to turn red under a perturbation of the line it
 *   covers (commit message of the pins).
 *   Model extensions: density exponents (closed form in rho, tests/test_urca9_like.py), analytic EOS
 *   (exact energy integral, tests/test_eos_cv.py), policy 1 (tests/test_oracle_reuse.py): pinned; 11 of
 *   12 perturbations of their lines turn a pin red.
 *   PARITY UNPINNED: only the VALUES of the heuristics constants (BIAS1..3, THRESH, ETAMAX, ETAMIN,
 *   ETAMXF, ETACF, NTOL, CRDOWN, RDIV, ADDON, SLIVER, the default limits; under policy 1 also CCMAX's
 *   value and the 2/(1 + gamma/gamma_P) scale of a stale solve, which moves the Newton iteration's path
 *   but not the corrector solution it converges to) -- any values pass the pins; they are fixed by
 *   DESIGN.md sections 3 and 12 only.
 */
#ifndef BZ_ORACLE_H
#define BZ_ORACLE_H
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define ORC_NMAX 32   /* max unknowns n = nspec + 1 */
#define ORC_KMAX 256  /* max reactions */

typedef struct {
  int32_t nspec, nreac;
  const double *aion;        /* [N]    mass numbers A_i                                  */
  const int32_t *reactant;   /* [K][3] reactant particle species ids, -1 unused          */
  const int32_t *stoich_id;  /* [K][4] species whose Y changes, -1 unused                */
  const double *stoich_dy;   /* [K][4] change per reaction event                         */
  const double *rate_A, *rate_n, *rate_B; /* [K] lambda = A T9^n exp(-B T9^(-1/3))       */
  const double *q_mev;       /* [K]    MeV per event                                     */
  double cv;                 /* erg/g/K                                                  */
  /* optional density exponents (weak rates that depend on rho, "the 9-isotope Urca
   * network"): lambda_k is multiplied by rho^rate_rho_exp[k] ON TOP of the rho^(m-1) of
   * the rate law, evaluated inside the exponent: arg_k += rate_rho_exp[k] * ln(rho).  NULL = none. */
  const double *rate_rho_exp; /* [K] or NULL */
  /* optional analytic equation of state for the specific heat ("supports arbitrary
   * equations of state").  zion != NULL selects it and `cv` is ignored:
   *   c_v(rho, T, Y) = 1.5 R (eos_extra + sum_i (1 + Z_i) Y_i) + 4 a T^3 / rho     [erg/g/K]
   * (ideal ions and electrons, radiation; R = 8.31446261815324e7 erg/mol/K, a = 7.565733250e-15
   * erg/cm^3/K^4).  eos_extra [mol/g]: the same sum over species that are not evolved (config 1's O16). */
  const double *zion;         /* [N] charges Z_i, or NULL */
  double eos_extra;
} orc_net_desc;

typedef struct {
  int32_t norm_lanes;  /* 1,2,4,8,16,32: association of the WRMS-norm sum */
  int32_t fixed_q;     /* test hook: 0 = adaptive; q>0 = fixed order, fixed step, no error test */
  double fixed_h;      /* test hook: the fixed step                                       */
  const double *z_init;/* test hook: [(fixed_q+1)][n] initial Nordsieck array (scaled by fixed_h) */
  int32_t nthreads;    /* OpenMP threads over zones; <=0 = runtime default                */
  /* constant per-zone source terms (SDC-style coupling): the system
   * integrated is dy/dt = f(rho, y) + s with dT/dt += src_T[z] [K/s] and
   * dY_i/dt += src_X[i][z] / A_i (src_X is a mass-fraction rate [1/s]).  NULL = no sources. */
  const double *src_T; /* [nz] or NULL */
  const double *src_X; /* [N][nz] or NULL (both or neither) */
  /* test hook (pins of C.2-B.5/D/E, tests/test_oracle_nordsieck.py): if trace != NULL, zone 0 writes
   * one record of ORC_TRACE_HEAD + 12*n doubles per event, at most trace_cap records, and the number
   * of events into *trace_n.  Record = {kind, t, h_used, q_used, dsm, eta_q, eta_qm1, eta_qp1, E-, E+,
   * action, eta, h_next, q_next, nef, ncf, Zacc[6][n], Zend[6][n]} with kind 0 = accepted step
   * (Zacc = Nordsieck array right after C at scale h_used, Zend = after E at scale h_next; t = the new
   * time), kind 1 = B.5 third error-test failure lowering the order and kind 2 = B.5 restart at
   * order 1 (Zend = the array the next attempt starts from, at scale h_next, expanded at the OLD time t;
   * kind 1: Zacc = the same array before its rescale by ETAMIN, at scale h_used).
   * Rows of Z are in the API order (Y_0..Y_{N-1}, T).  The hook only copies values out; with
   * fixed_q > 0 it also evaluates (but never applies) the estimators of C.2-D. */
  double *trace;
  int32_t trace_cap;
  int32_t *trace_n;
  /* limits of C.2 as call parameters (the library's bz_set_limits; CVODE exposes the same three):
   * accepted steps per zone (code -3), error-test failures per step (code -2), Newton failures per
   * step (code -1).  <= 0 = the defaults MXSTEP 20000, MXNEF 7, MXNCF 10. */
  int32_t mxstep, mxnef, mxncf;
  /* test hook: the attempts of accepted step number inject_step (1-based) fail the error test until
   * inject_nef failures have been counted, whatever dsm is.  Natural third failures come after two
   * step reductions that leave the high Nordsieck rows below rounding, where the order reduction of
   * C.2-B.5 cannot be observed; injected ones keep them large (tests/test_oracle_nordsieck.py). */
  int32_t inject_step, inject_nef;
  /* Newton-matrix policy.  0 ("BZ-BDF v1", the default and the parity reference of burn_zones): a
   * fresh Jacobian and LU on every attempt.  1 ("BZ-BDF v2", the library's bz_set_policy(net, 1);
   * VODE's reuse, ref. [33] PAPER.md:L184): the LU of
   * P = I - gamma_P J is kept; an attempt factorises (with a fresh J at the prediction) only if there is
   * no P yet, or |gamma/gamma_P - 1| > 0.3, or 20 steps were accepted since, or a failure asked for
   * it; otherwise it evaluates f only and every correction solved with the stale matrix is multiplied
   * by 2/(1 + gamma/gamma_P).  Evaluation (part of the contract): gl = gamma_P * l_1; drift test
   * |h - gl| > 0.3 * gl; scale (2 * gl)/(gl + h).  A Newton failure with a stale matrix repeats the attempt at the same h
   * with a fresh one (counted in *nstale, not in ncfn); any B.5 or B.6 failure forces a fresh matrix
   * for the retry (a reduced step of 0.7-0.74 h would not trip the drift test by itself). */
  int32_t policy;
  unsigned long long *nstale; /* test aid: stale-matrix retries, summed over zones; or NULL */
} orc_opts;
#define ORC_TRACE_HEAD 16

/* counters[8] = {nst, nrhs, njac, nlu, nsolve, netf, ncfn, nfailzones} summed over zones */
int orc_burn(const orc_net_desc *d, int64_t nz, const double *rho, const double *T,
             const double *X /*[N][nz]*/, double dt, double rtol, double atol,
             double *T_out, double *X_out, int32_t *nsteps, const orc_opts *opts,
             uint64_t counters[8]);

/* pieces exposed for the pins */
int orc_rates(const orc_net_desc *d, double rho, const double *y /*[n]*/, double *f /*[n]*/,
              double *J /*[n*n] row-major or NULL*/);
double orc_exp(double x);
double orc_log(double x);
/* a: [n*n] row-major, overwritten by LU (multipliers +l_ik below, U above, on the diagonal
 * the pivots); inv[n] = 1/pivot; ipvt[n].  returns 0, or k+1 if pivot k is exactly zero. */
int orc_lu_factor(int n, double *a, int32_t *ipvt, double *inv);
void orc_lu_solve(int n, const double *a, const int32_t *ipvt, const double *inv, double *b);
/* l[0..q], for step h and history tau[1..5] (tau[0] unused) */
void orc_bdf_coeffs(int q, double h, const double *tau, double *l);
double orc_wrms(int n, const double *v, const double *w, int lanes);
/* d(x) = x^2 prod_{i=1..cnt} (x + xi[i]) = sum_j d[j] x^j (xi[0] unused; d has 8 entries) */
void orc_build_d(int cnt, const double *xi, double *d);
int orc_max_threads(void);
/* test aid: number of row interchanges orc_lu_factor has performed since the last reset */
unsigned long long orc_interchanges(int reset);
/* test aid: {interchanges, order lowered after a 3rd error-test failure, order-1 restart} */
void orc_event_counts(int reset, unsigned long long out[3]);

#ifdef __cplusplus
}
#endif
#endif
