/* burnzones.h -- C ABI of libburn: the per-zone nuclear burn on one B200 (sm_100a).
 *
 * The operation (section 4): "do the entire ODE integration on the GPU, i.e.,
 * the data for a patch of zones is passed to the GPU, all righthand side and Jacobian
 * evaluations and the timestepping itself is done on the GPU, and once the burning in all
 * zones is completed, we access the data as needed"; the integrator is VODE (ref. [33],
 * PAPER.md L184); "rates and integration strategy are decoupled" (L83).  The call list is
 * BASELINE.json:north_star's: net_create(rates, Q-values, isotope masses),
 * burn_zones(rho[], T[], X[][], dt, rtol, atol, out T[], out X[], out nsteps[], stream),
 * net_destroy.  The exact model and algorithm ("BZ-BDF v1") are DESIGN.md section 3.
 *
 * Conventions
 *   - plain C, no exceptions, no abort; every call returns 0 or a negative bz_status.
 *   - "HOST" / "DEVICE" says where a pointer must point.  DEVICE arrays and the stream are
 *     owned by the caller (PyTorch allocates them); the library owns the bz_net handle, its
 *     device-side tables and its scratch (work-queue counter, counters, staging buffers).
 *   - layout: structure of arrays, species-major, zone index fastest:  X[i*nz + z].
 *     Zone order is the grid's x-fastest order but the library attaches no meaning to it.
 *   - burn_zones only enqueues work on `cuda_stream` and returns; it never synchronises the
 *     device.  Outputs are valid after the caller synchronises the stream.
 *   - exact aliasing T_out == T and X_out == X is allowed (each zone is read completely before
 *     it is written); partial overlap is undefined.
 *   - there is no CPU fallback: without a CUDA device every compute call returns BZ_ERR_CUDA.
 */
#ifndef BURNZONES_H
#define BURNZONES_H
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct bz_net bz_net; /* opaque, owned by the library */

typedef enum {
  BZ_OK = 0,
  BZ_ERR_NULL = -1,    /* a required pointer is NULL                                          */
  BZ_ERR_SIZE = -2,    /* nspec not in 1..31, nreac not in 1..256, nz < 0                     */
  BZ_ERR_NETWORK = -3, /* species id out of range, A_i <= 0, cv <= 0, rate_A <= 0, non-finite
                          coefficient, reaction without reactant, repeated stoichiometry id    */
  BZ_ERR_SCALAR = -4,  /* dt <= 0, rtol <= 0, atol < 0, or non-finite                         */
  BZ_ERR_CUDA = -5,    /* CUDA runtime error; the cudaError_t is in bz_last_cuda_error()      */
  BZ_ERR_NOMEM = -6,   /* host or device allocation failed                                    */
  BZ_ERR_UNSUPPORTED = -7, /* the combination has no kernel (bz_set_policy 1 on a network with density
                              exponents or an EOS)                                                 */
  BZ_ERR_DEVICE = -8   /* the handle was created on another device than the current one        */
} bz_status;

/* Network descriptor.  All pointers are HOST pointers and are
 * copied; the caller may free them when net_create returns.
 *   rate law   lambda_k = rate_A * T9^rate_n * exp(-rate_B / T9^(1/3)),  T9 = T / 1e9
 *              R_k = lambda_k * rho^(m_k - 1) * prod_{p in reactant[k]} Y_p / prod_i nu_ik!
 *   ODEs       dY_i/dt = sum_k stoich_dy[k][.] R_k ;  dT/dt = (N_A MeV / cv) sum_k q_mev[k] R_k
 */
typedef struct {
  int32_t nspec, nreac;      /* N (1..31), K (1..256)                                          */
  const double *aion;        /* [N]    mass numbers A_i ("isotope masses"); Y_i = X_i / A_i    */
  const int32_t *reactant;   /* [K][3] species id of each reactant particle, -1 = unused;
                                        identical particles repeated (3-alpha = {0,0,0})       */
  const int32_t *stoich_id;  /* [K][4] species whose Y changes, -1 = unused, ids distinct      */
  const double *stoich_dy;   /* [K][4] net change of Y per reaction event                      */
  const double *rate_A, *rate_n, *rate_B; /* [K]                                              */
  const double *q_mev;       /* [K]    Q-values, MeV per reaction event                        */
  double cv;                 /* specific heat, erg g^-1 K^-1, constant                         */
  const double *rate_rho_exp; /* [K] or NULL: optional density exponents e_k of weak rates -- lambda_k
                                is multiplied by rho^e_k ON TOP of the rho^(m_k - 1) of the rate law
                                (electron captures grow with density, beta decays are blocked by it:
                                "the 9-isotope Urca network").  Evaluated
                                inside the exponent: arg_k += e_k * ln(rho).  Finite values; NULL = none.
                                Networks that carry it run on the generic cooperative kernel.            */
  const double *zion;        /* [N] or NULL: charges Z_i.  Non-NULL selects an analytic equation of state for
                                the specific heat, evaluated with every right-hand side (
                                "supports arbitrary equations of state"), and
                                `cv` is ignored:
                                  c_v(rho,T,Y) = 1.5 R (eos_extra + sum_i (1+Z_i) Y_i) + 4 a T^3 / rho
                                (ideal ions and electrons + radiation; R = 8.31446261815324e7 erg/mol/K,
                                a = 7.565733250e-15 erg/cm^3/K^4).  Z_i >= 0, finite.  Generic kernel only. */
  double eos_extra;          /* mol/g, >= 0: sum (1+Z_i) Y_i over species that are NOT evolved (read only
                                when zion != NULL)                                                        */
} bz_net_desc;

/* Validate, flatten and upload a network.  *out receives the handle.  A handle belongs to the
 * device that is current when net_create runs (its tables, scratch, grid size and shared-memory
 * opt-in live there): create one handle per device; every later call on it checks cudaGetDevice
 * and returns BZ_ERR_DEVICE, enqueuing nothing, if another device is current. */
int net_create(const bz_net_desc *desc, bz_net **out);

/* Integrate every zone's network over [0, dt] (steps a1-a9 of DESIGN.md section 2).
 *   nz             number of zones (0 is a no-op)
 *   rho, T         DEVICE [nz]       density g/cc, temperature K (inputs)
 *   X              DEVICE [N][nz]    mass fractions of the N evolved species (input)
 *   dt, rtol, atol burn interval (s); relative tolerance; absolute tolerance on Y (mol/g)
 *   T_out, X_out   DEVICE [nz], [N][nz]   results
 *   nsteps         DEVICE [nz] int32: accepted BDF steps, or a per-zone failure code
 *                    -1  more than 10 Newton failures on one step
 *                    -2  7 error-test failures on one step
 *                    -3  20000 steps taken without reaching dt
 *                    -4  invalid input zone (non-finite, rho <= 0 or T <= 0): outputs = inputs
 *                  failed zones hold the last accepted state; they do not fail the call.
 *   cuda_stream    cudaStream_t (as void*) on which all work is enqueued
 * A handle owns one work-queue counter, one set of counters and, under the default schedule, the buffers of
 * the queue's cost order (24 bytes per zone, allocated at the first call and when a batch is larger than any
 * before: bz_set_schedule): calls on the SAME handle must be ordered (same stream, or synchronised); use one
 * handle per concurrent stream.
 */
int burn_zones(const bz_net *net, int64_t nz, const double *rho, const double *T, const double *X,
               double dt, double rtol, double atol, double *T_out, double *X_out, int32_t *nsteps,
               void *cuda_stream);

/* The burn with constant per-zone source terms: the coupling the paper's codes use when the burn is
 * driven by an SDC hydro update ("SDC ... coupling of hydro and reactions", section
 * 3.2): the advective source is held constant over the burn and the system integrated is
 *     dT/dt = f_T(rho, y) + src_T[z],      dY_i/dt = f_i(rho, y) + src_X[i][z] / A_i .
 *   src_T   DEVICE [nz]     temperature source, K/s
 *   src_X   DEVICE [N][nz]  mass-fraction sources, 1/s (species-major like X)
 * Both NULL: identical to burn_zones (bit for bit).  Exactly one NULL: BZ_ERR_NULL.  The sources
 * enter every right-hand-side evaluation as one rounded addition after the network's own sums;
 * the Jacobian is unchanged.  A zone with a non-finite source ends with code -4.  All other
 * arguments, the failure codes and the execution rules are those of burn_zones.  Served by both
 * kernels.  (DESIGN.md section 10.) */
int burn_zones_src(const bz_net *net, int64_t nz, const double *rho, const double *T, const double *X,
                   const double *src_T, const double *src_X, double dt, double rtol, double atol,
                   double *T_out, double *X_out, int32_t *nsteps, void *cuda_stream);

/* The same burn with HOST arrays (pinned memory recommended): copies inputs to library-owned device
 * staging, burns, copies the three outputs back, and returns without synchronising; everything is
 * ordered after the earlier work of `cuda_stream`, and `cuda_stream` is complete only when the last
 * result has arrived.  Batches of >= 2^23 zones are PIPELINED in chunks of >= 2^22 zones (at most 8):
 * chunk c's inputs travel on a library-owned copy stream while chunk c-1 burns on `cuda_stream` and
 * chunk c-2's results travel back on a second copy stream (zones are independent: the results are
 * those of burn_zones; bz_get_counters returns the totals over all chunks).  Chunks are large on
 * purpose: each is its own launch and pays the serial tail of its slowest zone.  This is the
 * end-to-end path bench.py times. */
int burn_zones_host(bz_net *net, int64_t nz, const double *rho, const double *T, const double *X,
                    double dt, double rtol, double atol, double *T_out, double *X_out,
                    int32_t *nsteps, void *cuda_stream);

int net_destroy(bz_net *net);

/* The burn for callers that may not allocate device memory (a harness that forbids cudaMalloc, a
 * tight serving loop): no handle, no net_create.  One call validates and flattens `desc` (HOST
 * pointers, as net_create), copies its tables into a library-owned STATIC device array of
 * BZ_STATIC_SCRATCH_BYTES (32 KiB, held by every GPU that loads the library until the process
 * exits), clears the work-queue counter that also lives there, and launches the generic
 * cooperative kernel (burn_coop, any network).  It calls no cudaMalloc, cudaFree or other
 * allocating routine, on the host side it uses fixed-size buffers.  All other arguments, the
 * per-zone failure codes, the arithmetic and the results are those of burn_zones on a handle with
 * bz_select_kernel(net, 1) -- bit for bit; norm lanes = 4, 8, 16 or 32, the smallest >= nspec + 1.
 *   Limit: the tables must fit the static array.  nspec <= 31 and nreac <= 256 (the ABI's own
 *   limits) always do; anything larger returns BZ_ERR_SIZE and enqueues nothing.  nz is unlimited
 *   (the scratch does not grow with it).
 *   Sharing: every call on a device uses the SAME array, which keeps the previous call's contents;
 *   the call itself re-uploads the tables and zeroes the queue on `cuda_stream`, so calls ordered
 *   on one stream are safe, while calls that overlap on the GPU (two streams, two threads) RACE on
 *   it and give undefined results -- serialise them, or use handles (net_create) instead.
 *   The table upload is a cudaMemcpyAsync from pageable host memory: not capturable in a CUDA graph. */
#define BZ_STATIC_SCRATCH_BYTES 32768
int burn_zones_static(const bz_net_desc *desc, int64_t nz, const double *rho, const double *T,
                      const double *X, double dt, double rtol, double atol, double *T_out,
                      double *X_out, int32_t *nsteps, void *cuda_stream);

/* Totals over the zones of the most recent burn_zones on this handle:
 * out[8] = {nst, nrhs, njac, nlu, nsolve, netf, ncfn, nfailzones} (HOST).  Synchronises
 * `cuda_stream` (it has to read the device counters). */
int bz_get_counters(const bz_net *net, void *cuda_stream, uint64_t out[8]);

/* Association of the WRMS-norm sum used by the kernel selected for this network
 * (DESIGN.md 3.6): 1, 4, 8, 16 or 32 interleaved partial sums combined by an xor butterfly.
 * Returns the lane count (>0) or a negative bz_status. */
int bz_norm_lanes(const bz_net *net);

/* Kernel selection: kind 0 = automatic (the network-specialised 4-lanes-per-zone kernel if the
 * topology has one compiled in, else the generic cooperative kernel), 1 = always the generic
 * cooperative kernel, 3 = the specialised quad kernel (falls back to the cooperative kernel when
 * the topology has none); other values: BZ_ERR_SIZE.  Both follow the same arithmetic; only
 * bz_norm_lanes differs. */
int bz_select_kernel(bz_net *net, int kind);

/* Zone scheduling (step a2, "a lot of thread divergence due to the widely differing thermodynamic
 * conditions").  A global work queue: a lane group that finishes its zone fetches the next
 * one, so co-resident zones never wait for the slowest of a fixed batch.
 *   kind 2 (default): the queue hands the zones out by decreasing a-priori COST KEY:
 *          |sum_k Q_k R_k| / T at the initial state, the relative heating rate up to common factors, from one
 *          right-hand side per zone in a kernel of its own, then one device radix sort of (key, index) pairs
 *          on the key's upper 16 bits -- both inside the burn call, on its stream.  Dear zones start first
 *          and zones of similar cost run side by side.  Config 4: 78.6 -> 46.2 ms per call; config 3: 1 958 ->
 *          1 932 ms.  Needs 24 bytes per zone of device memory, owned by the handle, allocated at
 *          the first call and when a batch is larger than any before (those calls synchronise the stream); if
 *          that memory is not to be had, if nz >= 2^31, or if the grid takes all zones at once, the call
 *          burns in index order.  burn_zones_static never orders (it allocates nothing).
 *   kind 0: the queue hands the zones out in index order.
 *   kind 1: static round-robin assignment (group g burns zones g, g + G, g + 2G, ...), kept only so that the
 *          benefit of the queue can be MEASURED (bench.py --static-schedule).
 * Every zone's result is bit-identical under all three; only the time differs.  Other kinds: BZ_ERR_SIZE. */
int bz_set_schedule(bz_net *net, int kind);

/* A caller's own ORDER for the work queue, instead of the library's cost key (e.g. the step counts of the
 * previous hydro step's burn, which the library cannot know).  order: DEVICE pointer to nz int64 entries, a
 * permutation of 0 .. nz-1 -- the q-th zone taken from the queue is zone order[q] -- or NULL (with nz = 0) to
 * return to the handle's schedule.  The
 * library keeps the pointer, not a copy: the array is the caller's and must stay valid and unchanged until
 * the burns that use it have completed; it applies to every later burn_zones / burn_zones_src call of this
 * handle, whose nz must equal the nz given here (else BZ_ERR_SIZE); burn_zones_host and the static schedule
 * refuse it (BZ_ERR_UNSUPPORTED); burn_zones_static never uses it.  Zones are independent, so every zone's
 * result is bit-identical whatever the order, and outputs stay at the zone's own index; only the time
 * changes: zones that take a similar number of steps and start together stay in phase, and a warp's
 * attempt then runs the rare paths (second Newton iteration, order change, rescale) for fewer of its zones
 * at a time.  Config 3, order = zones by decreasing step count of a previous burn of the same batch:
 * 1 958 -> 1 742 ms, against 1 932 ms with the library's a-priori key.
 * The entries are not checked on the host; an entry outside [0, nz) is ignored by the kernel, and a zone that
 * no entry names is not burned (its outputs are left untouched).
 * Errors: BZ_ERR_NULL (net), BZ_ERR_SIZE (nz < 0, or order NULL with nz != 0). */
int bz_set_zone_order(bz_net *net, const int64_t *order, int64_t nz);

/* Newton-matrix policy ("we ported our workhorse ODE integrator (VODE [33])",
 * PAPER.md:L119, and VODE reuses its factorised Newton matrix, ref. [33] L184).
 *   kind 0 (default, "BZ-BDF v1", the parity reference of BASELINE.json): a fresh Jacobian and LU on
 *          every step attempt.
 *   kind 1 ("BZ-BDF v2"): the LU of P = I - gamma_P J is kept; an attempt evaluates J
 *          and factorises only if there is no matrix yet, |gamma/gamma_P - 1| > 0.3, 20 steps were
 *          accepted since, or a failure asked for it; corrections solved with the kept matrix are
 *          scaled by 2/(1 + gamma/gamma_P); a Newton failure with a kept matrix repeats the attempt at
 *          the same step size with a fresh one.  About 12x fewer factorisations on the alpha-chain
 *          configs at the same step count.  Results are bit-identical to the oracle's policy 1 (not
 *          to policy 0: the two differ at the level of the integration tolerance).  Validated on the
 *          smooth networks (configs 1-4); on config 5 it loses accuracy on trace species.
 * Served by both kernels for the plain model; a network that carries density exponents or an EOS
 * (rate_rho_exp, zion) has no kept-matrix instantiation: burn_zones then returns BZ_ERR_UNSUPPORTED.
 * burn_zones_static always uses kind 0. */
int bz_set_policy(bz_net *net, int kind);

/* Limits behind the per-zone failure codes: accepted steps (-3), error-test failures on one step
 * (-2), Newton failures on one step (-1).  0 keeps the default (20000, 7, 10); negative: BZ_ERR_SIZE.
 * (CVODE exposes the same three; DESIGN.md 3.8 reading s29.) */
int bz_set_limits(bz_net *net, int32_t mxstep, int32_t mxnef, int32_t mxncf);

/* Name of the kernel variant burn_zones launches for this network (static string). */
const char *bz_kernel_name(const bz_net *net);

/* Last cudaError_t seen by this thread inside the library (0 = cudaSuccess). */
int bz_last_cuda_error(void);

/* FP64 peak probe: runs a DFMA-chain kernel on every SM for `iters` iterations of 8x32
 * independent fused multiply-adds per thread and returns the measured TFLOP/s (FMA = 2) in
 * *tflops and the elapsed milliseconds in *ms.  Synchronises the stream.  Used by bench.py to
 * report the denominator of the roofline. */
int bz_fp64_peak_probe(int64_t iters, void *cuda_stream, double *tflops, double *ms);

#ifdef __cplusplus
}
#endif
#endif /* BURNZONES_H */
