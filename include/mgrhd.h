/* mgrhd.h -- C ABI of the B200-native per-cell implicit matter-radiation source update
 * of arXiv 2407.18304 (He, Wibking & Krumholz), Section 3, PAPER.md:373-467 (Eq. 37-52),
 * with the group-mean opacities of Section 2.2 (Eq. 17-31).
 *
 * One call of mgrhd_source_update() advances every cell of a structure-of-arrays state from
 * the post-explicit state U^(t) to U^(t+1) by solving Eq. 37-40 with the paper's inner Newton
 * iteration on x = (E_gas, R_1..R_Nq) (Eq. 41-50; arrowhead Jacobian of Eq. 48 eliminated in
 * O(Nq)) and outer iteration on the lagged (v, F_g) (Eq. 51-52).
 *
 * All arithmetic is IEEE double precision on the device.  There is no CPU fallback: every
 * entry point that computes returns MGRHD_ERR_CUDA when no CUDA device can be used.
 *
 * Conventions (energy-density units; 4*pi/c never appears):
 *   x = h nu/(k_B T);  Bt_g = 4 pi B_g/c = a_R T^4 [Y(x_g+) - Y(x_g-)],
 *   Y(x) = (15/pi^4) int_0^x t^3/(e^t-1) dt  (Eq. 11 applied to the Planck function).
 *   chi_{0,g-} = rho * kappa_scale * kappa_lo[g] (absorption coefficient, 1/length), Eq. 19.
 *   C_v = rho k_B/((gamma-1) mean_mass) (volumetric), T = (E_gas - |rho v|^2/(2 rho))/C_v.
 *   Conserved by construction: E_gas + (c/c_hat) sum_g E_g and
 *   rho v + (c c_hat)^-1 sum_g F_g.
 */
#ifndef MGRHD_H
#define MGRHD_H

#ifdef __cplusplus
extern "C" {
#endif

#define MGRHD_MAX_GROUPS 64   /* largest Nq accepted (BASELINE.json config 5) */
#define MGRHD_HIST 64         /* iteration histograms are clamped to this many bins */

enum {
  MGRHD_OK = 0,
  MGRHD_ERR_ARG = -1,        /* null pointer, Nq out of range, ncells < 0, bad enum value      */
  MGRHD_ERR_RANGE = -2,      /* dt <= 0, c <= 0, c_hat <= 0 or c_hat > c, non-positive units or opacities */
  MGRHD_ERR_EDGES = -3,      /* edges not strictly ascending, negative, or NaN                  */
  MGRHD_ERR_ALPHA = -4,      /* alpha != 0 (or opacity_kind 2) in a group whose edge is 0 or +inf (Eq. 19, 20 undefined) */
  MGRHD_ERR_CUDA = -5,       /* CUDA runtime failure; mgrhd_last_error() has the text           */
  MGRHD_ERR_SIZE = -6        /* mgrhd_source_update_static: the launch needs more scratch than the static array holds */
};

typedef struct mgrhd_ctx mgrhd_ctx; /* opaque; created by mgrhd_init, destroyed by mgrhd_free */

/* Physical constants in the caller's unit system (independent inputs). */
typedef struct {
  double a_rad;      /* radiation constant a_R                       */
  double k_B;        /* Boltzmann constant                           */
  double h_planck;   /* Planck constant                              */
  double mean_mass;  /* mean particle mass mu*m_H                    */
  double gamma;      /* adiabatic index; C_v = rho k_B/((gamma-1) mean_mass) */
} mgrhd_units;

/* Opacity model and iteration controls.  HOST pointers, copied by mgrhd_init. */
typedef struct {
  const double *kappa_lo;  /* [Nq] specific opacity at each group's LOWER edge (Eq. 19)        */
  const double *alpha;     /* [Nq] in-group power-law slope alpha_{chi0,g}; 0 => PC (Eq. 17)   */
  int closure;             /* 0 = Levermore/M1, 1 = Eddington P = E/3 I (:603)  */
  int spectrum;            /* 0 = PPL fixed slope alpha_Q = -1 (the paper's favoured method);
                              1 = PPL free slope: alpha_B,g and alpha_E,g refitted at every Newton evaluation from
                              the group integrals B_g(T) and E_g^(t) + R_g + S_g by Eq. A1-A2,
                              both means from Eq. 30                                           */
  double newton_tol;       /* epsilon of Eq. 49 (paper default 1e-11)            */
  int newton_maxit;        /* cap on Newton steps per outer trip (paper silent; 50)            */
  int outer_maxit;         /* cap on outer trips (paper silent; 50)                            */
  double outer_tol;        /* 1e-13 of PAPER.md:465                                            */
  int outer_stop;          /* 0 = paper rule only; 1 = also |dF_g|<=rel*|F_g|, |d rho v|<=rel*|rho v|.
                              The "paper rule" is read as  sum_g |dW_g| (c_hat/c) dt <= outer_tol * max(sum_g |R_g|, E_tot):
                              a deviation from the literal text of PAPER.md:465 ("below 1e-13 sum R_g AND 1e-13 E_tot",
                              i.e. the smaller of the two), which cannot be met at equilibrium where sum_g R_g -> 0
                              (reading S10).                                                              */
  double outer_rel_tol;    /* rel of outer_stop == 1 (1e-12)                                   */
  /* ---- opacities that depend on the gas temperature: evaluated at every trial T of the Newton iteration ---- */
  int opacity_kind;        /* 0 = the table (kappa_lo, alpha) above, independent of T;
                              1 = kappa_lo[g] (T/T_ref)^p_T with the same alpha ("chi_g (T/T_0)^{3/2}");
                              2 = ln kappa tabulated at the Nq+1 group EDGES on a uniform grid in ln T (lnk_edge below):
                                  linear interpolation of ln kappa in ln T, end values outside the grid; the in-group
                                  slope alpha_g follows from the two edge values of the group, Eq. 20.
                                  kappa_lo and alpha are ignored (may be NULL); every edge must be finite and > 0.  */
  double T_ref, p_T;       /* opacity_kind 1                                                                        */
  int NT;                  /* opacity_kind 2: number of table temperatures (>= 1)                                   */
  double lnT0, dlnT;       /*                 T_j = exp(lnT0 + j dlnT), j = 0..NT-1                                 */
  const double *lnk_edge;  /*                 [Nq+1][NT] HOST, copied: ln of the specific opacity at edge e, temperature j */
  int outer_mode;          /* 0 = the paper's outer stage: the velocity in Eq. 51 is the lagged one, a fixed-point
                              iteration that contracts only while the radiation inertia q = (4/3) sum_g E_g/(rho c c_hat) is
                              small;
                              1 = "variant L" (not in the paper): the velocity in Eq. 51 is the NEW one, so
                              Eq. 51-52 are one 3x3 linear system for v^(t+1) per outer trip.  Same converged state; converges
                              for q >~ 1 (radiation-dominated cells, literal units) where mode 0 diverges.  General kernel.  */
} mgrhd_opacity_model;

/* Cell state, structure of arrays, float64, cell index fastest.  In mgrhd_source_update all
 * pointers are DEVICE pointers owned by the caller; mom, Egas, Erad, Frad are updated in
 * place, rho, kappa_scale and Srad are read only.  Arrays must not alias one another. */
typedef struct {
  const double *rho;         /* [n]      gas density                                           */
  double *mom[3];            /* [n] each rho v                                                 */
  double *Egas;              /* [n]      gas TOTAL energy density (internal + kinetic), Eq. 12 */
  double *Erad;              /* [Nq][n]  group radiation energy density E_g                    */
  double *Frad[3];           /* [Nq][n]  each: group radiation flux F_g^i                      */
  const double *kappa_scale; /* [n] per-cell multiplier on kappa_lo, or NULL (= 1)             */
  const double *Srad;        /* [Nq][n]  optional source term S_g of Eq. 41: energy density added to
                                group g during this update (e.g. stellar sources), or NULL (= 0).  Read only.
                                E_g^(t+1) = E_g^(t) + R_g + S_g, E_tot of Eq. 50 includes sum_g S_g,
                                and E_gas + (c/c_hat) sum_g (E_g - S_g) is conserved to round-off.                  */
} mgrhd_state;

/* Per-call diagnostics, accumulated on the device since the last mgrhd_reset_stats(). */
typedef struct {
  long long n_cells;                   /* cells processed                                       */
  long long n_newton_unconverged;      /* inner loops that hit newton_maxit                     */
  long long n_outer_unconverged;       /* cells that hit outer_maxit                            */
  long long n_T_nonpositive_steps;     /* Newton steps halved to keep T > 0, + invalid inputs   */
  long long n_chiF_guard;              /* cell-groups whose Eq. 27 denominator underflowed      */
  long long n_denominator_nonpositive; /* cell-groups with 1 + c_hat chi_F dt <= 0              */
  long long newton_evals_total;        /* residual evaluations (Eq. 41), summed over cells      */
  long long outer_trips_total;         /* outer trips, summed over cells                        */
  long long flops;                     /* algorithmic FP64 flops (0 unless counting is on)      */
  long long newton_hist[MGRHD_HIST];   /* per-cell residual evaluations (clamped)               */
  long long outer_hist[MGRHD_HIST];    /* per-cell outer trips (clamped)                        */
} mgrhd_stats;

/* Create a context for one group structure / unit system / opacity model.
 *   group_edges [Nq+1] HOST: nu_{g-}, ascending, >= 0; the last may be +inf.
 *   1 <= Nq <= MGRHD_MAX_GROUPS.  The context copies everything it needs (tables go to
 *   constant memory at launch); it uses the CUDA device current at the time of the call.
 * Which kernel runs: the fixed-slope spectrum with opacity_kind 0 or 1 and outer_mode 0 takes the tuned kernel
 * (L lanes per cell); the free-slope spectrum, opacity_kind 2 and outer_mode 1 take the general
 * kernel (one warp per cell, lane = group), which has a cell's groups side by side in a warp.
 * Returns MGRHD_OK and *out, or a negative error (and *out = NULL). */
int mgrhd_init(mgrhd_ctx **out, const double *group_edges, int Nq,
               const mgrhd_units *units, const mgrhd_opacity_model *model);

/* One implicit source update (Eq. 37-52) of `ncells` cells, in place, with dt = theta*Delta t
 * (PAPER.md:389), speed of light c and reduced speed of light c_hat <= c (Eq. 34).
 * Stream-ordered on `cuda_stream` (a cudaStream_t, NULL = default stream), asynchronous:
 * no host synchronisation, no allocation (one 256-byte memset of the work counter and one kernel
 * are enqueued).  ncells == 0 is a no-op.  A cell's result depends on that cell alone: results are
 * bit-identical from call to call and for any partition of the cells into calls.  Per-cell numerical
 * failures never abort; they are counted in mgrhd_stats.  A context owns one scratch buffer:
 * at most ONE mgrhd_source_update per context may be in flight at a time (calls on the same
 * stream are naturally serialised; use one context per stream for concurrent updates). */
int mgrhd_source_update(mgrhd_ctx *ctx, const mgrhd_state *state_dev, long long ncells,
                        double dt, double c, double c_hat, void *cuda_stream);

/* The same update for a state held in HOST memory (pinned or pageable): the cells are cut
 * into slabs that are copied to the device, updated and copied back on alternating streams,
 * so copies overlap kernels.  Synchronous: returns when the host arrays hold U^(t+1).
 * Scratch device memory (three slabs of up to 512 MB, sized to the largest call so far) is owned by the context and reused. */
int mgrhd_source_update_host(mgrhd_ctx *ctx, const mgrhd_state *state_host, long long ncells,
                             double dt, double c, double c_hat);

/* Explicit radiation transport of Eq. 34 in one dimension:
 *   dst.E_g += w_dt * [-(c_hat/c) dF_g^x/dx](src),   dst.F_g^i += w_dt * [-c c_hat dP_g^{xi}/dx](src)
 * for the nx cells of a row (cell index = position along x, spacing dx), every group; the gas fields have no
 * transport term.  The paper defers the discretisation to Paper II: here piecewise-constant states and local
 * Lax-Friedrichs interface fluxes with the signal speed c_hat, P_g from the context's closure (S22).
 * bc: 0 periodic, 1 zero-gradient.  src and dst are DEVICE states that must not alias; only Erad and Frad of
 * dst are touched.  Stream-ordered, asynchronous, one kernel. */
int mgrhd_transport_add(mgrhd_ctx *ctx, const mgrhd_state *src_dev, const mgrhd_state *dst_dev, long long nx,
                        double dx, double w_dt, double c, double c_hat, int bc, void *cuda_stream);

/* One two-stage IMEX step of Eq. 35-36 of a 1-D row, in place in U_dev (U^n -> U^(n+1)):
 *   stage 1: U* = U^n + dt T(U^n);  U^(n+1/2) = U* + dt S(U^(n+1/2))       (mgrhd_source_update, theta = 1)
 *   stage 2: U** = U^n + dt [T(U^n) + T(U^(n+1/2))]/2 + (dt/2) S(U^(n+1/2)); U^(n+1) = U** + (dt/2) S(U^(n+1)) (theta = 1/2)
 * work_dev: a caller-owned DEVICE scratch state of the same shape (its mom, Egas, Erad, Frad are overwritten; its
 * rho, kappa_scale, Srad are ignored).  U_dev->Srad must be NULL.  Stream-ordered, asynchronous: 8 copies, two
 * transport kernels, 8 averaging kernels and two source updates are enqueued. */
int mgrhd_imex_step_1d(mgrhd_ctx *ctx, const mgrhd_state *U_dev, const mgrhd_state *work_dev, long long nx,
                       double dx, double dt, double c, double c_hat, int bc, void *cuda_stream);

/* Per-cell conserved totals of a DEVICE state, for conservation checks:
 *   out_energy[n]      = E_gas + (c/c_hat) sum_g E_g
 *   out_momentum[3][n] = rho v^i + (c c_hat)^-1 sum_g F_g^i
 * Stream-ordered, asynchronous. */
int mgrhd_conserved_totals(mgrhd_ctx *ctx, const mgrhd_state *state_dev, long long ncells,
                           double c, double c_hat, double *out_energy, double *out_momentum,
                           void *cuda_stream);

/* Copy the device counters to *host_out (synchronises the last stream used). */
int mgrhd_get_stats(mgrhd_ctx *ctx, mgrhd_stats *host_out);
/* Zero the device counters (stream-ordered on the last stream used). */
int mgrhd_reset_stats(mgrhd_ctx *ctx);
/* Switch the instrumented kernels on (1) or off (0, default): they also accumulate the
 * ALGORITHMIC FP64 flop count of the update (FMA = 2) into
 * mgrhd_stats.flops.  Used by bench.py for the ALU roofline; never on in a timed region. */
int mgrhd_set_flop_counting(mgrhd_ctx *ctx, int on);
/* Number of kernels this context has launched so far (for bench.py's gpu_launches). */
long long mgrhd_launch_count(const mgrhd_ctx *ctx);

/* The source update (same operation, same kernel, same results as mgrhd_source_update) for callers that cannot
 * allocate device memory -- code under CUDA graph capture, serving loops, harnesses that forbid cudaMalloc.  It
 * needs no context: the group structure and the model are passed on every call (HOST pointers, as for mgrhd_init),
 * and the kernel's scratch (the work counter and the F_g^(t) copy of the cells in flight) and
 * its counter block live in file-scope `static __device__` arrays of the library:
 *   MGRHD_STATIC_SCRATCH_BYTES (12 MiB) of scratch + 1.2 KB of counters, held by EVERY GPU that loads the library
 *   until the process exits.
 * The call does no cudaMalloc / cudaFree and calls no allocating library routine; per device, its first call does
 * the one-time set-up (Planck tables to __constant__ memory, cudaGetSymbolAddress of the two arrays): make that
 * call outside a graph capture.
 * Limits.  Only the models the tuned kernel runs: spectrum 0, opacity_kind 0 or 1, outer_mode 0 (anything else:
 * MGRHD_ERR_ARG).  The scratch a launch needs is 256 + 24 NQL threads_per_CTA CTAs bytes (NQL = 4, 8, 8, 8, 16 and
 * 256, 384, 384, 384, 256 threads for Nq <= 4, 8, 16, 32, 64; CTAs = min(resident CTAs of the device,
 * ceil(ncells / cells per CTA))): on a 148-SM B200 every Nq <= 32 fits at any ncells (10.9 MB); 32 < Nq <= 64 fits
 * up to 8192 cells.  A launch that needs more returns MGRHD_ERR_SIZE (mgrhd_last_error() states both numbers)
 * and does nothing.
 * Sharing.  Every call on a device uses the same arrays, which keep the previous call's contents: the call clears
 * the work counter and the counters itself (stream-ordered memsets), the rest of the scratch is written before it is
 * read.  Two calls that overlap on the GPU (different streams, or two host threads) RACE on the arrays and give
 * wrong results: issue them on one stream, or order them with events.
 * stats_out: NULL, or a HOST struct that receives this call's counters; a non-NULL stats_out makes the call
 * synchronise the stream.  state: DEVICE pointers, as in mgrhd_source_update; updated in place.
 * Errors: as mgrhd_init and mgrhd_source_update for the same arguments, plus MGRHD_ERR_SIZE. */
#define MGRHD_STATIC_SCRATCH_BYTES (12ll << 20)
int mgrhd_source_update_static(const double *edges, int Nq, const mgrhd_units *u, const mgrhd_opacity_model *m,
                               const mgrhd_state *state, long long ncells, double dt, double c, double c_hat,
                               void *cuda_stream, mgrhd_stats *stats_out);

/* Diagnostic: the kernels' Planck edge functions on n DEVICE values x >= 0 (x = h nu/(k_B T)):
 *   is_y[i] = 1: yz[i] = Y(x) = (15/pi^4) int_0^x t^3/(e^t-1) dt;  is_y[i] = 0: yz[i] = 1 - Y(x);
 *   xi[i] = (15/pi^4) x^4/(e^x-1).  (Eq. 11 applied to B_nu.)
 * form 0: the per-interval polynomial rows (Y below x = 1) every update kernel uses; form 1: the three-branch
 * evaluation (Y below x = 1.25) kept for a kernel instantiation without room for the rows (none is dispatched
 * today).  Other values: MGRHD_ERR_ARG.
 * Stream-ordered. */
int mgrhd_planck_edge_functions(const double *x_dev, long long n, double *yz_dev, double *xi_dev,
                                int *is_y_dev, int form, void *cuda_stream);

/* Sustained FP64 FMA rate of the current device in FMA/s (a dependent-chain-free DFMA
 * microbenchmark, `iters` FMAs per thread; used as the ALU roofline denominator). */
int mgrhd_measure_dfma_peak(long long iters, double *fma_per_second);

/* Text of the last CUDA error seen by this library on the calling thread ("" if none). */
const char *mgrhd_last_error(void);

void mgrhd_free(mgrhd_ctx *ctx);

#ifdef __cplusplus
}
#endif
#endif /* MGRHD_H */
