/* geo.h -- C ABI of libgeo: batched fixed-step RK4 integration of independent null / timelike
 * geodesics in Schwarzschild and Kerr spacetimes on NVIDIA B200 (sm_100a).
 *
 * The operation is the hot path of MALBEC (arXiv:1803.08320): "a large set of system[s solved]
 * independently" (sec. 5), each system being Hamilton's equations (3),(4)
 * of H = 1/2 g^{mu nu} p_mu p_nu for the Kerr metric (6) written
 * in the 3+1 variables of eqs.(1),(8) (lapse alpha, shift beta^i, spatial metric
 * gamma_ij), advanced with the classical fourth-order Runge-Kutta method and
 * stopped per particle at the event horizon r_+ = M + sqrt(M^2 - a^2).
 * Schwarzschild is a = 0, eqs.(29)-(32).  Units G = c = 1.
 *
 * State per geodesic, paper order:  y = (t, r, theta, phi, p_t, p_r, p_theta, p_phi),
 * Boyer-Lindquist coordinates, covariant momenta, independent variable tau (proper time / affine
 * parameter).  p_t is stored with the PAPER's sign, p_t = E > 0 (eq.(29); DESIGN.md
 * reading G1); p_phi = L.  p_t and p_phi are constants of motion (eqs.(13),(32)).
 *
 * Every compute step runs in hand-written CUDA kernels; there is no CPU fallback.  All functions
 * return GEO_OK (0) or an error code; nothing throws, nothing aborts.  Argument errors are reported
 * synchronously before any launch.  geo_integrate only ENQUEUES work on `cuda_stream`.
 */
#ifndef GEO_H_
#define GEO_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct geo_ctx geo_ctx; /* opaque; owned by the library */

enum { GEO_SCHWARZSCHILD = 0, GEO_KERR = 1, GEO_TABULATED = 2,    /* metric (2: geo_create_tabulated,          */
       GEO_TABULATED_GENERAL = 3,                                    /*         3: geo_create_tabulated_general)  */
       GEO_KERR_SCHILD = 4 };   /* Kerr in Cartesian Kerr-Schild coordinates (geo_create; see below)               */
enum { GEO_TIMELIKE = 0, GEO_NULL = 1 };                            /* geo_stop.kind: kappa=1/0 */
enum { GEO_OK = 0, GEO_EINVAL = 1, GEO_ECUDA = 2, GEO_ENOMEM = 3 }; /* return codes            */
/* per-particle termination class (geo_out.status) */
enum { GEO_ST_MAXSTEPS = 0, GEO_ST_CAPTURED = 1, GEO_ST_ESCAPED = 2, GEO_ST_NUMERIC = 3,
       GEO_ST_OUTSIDE = 4 /* tabulated metrics only: an evaluation point left the table's domain */ };
/* geo_stop.flags */
enum {
    GEO_FLAG_PLAIN_UPDATE = 1, /* y <- y + delta without the Kahan error term (P1)     */
    GEO_FLAG_STATIC_MAP = 2,   /* thread i integrates particle i; no work queue (for comparison) */
    GEO_FLAG_CARTESIAN_SNAP = 8, /* snapshot components 1..3 hold (x, y, z) of eq.(7) PAPER.md:88-93 instead
                                  of (r, theta, phi): with snap_mask = 0x0F a record is (t, x, y, z), the paper's
                                  output format -- tau is implicit, slot j <-> tau = j*snapshot_every*h */
    GEO_FLAG_TAB_GATHER = 16,  /* tabulated metrics: gather the 4 x 4 stencil through L1/L2 on every evaluation instead
                                  of keeping the current cell's stencil in shared memory (for comparison)  */
    GEO_FLAG_STAGED_SNAP = 4   /* snapshot records staged in shared memory and flushed by the warp with
                                  coalesced stores (for comparison).  Without the flag each lane stores its record
                                  straight from registers with 256-bit stores, at every cadence.  Both writers put
                                  the same bits into the same slots.                                       */
};

/* Stop rules (PAPER.md:322-327 gives "final time reached" and "r <= r_+"; B1-B4):
 *  - CAPTURED at the first step in which the start point, any RK4 stage point or the end point has
 *    !(r >= r_capture); that step is not taken, the final state is the last accepted one.
 *  - ESCAPED when, after an accepted step, r > r_escape.
 *  - MAXSTEPS after `nsteps` accepted steps.  Use r_capture = -inf, r_escape = +inf to disable. */
typedef struct geo_stop {
    double r_capture;
    double r_escape;
    int32_t kind;  /* GEO_TIMELIKE or GEO_NULL: kappa in the mass shell 2H = -kappa, eq.(5) */
    int32_t flags; /* GEO_FLAG_* */
} geo_stop;

/* Output buffers.  geo_integrate: DEVICE pointers; geo_integrate_host: HOST pointers.  All caller-owned.
 * Pointers must be 16-byte aligned.  Optional ones may be NULL. */
typedef struct geo_out {
    double *final_state;   /* [8][n] SoA, paper order t,r,theta,phi,p_t(=E),p_r,p_theta,p_phi          */
    int32_t *status;       /* [n] GEO_ST_*                                                             */
    int64_t *steps_done;   /* [n] accepted RK4 steps                                                   */
    double *eq_cross_r;    /* [n] optional: r at the first crossing of theta = pi/2, linear in theta
                              between the two accepted states that bracket it; quiet NaN if none (B5)  */
    double *health;        /* [n] optional: |2H + kappa| of the final state (0 on the exact solution)  */
    double *snapshots;     /* [n][snap_capacity][ncomp] particle-major; required iff snapshot_every>0  */
    int64_t snap_capacity; /* slots per particle; records beyond it are dropped, still counted (S3)    */
    uint32_t snap_mask;    /* bit k set => component k of the 8-vector is stored; ncomp = popcount      */
    int32_t *snap_count;   /* [n] records produced (slot 0 = initial state; slot j = after
                              j*snapshot_every accepted steps; none after termination) (S1)            */
    int32_t *coarse_steps; /* [n] optional diagnostic: RK4 step attempts of this particle in which a stage angle moved
                              by >= 2^-7 rad, so that the step was evaluated with a full sin/cos at every stage point
                              instead of the angle-addition kernels (same result to rounding).
                              Analytic metrics, geo_integrate / geo_integrate_host only; ignored elsewhere.           */
} geo_out;

/* Create a context for metric (6) with mass M > 0 and spin |a| <= M; Schwarzschild
 * requires a == 0.  metric: GEO_SCHWARZSCHILD, GEO_KERR (Boyer-Lindquist coordinates, eq.(8)) or GEO_KERR_SCHILD (below).  Allocates a few bytes of device memory on the CURRENT CUDA device; the ctx belongs to that
 * device: every entry point switches to it for the duration of the call and restores the caller's current
 * device before returning, so device pointers passed with a ctx must live on the ctx's device. */
int geo_create(geo_ctx **ctx, int metric, double M, double a);

/* GEO_KERR_SCHILD -- SURVEY 8(f).3, second clause ("further analytic metrics / horizon-penetrating, axis-regular
 * coordinates"; the reason the paper gives for the 3+1 form): the SAME spacetime, metric (6)
 * (PAPER.md:73-84), in Cartesian Kerr-Schild coordinates (t~, x, y, z) (readings K1-K5):
 *     g = eta + f l l,  f = 2 M r^3/(r^4 + a^2 z^2),  l_mu = (1, (r x + a y)/(r^2+a^2), (r y - a x)/(r^2+a^2), z/r),
 *     r(x, y, z) >= 0:  (x^2 + y^2)/(r^2 + a^2) + z^2/r^2 = 1        (the Boyer-Lindquist r of the same event),
 * i.e. line element (1) with alpha^2 = 1/(1+f), beta^i = f l_i/(1+f), gamma_ij = delta_ij + f l_i l_j; related to
 * Boyer-Lindquist by t~ = t + int 2Mr/Delta dr, phi~ = phi + int a/Delta dr, x + iy = (r + ia) sin(theta) e^{i phi~},
 * z = r cos(theta).  Regular on the polar axis and through the future horizon r_+ (only the ring r = 0, z = 0 is singular):
 * rays through the axis and particles followed inside the hole -- where eq.(8) divides by sin^2(theta) or Delta -- integrate
 * without loss of accuracy.  Equations of motion: Hamilton's equations (3),(4) of
 * H = 1/2 [ -(p_t - beta^k p_k)^2/alpha^2 + gamma^{ij} p_i p_j ]; p_t = -E is the only cyclic momentum of the chart.
 * Use with geo_integrate / geo_integrate_host:
 *   state_in SoA [6][n] = (x, y, z, p_x, p_y, p_z) (covariant); t~ starts at 0, E from the mass shell eq.(5) in 3+1 variables.
 *   final_state [8][n] and trajectory records = (t~, x, y, z, p_t = E, p_x, p_y, p_z) (snap_mask over these).
 *   r_capture / r_escape refer to r(x, y, z); the capture guard runs on y0, every RK4 stage point and the end point.
 *   eq_cross_r: r at the first sign change of z between two accepted states, linear in z between them; quiet NaN if none.
 *   health = |2H + kappa|.  coarse_steps is ignored.  flags: GEO_FLAG_PLAIN_UPDATE, GEO_FLAG_STATIC_MAP
 *   (records are Cartesian already: GEO_FLAG_CARTESIAN_SNAP and the staged writer return GEO_EINVAL).
 * geo_integrate_adaptive / geo_integrate_adaptive_host take this metric too (reading K6; flags must be 0): the pair,
 *   controller, landing rule and dense output documented at geo_integrate_adaptive, over the SEVEN components
 *   (t~, x, y, z, p_x, p_y, p_z), with two rules of this chart's own -- (a) no attempt moves the particle by more than a
 *   quarter of its current radius, h <- min(h, r / (4 |dx/dtau|)) (far from the hole the geodesics are straight lines here and
 *   the error estimate alone would let a step jump over the hole; not applied in fixed-step mode), (b) the capture test runs on
 *   y0 and on the END POINT of an attempt, not on the stage points (the chart is regular through the horizon).
 * geo_integrate_host_noalloc returns GEO_EINVAL for this metric; geo_horizon_radius works. */

/* Integrate n geodesics for at most nsteps (< 2^31) RK4 steps of size h (h < 0 integrates backwards in tau).
 * state_in: DEVICE, SoA [6][n] = (r, theta, phi, u_r, u_theta, u_phi) (covariant); t starts at 0 and
 * p_t is derived from the mass shell eq.(5) in 3+1 variables.  snapshot_every = 0: no snapshots.
 * cuda_stream: a cudaStream_t (NULL = default stream).  Enqueue-only: outputs are valid after the
 * caller synchronises the stream.  A ctx must not be used from two streams concurrently. */
int geo_integrate(geo_ctx *ctx, const double *state_in, int64_t n, double h, int64_t nsteps,
                  const geo_stop *stop, int64_t snapshot_every, const geo_out *out, void *cuda_stream);

/* Same operation with HOST buffers (pageable or pinned; pinned lets the copies overlap the kernels):
 * copies state_in to the device, integrates, copies every non-NULL output back and synchronises before
 * returning.  Large jobs are cut into particle chunks that are double-buffered on two streams, so the
 * D2H of one chunk overlaps the integration of the next (the paper's bottleneck).
 * Snapshot slots >= snap_count[i] are returned as NaN (all-ones bit pattern).  Device scratch is owned
 * by the ctx and reused between calls. */
int geo_integrate_host(geo_ctx *ctx, const double *state_in, int64_t n, double h, int64_t nsteps,
                       const geo_stop *stop, int64_t snapshot_every, const geo_out *out);

/* adaptive embedded Runge-Kutta 5(4) (Dormand-Prince pair, first-same-as-last) with a step
 * size per geodesic ("others method of the RK family will be included soon").
 *   err = max_c |e_c| / (atol + rtol max(|y_c|, |ynew_c|)) over the 6 evolving components; a step is accepted
 *   iff err <= 1; h <- h min(5, max(0.2, 0.9 err^(-1/5))) (not enlarged after a rejection).
 * h0 > 0: first trial step.  rtol = +INFINITY: fixed step h0 (no error test; a non-finite
 * attempt then ends the particle with GEO_ST_NUMERIC at once).  h_min: a rejected step that would fall below it -- or,
 * with h_min = 0, a step that has shrunk to zero -- ends the particle with GEO_ST_NUMERIC.  tau_end: final value of the affine parameter,
 * landed on exactly ("the final evolution time is reached"; +INFINITY: none); reaching it, or
 * max_attempts (< 2^31, accepted + rejected), ends with GEO_ST_MAXSTEPS.  Capture / escape as in geo_stop
 * (capture guard on every stage point).  out: as for geo_integrate; steps_done = accepted steps.
 * rejected: DEVICE [n] int32 or NULL.  Enqueue-only on cuda_stream.
 * DENSE OUTPUT (reading A3): snap_dtau > 0 writes trajectory records at the FIXED affine times
 * tau_j = j * snap_dtau, j = 0, 1, ... (slot 0 = the initial state), for every tau_j up to the last accepted state of the
 * particle, from the pair's fourth-order continuous extension (the dense output of DOPRI5) -- no step is shortened for a
 * record.  out->snapshots / snap_capacity / snap_mask / snap_count as for geo_integrate (records beyond the capacity are
 * dropped, still counted).  snap_dtau = 0: no records, the snapshot fields of `out` are ignored.
 * flags: 0 or GEO_FLAG_CARTESIAN_SNAP (records carry (x, y, z) of eq.(7)). */
typedef struct geo_adaptive {
    double h0, rtol, atol, h_min, tau_end;
    double snap_dtau; /* spacing of the dense-output records in tau; 0 = none */
} geo_adaptive;
int geo_integrate_adaptive(geo_ctx *ctx, const double *state_in, int64_t n, const geo_adaptive *ctl,
                           int64_t max_attempts, const geo_stop *stop, const geo_out *out, int32_t *rejected,
                           void *cuda_stream);

/* Same operation with HOST buffers (state_in, every non-NULL output and `rejected` are host pointers; pinned lets the
 * copies run at full speed): H2D, launch, D2H, synchronise -- through the same double-buffered chunk pipeline as
 * geo_integrate_host (record slots >= snap_count[i] come back as NaN).  Device scratch is owned by the ctx. */
int geo_integrate_adaptive_host(geo_ctx *ctx, const double *state_in, int64_t n, const geo_adaptive *ctl,
                                int64_t max_attempts, const geo_stop *stop, const geo_out *out, int32_t *rejected);

/* a NUMERICALLY GIVEN metric ("the 3+1 formulation is important in order to bring future support
 * to numerical metrics"; "a new algorithm to handle numerically computed metrics").
 * Line element (1) with the structure of eq.(8): stationary, axisymmetric,
 * beta^i = (0, 0, beta^phi), gamma_ij = diag(gamma_11, gamma_22, gamma_33), five functions of (x^1, x^2) sampled at
 * the nodes x^1_i = x1_0 + i d1 (0 <= i < n1), x^2_j = x2_0 + j d2 (0 <= j < n2):
 *     tab[f][j][i], f = 0..4 = alpha, beta^phi, gamma_11, gamma_22, gamma_33      (HOST, n1 fastest; copied, not kept).
 * (x^1, x^2) are the metric's own coordinates -- (r, theta) for Boyer-Lindquist Kerr.  Between the nodes each field is
 * the tensor-product cubic-convolution interpolant (Keys 1981, parameter -1/2: C^1, exact on quadratics, value error
 * O(d^3), gradient error O(d^2)) and the equations of motion are Hamilton's equations (3),(4) of
 *     H = 1/2 [ -(p_t - beta^phi p_phi)^2/alpha^2 + p_1^2/gamma_11 + p_2^2/gamma_22 + p_phi^2/gamma_33 ]
 * with the EXACT gradient of the interpolant, so p_t and p_phi are constants of motion (T1-T5).
 * The interpolant exists where its 4 x 4 stencil does: floor((x - x_0)/d) in [1, n - 3] in both directions.
 * A ctx created here is used with geo_integrate / geo_integrate_host: state_in = (x^1, x^2, phi, p_1, p_2, p_phi),
 * r_capture / r_escape refer to x^1, the equatorial event to x^2 = pi/2; an evaluation point (y0, a stage point, the
 * end point of a step) outside the domain ends the particle with GEO_ST_OUTSIDE, that step is not taken (per
 * evaluation point the capture test comes first).  Trajectory records (snapshot_every > 0) as for the analytic metrics,
 * components (t, x^1, x^2, phi, p_t = E, p_1, p_2, p_phi) by snap_mask; flags: GEO_FLAG_PLAIN_UPDATE, GEO_FLAG_TAB_GATHER
 * (no staged writer, no Cartesian records: the coordinates are the table's own).
 * geo_integrate_adaptive / geo_integrate_adaptive_host accept such a ctx too -- and one made by geo_create_tabulated_general
 * (reading T7: the domain test joins the capture test on every stage point and the end point; flags must be 0);
 * geo_horizon_radius returns NaN.
 * Errors: GEO_EINVAL (NULL, n1 or n2 < 4, d1 or d2 <= 0, non-finite grid), GEO_ENOMEM, GEO_ECUDA. */
typedef struct geo_table {
    const double *tab;  /* HOST [5][n2][n1] (geo_create_tabulated) or [10][n2][n1] (geo_create_tabulated_general) */
    int64_t n1, n2;
    double x1_0, d1, x2_0, d2;
} geo_table;
int geo_create_tabulated(geo_ctx **ctx, const geo_table *table);

/* SURVEY 8(f).3, general form (reading T6): line element (1) for ANY stationary, axisymmetric
 * metric -- all ten functions of (x^1, x^2), x^3 = phi being the symmetry direction:
 *     tab[f][j][i], f = 0..9 = alpha, beta^1, beta^2, beta^3, gamma_11, gamma_12, gamma_13, gamma_22, gamma_23, gamma_33
 * (HOST, same grid conventions as geo_create_tabulated; copied, not kept).  No circularity and no diagonal 3-metric is
 * assumed: horizon-penetrating coordinates (e.g. Kerr in Kerr-Schild form: beta^r != 0, gamma_r phi != 0) are in scope.
 * Same interpolant with its exact gradient; equations of motion = Hamilton's equations (3),(4) of
 *     H = 1/2 [ -(p_t - beta^k p_k)^2/alpha^2 + gamma^{ij} p_i p_j ],   gamma^{ij} = inverse of gamma_ij (3 x 3, per evaluation),
 * p_t and p_phi constants of motion.  Use with geo_integrate / geo_integrate_host exactly like a geo_create_tabulated
 * ctx (state_in = (x^1, x^2, phi, p_1, p_2, p_phi); GEO_ST_OUTSIDE; trajectory records by snap_mask over
 * (t, x^1, x^2, phi, E, p_1, p_2, p_phi); flags: GEO_FLAG_PLAIN_UPDATE, GEO_FLAG_TAB_GATHER), and with
 * geo_integrate_adaptive / geo_integrate_adaptive_host (reading T7 with the T6 right-hand side, dense output included). */
int geo_create_tabulated_general(geo_ctx **ctx, const geo_table *table);

/* ALLOCATION-FREE entry point, for callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving
 * loops, harnesses that forbid it): the operation of geo_integrate_host -- fixed-step RK4 of n independent
 * geodesics in the analytic metric (6), HOST buffers in and out -- without a ctx (geo_create
 * allocates) and without trajectory records.  Its device scratch -- the persistent kernel's work-queue head and the
 * staging of state_in and of every output -- is a `static __device__` array inside the library of
 *     256 + 144 * GEO_NOALLOC_MAX_N bytes = 9 437 440 B (9.0 MiB),
 * which every GPU that loads the library holds until the process exits.  The call makes no cudaMalloc, cudaFree,
 * stream / event creation or other allocating library call; the first use on a device resolves the array's device
 * address (cudaGetSymbolAddress) and reads the SM count, nothing else.
 *   metric, M, a: as geo_create (GEO_SCHWARZSCHILD or GEO_KERR).  state_in, h, nsteps, stop: as geo_integrate_host;
 *   stop->flags: 0, GEO_FLAG_PLAIN_UPDATE, GEO_FLAG_STATIC_MAP.  out: HOST pointers; final_state, status, steps_done
 *   required, eq_cross_r, health, coarse_steps optional, the snapshot fields are ignored.  cuda_stream: the stream the
 *   copies and the kernel are enqueued on (NULL = default stream); the call synchronises it before returning.
 * Same kernels, same launch configuration, same bits as geo_integrate_host on the current device.
 * n > GEO_NOALLOC_MAX_N returns GEO_EINVAL (text from geo_noalloc_last_error) before anything is enqueued.
 * The scratch is SHARED by all calls and keeps the previous call's contents: the queue head is cleared on the stream
 * before every launch and every staged output element of particles 0..n-1 is overwritten by the kernel, so nothing else
 * needs to start at zero.  Calls from several host threads are serialised by a lock inside the library; anything else
 * that would make two such calls overlap on one GPU (there is none through this interface) would race on the scratch.
 * Errors: GEO_EINVAL, GEO_ECUDA; never GEO_ENOMEM. */
#define GEO_NOALLOC_MAX_N 65536
int geo_integrate_host_noalloc(int metric, double M, double a, const double *state_in, int64_t n, double h,
                               int64_t nsteps, const geo_stop *stop, const geo_out *out, void *cuda_stream);
const char *geo_noalloc_last_error(void); /* text of the calling thread's last geo_integrate_host_noalloc error */

void geo_destroy(geo_ctx *ctx);

double geo_horizon_radius(const geo_ctx *ctx); /* r_+ = M + sqrt(M^2 - a^2) */
const char *geo_last_error(const geo_ctx *ctx); /* text of the last error on this ctx ("" if none) */

#ifdef __cplusplus
}
#endif
#endif /* GEO_H_ */
