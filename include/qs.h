/* qs.h — C ABI of the B200-native quench-simulation hot path (after arXiv:2403.07666).
 *
 * One handle = one simulation of a solenoid cross-section of N coaxial current rings ("cells")
 * advanced step by step under a ramped transport current I_a(t) and a ramped axial background
 * field (the problem statement; J^{k+1} from rho^k = rho(J^k),
 * then the heat equation with the Joule source E.J).  Every step of the path runs in
 * hand-written CUDA kernels for sm_100a; there is no CPU fallback: a call made without a usable
 * CUDA device fails with QS_ERR_CUDA.
 *
 * Readings of the points the paper leaves to its (unavailable) Supplementary Information are
 * numbered C1..C13 in SURVEY.md §8(c) and restated in DESIGN.md; they are cited as "C<k>" below.
 *
 * Conventions
 *   - All array arguments of the plain calls are HOST pointers owned by the caller, valid for the
 *     duration of the call only; the library copies what it needs.  The *_device variants take
 *     DEVICE pointers (FP64, at least n_rings elements, 16-byte aligned) and enqueue on the handle's
 *     stream; they return after the work has been enqueued and checked for launch errors only.
 *   - FP64 throughout (BASELINE.json configs[0]).  SI units.  Ring order is the caller's order
 *     (lattice: canonical c = ir*Nz + iz, C1); any internal re-ordering is invisible.
 *   - Return value: 0 = OK, negative = error (state unchanged: J, T, t, I, the fields B, E of qs_read, the event
 *     flags / counters and the per-wire statistics are what they were before the call), and for qs_step a
 *     non-negative event bitmask.  qs_last_error() returns a human-readable message for the calling thread.
 *   - One handle per host thread; calls on one handle are serialised on its stream.  A handle lives on the CUDA
 *     device that was current at qs_init; every call makes that device current for its duration and restores
 *     the caller's, so handles on different devices can be used from one process.
 */
#ifndef QS_H_
#define QS_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct qs_ctx qs_ctx;

/* error codes */
#define QS_OK            0
#define QS_ERR_ARG      -1   /* bad argument (NULL, size, inconsistent lattice, rings outside the validity domain) */
#define QS_ERR_CUDA     -2   /* CUDA error or no device */
#define QS_ERR_NONFINITE -3  /* NaN/Inf in J or T after the step (state restored)            */
#define QS_ERR_CG       -4   /* CG breakdown p^T A p <= 0 (state restored)                  */
#define QS_ERR_DT       -5   /* dt <= 0                                                      */

/* qs_step return bits */
#define QS_EV_FLUXJUMP   1   /* some turn's flux-jump flag group (FJ_T|FJ_E|FJ_J) rose this step */
#define QS_EV_QUENCH     2   /* some turn has a quench flag (Q_T|Q_RHO) set                    */
#define QS_EV_CG_MAXIT   4   /* CG stopped at cg_maxit; the state was advanced anyway          */

/* per-turn flag bits (C10; PAPER.md:105 |J/Jc| > 1, PAPER.md:119 rho > 0.95 rho_n; configs[3]) */
#define QS_FJ_T    1         /* Tmax_w > T_fluxjump                                            */
#define QS_FJ_E    2         /* d(mean|E|_w)/dt > dEdt_spike                                   */
#define QS_FJ_J    4         /* max |J|/Jc > 1 in the turn                                     */
#define QS_Q_T     8         /* Tmax_w > Tc                                                    */
#define QS_Q_RHO  16         /* min rho/rho_n > 0.95 in the turn                               */

/* qs_geometry.flags */
#define QS_GEO_NO_OPERATOR 1 /* thermal / pointwise use only: no pair operator is set up, qs_step,
                                qs_matvec, qs_solve, qs_field return QS_ERR_ARG (roofline runs of
                                the HBM-bound passes on lattices whose N^2 sweep is out of reach)  */

#define QS_GEO_LATTICE_TABLES 2 /* lattice geometries: evaluate every unique pair value once at qs_init into tables over
                                  (ir, jr, |iz - jz|) (3 x 8 Nr^2 Nz bytes of workspace) and apply M and G_B as block-
                                  Toeplitz products instead of on-the-fly pair sweeps.  Same
                                  arithmetic per unique pair, same results up to summation order.  */

#define QS_GEO_NO_PATCH_PRECOND 4 /* lattice geometries whose constraint groups are the wires: do NOT build the patch
                                    (block-Jacobi over p x p cells of a wire, p <= 16: whole wires of up to 16 x 16
                                    cells) constraint preconditioner of the projected CG (up to 2 x 8 N p^2 bytes of
                                    workspace); the solver then keeps diag(A) (C8).
                                    The preconditioner is free: the solution of a step is unique (C4).  */

#define QS_GEO_PATCH_SUBWIRE 16   /* constraint preconditioner: plain patches of p x p cells, p <= 8, only - no whole-wire
                                    blocks (wires of up to 16 x 16 cells) and no second level of patch-wise constants
                                    (larger wires); a preconditioner only either way (C8).  */

#define QS_GEO_HEAT_BLOCKED 8     /* measurement: use the temporally blocked heat kernel (<= 4 explicit sub-steps per
                                    launch from a shared-memory tile with a 4-cell halo) at ANY lattice size; by
                                    default it serves lattices up to 2 M cells (L2-resident), larger ones run one
                                    marching kernel per sub-step.  Same arithmetic per cell either way (C9).  */

typedef struct {
  int32_t  n_rings;                 /* N                                                         */
  const double *r, *z, *area;       /* [N] ring centre radius, height, cross-section [m, m, m^2] */
  const int32_t *turn_id;           /* [N] in 0..n_turns-1, or NULL when n_turns == 0            */
  int32_t  n_turns;                 /* N_w; 0 = no net-current constraint (config 4)             */
  int32_t  lattice;                 /* 1: regular winding pack described below (enables qs_step);
                                       0: free rings (operator / solve only)                     */
  int32_t  layers, turns_per_layer, cells_per_side;  /* lattice: L along r, T_n along z, n (C1)  */
  double   wire_size, r_inner;      /* lattice: wire side s [m] (h = s/n), inner radius [m];
                                       r = r_inner+(ir+1/2)h, z = (iz+1/2)h - Nz h/2 are CHECKED
                                       against r[], z[] to 1e-9 relative                          */
  double   softening;               /* g [m] (C2): lattice: M_ii = M(r_i, r_i, dz = g) and the
                                       self-field term; free rings: dz^2 + g^2 for ALL pairs      */
  double   h_conv[4];               /* bath film coefficient on the r_min, r_max, z_min, z_max
                                       borders of the winding pack [W/m^2K]        */
  double   T_bath;                  /* [K]                                                       */
  double   Bext0, Bext_rate, Bext_max; /* axial background field B_ext(t) = min(Bext0 + rate t, max);
                                       rate == 0: constant Bext0                                  */
  int32_t  flags;                   /* QS_GEO_*                                                  */
  const double *turn_share;         /* [n_turns] share of the transport current each constraint group carries
                                       (C16; PAPER.md:61-67 sub-elements): the constraint is
                                       sum_{i in group w} I'_i = turn_share[w] * I_ramp, and U_terminal =
                                       -sum_w turn_share[w] V_w.  NULL = 1 for every group (wires in series).
                                       Sub-elements of a wire are groups of their own (turn_id = sub-element id)
                                       with shares summing to 1 per wire; share 0 = zero-net-current group
                                       (uncoupled sub-element under a field ramp).  Must be finite.          */
} qs_geometry;

typedef struct {
  double Ec, n_exp, Jc0, Tc, B0, eps_coef, eps_exp, Y, rho_n;  /* C5: 1e-4, 20, 2e9, 18, 1, 900, 1.7, 1e11, 5e-10 */
  const double *jc0_scale;          /* [N] per-cell Jc0 multiplier, NULL = 1                     */
  double C3, C1;                    /* C(T) = C3 T^3 + C1 T  [J/m^3K]  (2000, 500)               */
  double k_in, k_between;           /* k = k_in T inside a wire, k_between T across wires (5, 0.5) */
  double theta;                     /* C7: 0 explicit Euler (literal), 1 linearly implicit (default) */
  double cg_tol; int32_t cg_maxit;  /* stop when sqrt(r^T g) <= cg_tol * nu (C8)                 */
  double T_fluxjump, dEdt_spike;    /* C10: 10 K, 1 V/m/s                                        */
  int32_t heat_adi_substeps;        /* 0: explicit heat sub-steps (C9, default); m > 0: m ADI sub-steps per step
                                       (C15; the paper's thermal method)      */
} qs_material;

typedef struct {
  int32_t cg_iters;                 /* projected-CG iterations of the last step / solve          */
  int32_t heat_substeps;            /* m of the last step (C9)                                   */
  int32_t event_word;               /* last qs_step return value                                 */
  int32_t sweeps;                   /* pair sweeps (operator applications) of the last step/solve */
  double  cg_relres;                /* sqrt(r^T g)/nu reached                                    */
  double  U_terminal;               /* -sum_w V_w [V] (PAPER.md:99 terminal voltage)             */
  double  Tmax;                     /* max T after the step [K]                                  */
  double  joule_power;              /* sum_i Q_i 2 pi r_i a_i [W] of the step's material evaluation */
  double  t, I;                     /* time [s] and transport current [A] after the step         */
  int64_t launches;                 /* kernels launched by this handle since qs_init             */
  int64_t pair_evals;               /* ring-pair evaluations since qs_init                       */
  double  dJ_max;                   /* max_c |J^{k+1} - J^k| of the last step [A/m^2] (input of the caller's
                                       time-step controller, C11)                                */
} qs_stats_t;

/* ---- the three calls north_star names -------------------------------------------------------- */

/* Create a simulation: copies geometry and material, allocates device state with cudaMalloc on
 * the current device, uses its own stream.  State: J = 0, T = T_bath, t = 0, I = 0.  */
int  qs_init(const qs_geometry *geo, const qs_material *mat, qs_ctx **out);

/* One time step k -> k+1 (order C6):
 *   S1 B^k = G_B (a J^k) + B_ext(t^k)            all-pairs ring field, K/E by AGM per pair (C3)
 *   S2 eps, Jc, rho, E, dE/dJ, Q at (J^k, T^k, B^k); rhs b = -2 pi r (E + r Bdot_ext/2)   (C5, C4)
 *   S3 projected CG on (M + theta dt D) I' + C V = b, C^T I' = I_ramp     (C4, C7, C8)
 *   S4 per-turn Schur projection inside S3; multipliers V_w -> terminal voltage
 *   S5 J += dt I'/a ; I += dt I_ramp ; t += dt
 *   S6 m explicit 5-point finite-volume heat sub-steps with Q^k frozen, Robin borders (C9)
 *   S7 per-turn event flags (C10)
 * I_ramp = dI/dt [A/s] held over the step.  Lattice geometries only.  Synchronous.  */
int  qs_step(qs_ctx *ctx, double dt, double I_ramp);

/* One ACCEPTED step of the embedded Heun-Euler (RK12) pair with step-size control (the paper
 * integrates the electromagnetic equations by a "Runge-Kutta method with variable time step"; readings
 * C14 in DESIGN.md §3).  With T frozen at T^k:
 *   stage 1: I'_1 from M I' + C V = b(J^k, t^k), C^T I' = I_ramp;  predictor J* = J^k + dt I'_1 / a
 *   stage 2: I'_2 at (J*, t^k + dt);  J^{k+1} = J^k + dt (I'_1 + I'_2) / (2a)
 *   err = max_i |dt (I'_2 - I'_1)_i / (2 a_i)| / (Jc0 (1 - T_bath/Tc)^2)
 * The step is accepted if err <= rtol or dt == dt_min, else retried with dt <- max(dt_min, dt max(0.2, 0.9
 * sqrt(rtol/err))).  Then the heat step with the trapezoid source (Q_1 + Q_2)/2 and the events; qs_read's B, E are
 * those of stage 2.  Outputs (may be NULL): the dt taken, the suggestion dt min(2, max(0.2, 0.9 sqrt(rtol/err))) for
 * the next call, and err.  Returns like qs_step.  */
int  qs_step_rk(qs_ctx *ctx, double dt_try, double I_ramp, double rtol, double dt_min,
                double *dt_taken, double *dt_next, double *err);

/* Copy out J [N], T [N], B [2N: Br then Bz], E [N]; NULL = skip.  J, T are the state after the
 * last step; B, E are those of the last step's material evaluation (time level k).  */
int  qs_read(qs_ctx *ctx, double *J, double *T, double *B, double *E);

/* ---- extras (tests, resume, config 4, roofline runs) ----------------------------------------- */

/* Bytes of device workspace qs_init_device needs for this geometry.  */
size_t qs_workspace_bytes(const qs_geometry *geo);

/* As qs_init, but all device state lives in the caller's DEVICE buffer `workspace` (256-byte
 * aligned, >= qs_workspace_bytes(geo), owned by the caller and kept alive until qs_free) and all
 * work is enqueued on `stream` (a cudaStream_t passed as void*; NULL = default stream).  This is
 * how the Python binding lets PyTorch own device memory and streams.  */
int  qs_init_device(const qs_geometry *geo, const qs_material *mat, void *workspace,
                    size_t workspace_bytes, void *stream, qs_ctx **out);

/* Set the state (resume, prepared variants C12).  NULL J or T keeps the current array.  Resets the
 * dE/dt history of the event detector and the per-wire statistics; the previous I' is kept as the CG's initial guess (the
 * solution of the step does not depend on it beyond cg_tol).  */
int  qs_write(qs_ctx *ctx, const double *J, const double *T, double t, double I);

/* Checkpoint / resume of the solver's warm start (SURVEY.md §5 "Checkpoint / resume"; C8 "x0 = previous I'"): the
 * rate I' = dI/dt [A/s per ring, N values, caller's order] of the last step's solve (S3), which the next qs_step uses
 * as the projected CG's initial guess.  qs_read_rate copies it out; qs_write_rate sets it (host buffers).  A guess
 * only: the solution of a step does not depend on it beyond cg_tol, but a run resumed with (J, T, t, I) through
 * qs_write and I' through qs_write_rate continues with the iteration counts of the uninterrupted run.  */
int  qs_read_rate(qs_ctx *ctx, double *Idot);
int  qs_write_rate(qs_ctx *ctx, const double *Idot);

/* y = M x (C2): x [A] -> y [Wb], symmetric mutual-inductance matrix, evaluated pair by pair.  */
int  qs_matvec(qs_ctx *ctx, const double *x, double *y);
int  qs_matvec_device(qs_ctx *ctx, const double *d_x, double *d_y);

/* y = M x on FREE rings (C2: dz^2 + softening^2 for all pairs; the config-4 operator) WITHOUT ANY ALLOCATION, for
 * callers that cannot call cudaMalloc (CUDA graph capture, tight serving loops, harnesses that forbid it).  No handle:
 * the sweep's scratch memory (padded copies of r, z, x, block boxes, FP64 accumulators, work counter) is one
 * file-scope static __device__ array of 557,312 bytes, sized for at most QS_NOALLOC_MAX_RINGS rings, which every GPU
 * that loads the library holds until the process exits.
 *   d_r, d_z, d_x [n_rings]: DEVICE pointers, inputs (r > 0, finite; the ring set must satisfy qs_init's validity
 *   domain k'^2 <= 0.98 - not checked here, the data are on the device); d_y [n_rings]: DEVICE pointer, output [Wb],
 *   may alias d_x; stream: a cudaStream_t of the CURRENT device (NULL = default stream).
 * Enqueues three kernels on `stream` and returns without synchronising; calls no cudaMalloc / cudaFree / allocating
 * library routine.  The first call on a device takes the array's device address (cudaGetSymbolAddress) - a call with
 * n_rings == 0 does only that.  Rings are swept in the caller's order (no Morton re-ordering as qs_init does), so
 * scattered sets take deeper AGM classes: same numbers, more work.
 * SHARED STATE: every call uses the same array, which keeps the last call's contents; each call rewrites its inputs
 * and clears the accumulators first.  Calls that overlap on the GPU (two streams, two threads) RACE: serialise them.
 * Returns QS_OK; QS_ERR_ARG for n_rings < 0 or > QS_NOALLOC_MAX_RINGS, NULL arrays, softening <= 0; QS_ERR_CUDA.  */
#define QS_NOALLOC_MAX_RINGS 16384
int  qs_matvec_noalloc(int32_t n_rings, const double *d_r, const double *d_z, double softening,
                       const double *d_x, double *d_y, void *stream);

/* Br, Bz [N each, B = Br then Bz] of ring currents I [A] (C3), without B_ext; lattice only.  */
int  qs_field(qs_ctx *ctx, const double *I, double *B);

/* Solve M x = b (plus C^T x = 0 when the geometry has turns) by projected CG to the material's
 * cg_tol / cg_maxit; maxit_override > 0 replaces cg_maxit.  Returns 0 or QS_EV_CG_MAXIT.  */
int  qs_solve(qs_ctx *ctx, const double *b, double *x, int32_t maxit_override, int32_t *iters, double *relres);
int  qs_solve_device(qs_ctx *ctx, const double *d_b, double *d_x, int32_t maxit_override, int32_t *iters, double *relres);

/* S2 alone on the current (J, T, B) and S6 alone (m sub-steps of dt with the current Q): unit
 * parity of the pointwise passes and their HBM-roofline runs.  qs_set_fields loads B [2N] and/or
 * Q [N] (NULL = keep).  qs_heat returns m.  */
int  qs_material_eval(qs_ctx *ctx, double dt);
int  qs_set_aux(qs_ctx *ctx, int32_t on);   /* on: qs_material_eval also stores dE/dJ for qs_read_aux (off by default:
                                               the step itself never needs the array) */
int  qs_heat(qs_ctx *ctx, double dt);
int  qs_heat_adi(qs_ctx *ctx, double dt, int32_t m);   /* S6 alone by m ADI sub-steps (C15) with the current Q; returns m */
int  qs_set_fields(qs_ctx *ctx, const double *B, const double *Q);
int  qs_read_aux(qs_ctx *ctx, double *Q, double *dEdJ, double *Jc, double *rho);   /* dEdJ: see qs_set_aux */

/* Observables of the last step / solve (qs_stats_t above): CG iterations and residual (C8), the terminal voltage
 * U = -sum_w share_w V_w of the per-turn multipliers (S4; PAPER.md:99 coil voltage), Tmax and the Joule power
 * sum_i E_i J_i 2 pi r_i a_i (PAPER.md:75 source term E.J; PAPER.md:65 figures), t, I, the step's event word, and
 * the launch / pair-evaluation counters.  Host struct, filled without touching the device.  */
int  qs_stats(qs_ctx *ctx, qs_stats_t *out);

/* Test hook: make the NEXT qs_step / qs_step_rk fail after the current update S5 has been applied, to exercise the
 * transactional restore: where = 1 -> QS_ERR_CUDA reported by the heat stage; 2 -> a NaN planted in J (the step's
 * own NaN/Inf check then returns QS_ERR_NONFINITE); 0 -> cancel.  One-shot.  */
int  qs_debug_inject_failure(qs_ctx *ctx, int32_t where);

/* ---- measurement (bench.py) ---------------------------------------------------
 * Device-side timing of the library's own kernels with cudaEvent pairs recorded on the handle's
 * stream around the launches of each kernel class.  Off by default (no events are recorded).
 * qs_profile_read waits for the stream, writes the totals accumulated since the last read (or since
 * qs_profile_enable) and resets them.  ms[k] = summed launch durations of class k, launches[k] =
 * kernels launched in class k.  A class that launches m kernels back to back (the heat sub-steps of
 * one step) is bracketed once and counts m launches.  */
#define QS_PROF_SWEEP_M      0   /* K1: y = M x pair sweep                                          */
#define QS_PROF_SWEEP_FIELD  1   /* K2: fused M x + Br, Bz pair sweep                               */
#define QS_PROF_MATERIAL     2   /* K5                                                              */
#define QS_PROF_HEAT         3   /* K6 (all sub-steps of a step)                                    */
#define QS_PROF_EVENTS       4   /* K7 + step statistics                                            */
#define QS_PROF_CG_VECTOR    5   /* K3/K4 kernels of one projected-CG iteration                     */
#define QS_PROF_CLASSES      8
typedef struct {
  double  ms[QS_PROF_CLASSES];
  int64_t launches[QS_PROF_CLASSES];
} qs_profile_t;
int  qs_profile_enable(qs_ctx *ctx, int32_t on);
int  qs_profile_read(qs_ctx *ctx, qs_profile_t *out);

/* Test hook for the per-pair arithmetic of the sweeps (C2, C3): for each i, with A2 = (ri+rj)^2 + dz^2 and
 * B2 = (ri-rj)^2 + dz^2 given (host arrays [n], A2 >= B2 > 0), evaluates through evaluation class `cls`
 * (0..9, cheapest first; < 0: the class the sweep would choose from k'^2 = B2/A2) and returns
 * M = mu0 sqrt(ri rj)[(2/k - k)K - (2/k)E] [H], K(k), E(k) and the class used.  Needs no handle.  */
int  qs_pair_eval(int32_t n, const double *A2, const double *B2, int32_t cls,
                  double *M, double *K, double *E, int32_t *used);

/* FP64 FMA throughput of the current device [TFLOP/s, FMA = 2 flop]: 16 independent DFMA chains per
 * thread on every SM, timed with CUDA events (best of 5).  The denominator of the operator's
 * roofline ("bound": "alu"); needs no handle.  Returns 0 or QS_ERR_CUDA.  */
int  qs_fp64_peak(double *tflops, double *sm_clock_mhz_effective);

/* Issue-model probes behind the sweeps' roofline: SM cycles (at the maximum SM clock) per DFMA
 * warp-instruction per SM sub-partition for 8 independent chains per thread with mode 1: three distinct register
 * operands; mode 2: two register operands and an immediate; mode 3: mode 2 plus one integer ALU instruction per
 * DFMA.  Needs no handle.  */
int  qs_issue_probe(int32_t mode, double *cycles_per_dfma);
/* Per-turn state of the event detector S7 (C10) after the last step: flag word (QS_FJ_* | QS_Q_*: the paper's
 * flux-jump criterion |J/Jc| > 1, and quench criterion rho > 0.95 rho_n, plus configs[3]'s
 * T > 10 K, dE/dt spike and T > Tc), time of the first step in which any flag of the turn was set (-1: never) and the
 * number of rising edges of FJ_T|FJ_E (the per-wire flux-jump count of PAPER.md:93, Fig. 3(b)).  HOST buffers of N_w
 * entries each, NULL = skip; with constraint groups finer than wires (C16) the entries are per group.  */
int  qs_events(qs_ctx *ctx, int32_t *flags /*[N_w]*/, double *t_first /*[N_w]*/, int32_t *count /*[N_w]*/);
/* Per-wire statistics accumulated by the event pass since qs_init / the last qs_write (
 * PAPER.md:107 T_max, P_max, Q_FJ per wire; PAPER.md:119-121 Q_q, P_q, T_q at the quench time).  out: HOST buffer of
 * 8 * N_w doubles, row k of N_w entries:
 *   0 E_joule [J]  time integral of the wire's Joule power sum_i Q_i 2 pi r_i a_i
 *   1 Q_FJ [J]     the same, over the steps in which a flux-jump flag (FJ_T|FJ_E|FJ_J) of the wire is set
 *   2 P_max [W/m^3], 3 T_max [K]   running maxima of max_i Q_i and of the wire's Tmax
 *   4 t_q [s] (-1: never), 5 T_q [K], 6 P_q [W/m^3]   time, Tmax and max_i Q_i at the first step with a quench flag
 *   7 Q_q [J]      Joule energy of the wire from its first event to the quench  */
int  qs_wire_stats(qs_ctx *ctx, double *out);
/* Wait until all work enqueued on the handle's stream has finished (the *_device variants return after enqueueing;
 * SURVEY.md §8(b) "calls on one handle are serialised on its stream").  Returns 0 or QS_ERR_CUDA.  */
int  qs_sync(qs_ctx *ctx);
const char *qs_last_error(void);
/* Destroy the handle (SURVEY.md §8(b) ownership): waits for its stream, frees what qs_init allocated (workspace and
 * stream of the owning variant, pinned staging buffers, CUDA graphs); never frees caller memory - the workspace and
 * stream handed to qs_init_device stay the caller's.  NULL is a no-op.  */
void qs_free(qs_ctx *ctx);

#ifdef __cplusplus
}
#endif
#endif /* QS_H_ */
