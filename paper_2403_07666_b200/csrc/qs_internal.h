// qs_internal.h — declarations shared by the CUDA translation units of libqs (not part of the ABI).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace qs {

constexpr double kMu0 = 1.2566370614359172953850573533118e-6;   // 4 pi 1e-7
constexpr double kPi = 3.1415926535897932384626433832795;

// records the message qs_last_error() returns for the calling thread and hands back `code` (qs_api.cu)
int set_error(int code, const char* msg);

// ---- pair sweeps (qs_operator.cu) -------------------------------------------------------------
struct SweepParams {
  const double* r;        // [Np] ring radius, padded to a multiple of 32
  const double* z;        // [Np]
  const double* x;        // [Np] vector multiplied by M (padding = 0)
  const double* cur;      // [Np] ring currents whose field is wanted (FIELD sweeps; padding = 0)
  const double4* bbox;    // [nb] (rmin, rmax, zmin, zmax) of each block of 32 rings
  double* yacc;           // [Np] += sum_j S/a_inf x_j        (scale mu0 pi/2 applied by the consumer)
  double* bracc;          // [Np] += sum_j dz(-Kt + mid Qt) I_j   (scale mu0/(4 r_i) by the consumer)
  double* bzacc;          // [Np] += sum_j (Kt + c_ij Qt) I_j     (scale mu0/4 by the consumer)
  unsigned long long* counter;
  const int* done;        // fused CG: the sweep returns at once when *done != 0 (nullptr: always run)
  long long n_items;      // work items of the sweep: sweep_items(nb, field)
  int nb;
  int chunk;
  double soft_all;        // g^2 added to dz^2 of every pair (free rings) or 0 (lattice)
  double soft_self;       // extra dz^2 of the self pair (lattice: g^2)
  double minsep2;         // lower bound on the squared centre distance of two distinct rings
  double diag_d2;         // smallest B2 inside a diagonal item (self pair included)
};
int sweep_grid(int sm_count, bool field, int nb);
long long sweep_items(int nb, bool field);   // multi-target + triangle items covering every unordered block pair once
int sweep_warps_per_cta();
cudaError_t launch_sweep(const SweepParams& prm, bool field, int grid, cudaStream_t stream);
// diagM_i = M(r_i, r_i, dz^2 = d2self) in henry
cudaError_t launch_diag(int n, const double* r, double d2self, double* diagM, cudaStream_t stream);

// ---- lattice-aware operator (qs_lattice.cu): tables over (ir, jr, |iz - jz|) + block-Toeplitz sweeps ------------------
struct LatticeSweepParams {
  int Nr, Nz;
  int jr_chunk;           // source rows per CTA (set by the launcher)
  const double *TM, *TBz, *TBr;   // [Nr][Nr][Nz] unscaled pair quantities (TBz, TBr: field sweeps only)
  const double *x, *cur;  // [Nr Nz] vectors (canonical order)
  double *yacc, *bracc, *bzacc;   // accumulators, same meaning and scaling as the pair sweeps'
  const int* done;        // fused CG guard (nullptr: always run)
};
cudaError_t launch_table_build(int Nr, int Nz, double r_inner, double h, double soft_self2, double* TM, double* TBz,
                               double* TBr, int sm_count, cudaStream_t stream);
cudaError_t launch_table_sweep(const LatticeSweepParams& prm, bool field, int sm_count, cudaStream_t stream);

// block-Jacobi preconditioner of the unconstrained solve (qs_operator.cu): L [nb][32][32], 1/L_ii on the diagonal
cudaError_t launch_blockprec_build(int nb, const double* r, const double* z, double soft_all, double soft_self, double* L,
                                   cudaStream_t stream);
cudaError_t launch_blockprec_apply(int nb, int n, const double* L, const double* rvec, double* g, double* rg_out,
                                   const int* done, cudaStream_t stream);

// test hook: per-pair evaluation through evaluation class cls (or the class the sweep would pick when cls < 0)
cudaError_t launch_pair_eval(int n, const double* A2, const double* B2, int cls, double* M, double* K, double* E,
                             int* used, cudaStream_t stream);
int pair_num_classes();
// FP64 FMA throughput probe (qs_operator.cu): TFLOP/s and the SM clock seen by the kernel
cudaError_t fp64_peak_probe(double* tflops, double* sm_mhz);
cudaError_t issue_probe(int mode, double* cycles_per_dfma);

// ---- vector / CG kernels (qs_vector.cu) -------------------------------------------------------
// Device scalars of the solver; all reductions land here (no host round trip inside an iteration).
struct Scalars {
  double rg[2];          // r^T g, double buffered by iteration parity
  double pq[2];          // p^T A p, double buffered by iteration parity
  double nu2;            // reference norm squared
  double uterm;          // sum_w vsum_w = terminal voltage
  double tmax, joule;    // step statistics
  double djmax;          // max |J_new - J_old| of the step
  double thresh2;        // (cg_tol * nu)^2: the fused CG iterations stop themselves when rg <= thresh2
  int nonfinite;         // set when J or T is NaN/Inf
  int event_or;          // OR of per-turn return bits
  int done;              // fused CG: 0 running, 1 converged, 2 breakdown (p^T A p <= 0 or NaN); later launches no-op
  int iters;             // fused CG: completed iterations
  unsigned int blocks_done;   // last-block-done counter of the direction kernel
  int pad;
  double rd[2];          // patch-preconditioned solves: r^T diag(A)^-1 r, double buffered like rg - the quantity the
                         // stopping rule tests, so that it is the same rule whatever the preconditioner
};

struct VecCtx {
  int N;                 // rings
  int Np;                // padded
  int n_turns;
  const int* turn_id;    // [N] (internal order)
  const int* turn_ptr;   // [n_turns+1] CSR of cells per turn
  const int* turn_idx;   // [N]
  const double* share;   // [n_turns] share of the transport current per constraint group (C16)
  cudaStream_t stream;
  Scalars* sc;
  long long* launches;   // host counter
  int sm_count;          // SMs of the handle's device (grid sizing)
};

// ---- fused projected-CG iteration (C8): four launches after the sweep, no host round trip; every kernel returns at
// once when sc->done is set, so a batch of iterations can be enqueued blind -----------------------------------------
// patch (block-Jacobi) constraint preconditioner of the lattice solves (qs_vector.cu)
struct PatchPrec {
  int pp = 0;               // cells per patch (0: off), p x p inside one wire
  int n_patches = 0;
  int big = 0;              // 1: patches of more than 64 cells (p = 9..16): inverse per solve in global memory, the
                            //    constant part shared between the patches of one (layer, radial slot of the wire)
  int per = 1;              // patches per wire side (patches are numbered ((layer * per_layer + turn) * per + a) * per + b)
  int layers = 0, per_layer = 0;
  const int* pidx = nullptr;    // [n_patches][pp] cell of slot t of the patch
  const int* pturn = nullptr;   // [n_patches] constraint group of the patch
  double* Pm = nullptr;         // [n_patches][pp][pp] constant part M_patch [H]   (big: [layers * per][pp][pp])
  double* Pinv = nullptr;       // [n_patches][pp][pp] (M_patch + diag(shift))^-1 of the current solve
  // second level (wires larger than one patch): piecewise constants per patch, H^-1 = B + Z C Z^T with B the patch
  // inverses, Z the patch indicators and C = blockdiag over wires of (Z_w^T (M + shift) Z_w)^-1
  int nc = 0;                   // coarse unknowns per wire = per * per (0: no second level)
  double* C0m = nullptr;        // [layers][nc][nc] constant part Z^T M Z of a wire of the layer [H]
  double* C0inv = nullptr;      // [n_turns][nc][nc] coarse inverses of the current solve
  double* rc = nullptr;         // [n_patches] restricted residual Z^T r
  double* yc = nullptr;         // [n_patches] coarse correction C Z^T r
  const int* pid = nullptr;     // [N] cell -> patch
  double* h1 = nullptr;         // [N] H^-1 1
  double* sw = nullptr;         // [n_turns] per-turn Schur scalars sum h1
};
struct CgIter {
  int par;                   // parity of this iteration: rg[par] old, rg[par^1] new, pq[par]
  const double* yacc_in;     // sweep accumulators of p
  const double* shift;       // diagonal shift theta dt D (zeros for the plain operator)
  const double* Hd;          // diag(M) + shift
  const double* sw;          // per-turn Schur scalars
  double *x, *r, *g, *p, *q;
  double* tw;                // [n_turns] per-turn sums of r/H (zero on entry, zero on exit)
  double* vsum;              // [n_turns] accumulated multipliers
  double* yacc_zero;         // accumulators to clear for the next sweep (Np doubles) ...
  unsigned long long* counter;   // ... and its work counter
  double cM;
  const double* Lblk;        // non-null: block-Jacobi factors (unconstrained solves): g = B^-1 r instead of r / Hd
  int nb;                    // blocks of 32
  PatchPrec patch;           // pp > 0: patch preconditioner (sw then points to patch.sw)
};
void k_cg_Ap(const VecCtx& v, const CgIter& it);          // q = shift p + cM yacc ; pq[par] += p.q
void k_cg_update(const VecCtx& v, const CgIter& it);      // alpha = rg[par]/pq[par]; x += alpha p; r += alpha q; tw += r/H
void k_cg_project(const VecCtx& v, const CgIter& it);     // r -= tw/sw; g = r/H; rg[par^1] += r.g
void k_cg_direction(const VecCtx& v, const CgIter& it);   // p = -g + beta p; clears accumulators; last block: bookkeeping
void k_cg_begin(const VecCtx& v, double thresh2);         // done = 0, iters = 0, pq = 0, blocks_done = 0
void k_patch_build(const VecCtx& v, const PatchPrec& pc, const double* r, const double* z, double soft_all,
                   double soft_self);
void k_patch_start(const VecCtx& v, const CgIter& it, const double* shift);   // Pinv, then g, p, rg[0], vsum from the current r

// Right-hand side of the circuit equations: a given array, or (inside qs_step) evaluated on the fly from the
// material law's E as b_i = -2 pi r_i (E_i + r_i Bdot_ext / 2)   (C4)
struct Rhs {
  const double* b;       // non-null: use this array
  const double* E;       // else: E [V/m] ...
  const double* radius;  // ... ring radius [m] ...
  double Bdot;           // ... and the background-field slope [T/s]
};

// q = cM*yacc + shift*p ; pq = p.q
void k_finish_Ap(const VecCtx& v, const double* yacc, const double* shift, const double* p, double* q, double cM);
// r = cM*yacc + shift*x - b
void k_residual(const VecCtx& v, const double* yacc, const double* shift, const double* x, const Rhs& b, double* r,
                double cM);
void k_rhs_fill(const VecCtx& v, const Rhs& b, double* r);      // r = b
// alpha = rg[par]/pq ; x += alpha p ; r += alpha q
void k_update_xr(const VecCtx& v, int par, const double* p, const double* q, double* x, double* r);
// tw = sum_{i in w} r_i/H_i ; vw = tw/s_w ; vsum += vw      (one warp per turn)
void k_turn_project(const VecCtx& v, const double* r, const double* Hd, const double* sw, double* vw, double* vsum);
// s_w = sum_{i in w} 1/H_i
void k_turn_schur(const VecCtx& v, const double* Hd, double* sw);
// r -= v[turn] ; g = r/H ; rg[par] = r.g
void k_project_apply(const VecCtx& v, int par, const double* vw, const double* Hd, double* r, double* g);
// first direction p = -g ; later p = -g + (rg[par]/rg[par^1]) p ; also zeroes rg[par^1], pq for the next iteration
void k_direction(const VecCtx& v, int par, bool first, const double* g, double* p);
// deficit_w = d - sum_{i in w} x_i ; x_i += deficit_w / (H_i s_w)   (moves a warm start onto the constraint)
void k_turn_deficit(const VecCtx& v, const double* x, double d, double* defw);
void k_apply_deficit(const VecCtx& v, const double* defw, const double* Hd, const double* sw, double* x);
// ---- fused step kernels (qs_step on geometries with constraint groups) ---------------------------------------------
struct StepBegin {
  int N, n_turns;
  bool extrapolate;                 // CG start 2 I'_k - I'_{k-1} instead of I'_k
  const double *J, *H, *area;
  double *Jold, *Hold, *x, *xold, *xprev2, *cur;
  const unsigned long long *fld, *ev;           // contiguous blocks backed up word by word
  unsigned long long *fld_backup, *ev_backup;
  size_t fld_words, ev_words;
  unsigned long long* acc;          // work counter + sweep accumulators, cleared
  size_t acc_words;
  double *vsum, *tw;                // [n_turns] cleared
  unsigned long long *xmax_bits, *rmin_bits;    // [n_turns] presets of the event observables (may be null)
};
struct TurnStart {
  const int *ptr, *idx;             // CSR of cells per constraint group
  double I_ramp, cM;
  Rhs b;
  const double *Hd, *shift, *x, *yacc, *xp1, *Mxp1;
  double *r, *g, *p, *sw, *vnu, *vsum;
};
void k_step_begin(const VecCtx& v, const StepBegin& a);   // backups, CG start, I = a J, zeroing: one launch
void k_turn_fix(const VecCtx& v, double d, const double* Hd, const double* sw, double* x);   // deficit + correction
void k_turn_start(const VecCtx& v, const TurnStart& a);   // Schur scalars, reference norm, start residual, projection, p
void k_step_update(const VecCtx& v, double dt, const double* x, const double* area, double* J, const double* vsum);
void k_axpy(const VecCtx& v, double a, const double* x, double* y);                     // y += a x
void k_lincomb(const VecCtx& v, double a, const double* x, double b, double* y);        // y = a x + b y
// sc->djmax = max_i |s (x1_i - x2_i) / d_i|   (error estimate of the embedded Heun-Euler pair)
void k_max_scaled_diff(const VecCtx& v, double s, const double* x1, const double* x2, const double* d);
void k_scale_div(const VecCtx& v, double a, const double* x, const double* d, double* y);   // y += a x / d
void k_mul(const VecCtx& v, const double* a, const double* b, double* y);               // y = a b
void k_set_scalars(const VecCtx& v);                                                    // zero the Scalars block
void k_copy_rg_to_nu2(const VecCtx& v, int par);
// r = I_ramp (Mxp1 + shift xp1) - b : residual of the cold start x_p = I_ramp xp1 (reference norm, C8)
void k_nu_residual(const VecCtx& v, double I_ramp, const double* Mxp1, const double* shift, const double* xp1,
                   const Rhs& b, double* r);
// Br = mu0/(4 r) bracc ; Bz = mu0/4 bzacc + selfcoef I : output scaling of the field accumulators (qs_field)
void k_field_scale(const VecCtx& v, const double* bracc, const double* bzacc, const double* r, const double* selfcoef,
                   const double* cur, double* Br, double* Bz);
void k_sum_uterm(const VecCtx& v, const double* vsum);                                  // sc->uterm = sum vsum
void k_gather(const VecCtx& v, const double* src, const int* perm, double* dst, int n, int npad);   // dst[k] = src[perm[k]], pad 0
void k_scatter_scaled(const VecCtx& v, const double* src, const int* perm, double* dst, int n, double scale);  // dst[perm[k]] = scale*src[k]

// ---- pointwise passes (qs_pointwise.cu) ---------------------------------------------------------
struct MaterialParams {
  double Ec, n_exp, Jc0, Tc, B0, eps_coef, eps_exp, Y, rho_n;
  double C3, C1, k_in, k_between, theta;
  double T_fluxjump, dEdt_spike;
  int n_int;             // n_exp when it is a small integer, else 0
};
struct LatticeParams {
  int Nr, Nz, n;         // cells along r, along z, per wire side
  double h, r_inner;
  double h_conv[4];
  double T_bath;
  // face and border coefficients of the finite-volume heat step divided by the cell volume (C9), set up at init:
  //   hr_p[ir] = kappa(ir|ir+1) (r_c + h/2) / (2 h^2 r_c)   (0 on the outer border)     hr_m likewise for ir-1|ir
  //   hz_p[iz] = kappa(iz|iz+1) / (2 h^2)                    (0 on the border)           hz_m likewise
  //   rb_r[ir], rb_z[iz] = Robin film coefficient x border face area / cell volume (0 for interior rows / columns)
  const double *hr_p, *hr_m, *rb_r;   // [Nr]
  const double *hz_p, *hz_m, *rb_z;   // [Nz]
};
struct MaterialArgs {
  int N;
  int Nz;                // > 0: lattice, per-row geometry from rowtab[i / Nz]; 0: per-cell arrays r, area, selfcoef, diagM
  const double *J, *H, *jc0_scale, *bracc, *bzacc;
  const double4* rowtab; // [Nr] (r, selfcoef, diagM, area) of the cells of radial row ir
  const double *r, *area, *selfcoef, *diagM;
  double *Br, *Bz;       // read when !from_acc, written when from_acc
  double *E, *Q, *shift, *Hd;
  double *dEdJ, *Jc, *rho;   // optional (test hook qs_read_aux), may be null: the step itself never stores them
  // per-turn event observables folded into this pass (C10; lattice with turns only, else null):
  // bit patterns of max |J|/Jc and min rho over the cells of each turn, combined with 64-bit atomics
  const int* rowturn;    // [Nr] (ir / n) * turns_per_layer, when the caller's turn ids are the canonical l*Tn + tau
  const int* turn_id;    // else: per-cell turn ids
  int cells_per_side;    // n
  unsigned long long *xmax_bits, *rmin_bits;   // [n_turns], preset to 0 and ~0
  double Bext, Bdot, dt;
  double inv_area;       // lattice: 1 / (h h)
  bool from_acc;         // true: B from the sweep accumulators (+ self + Bext); false: B arrays given
};
void k_build_rowtab(const VecCtx& v, int Nr, int Nz, const double* r, const double* selfcoef, const double* diagM,
                    const double* area, double4* rowtab);
void k_material(const VecCtx& v, const MaterialParams& mp, const MaterialArgs& a);
void k_enthalpy_from_T(const VecCtx& v, const MaterialParams& mp, const double* T, double* H, int n);
void k_T_from_enthalpy(const VecCtx& v, const MaterialParams& mp, const double* H, double* T, int n);
void k_heat_substep(const VecCtx& v, const MaterialParams& mp, const LatticeParams& lp, const double* Hin,
                    const double* Q, double* Hout, double dtsub);
// all m sub-steps in one launch for lattices small enough to live in one SM; false: not applicable (use k_heat_substep)
bool k_heat_all_substeps(const VecCtx& v, const MaterialParams& mp, const LatticeParams& lp, int m, const double* Hin,
                         const double* Q, double* Hout, double dtsub);
// one ADI sub-step (qs_adi.cu, C15); scratch: six arrays of N doubles; returns the number of launches
// temporally blocked explicit heat sub-steps: msub <= k_heat_block_max() sub-steps of length dtsub in one launch
int k_heat_block_max();
void k_heat_block(const VecCtx& v, const MaterialParams& mp, const LatticeParams& lp, int msub, const double* Hin,
                  const double* Q, double* Hout, double dtsub);
// opt-in shared-memory sizes of the heat kernels on the CURRENT device (cudaFuncSetAttribute is per device): called by
// every qs_init with the handle's device current
void pointwise_prepare_device();
int k_heat_adi_substep(const VecCtx& v, const MaterialParams& mp, const LatticeParams& lp, const double* Hin,
                       const double* Q, double* Hout, double delta, double* const scratch[6]);
struct EventArgs {
  const double *H, *E;
  const unsigned long long *xmax_bits, *rmin_bits;   // per turn, from the material pass
  const double *Q, *r, *area;   // Joule power density, ring radius and cross-section per cell (per-wire statistics)
  const double *J = nullptr, *Jold = nullptr;   // non-null: the step statistics (max |dJ|, Tmax, Joule power, NaN/Inf check)
                                                // are taken in this pass too and k_step_stats is not launched
  double* wire;          // [9][n_turns]: E_joule, Q_FJ, P_max, T_max, t_q, T_q, P_q, Q_q, E_at_first (f3)
  double* ebar_prev;     // [n_turns]
  int* flags;            // [n_turns]
  double* t_first;       // [n_turns]
  int* count;            // [n_turns]
  double dt, t_new;
  bool have_prev;
};
void k_events(const VecCtx& v, const MaterialParams& mp, const EventArgs& e);
void k_step_stats(const VecCtx& v, const MaterialParams& mp, const double* J, const double* Jold, const double* H,
                  const double* Q, const double* r, const double* area);

}  // namespace qs
