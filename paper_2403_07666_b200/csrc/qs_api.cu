// qs_api.cu — the C ABI of include/qs.h: context, workspace layout, step driver (S1..S7), projected CG.
//
// Host code only enqueues kernels on the handle's stream and reads back one small Scalars block per CG
// iteration (the convergence test) and per step (events, statistics).  No arithmetic of the method runs
// on the host except set-up constants (bounding boxes, Morton order of free rings, self-field coefficients).
// Every entry point makes the handle's device current for the duration of the call (DeviceGuard).
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <string>
#include <vector>

#include "../../include/qs.h"
#include "qs_internal.h"

using namespace qs;

namespace {

thread_local std::string g_err;
int fail(int code, const std::string& msg) {
  g_err = msg;
  return code;
}
#define QS_CUDA(call)                                                                          \
  do {                                                                                         \
    cudaError_t e_ = (call);                                                                   \
    if (e_ != cudaSuccess)                                                                     \
      return fail(QS_ERR_CUDA, std::string(#call) + ": " + cudaGetErrorString(e_));            \
  } while (0)

size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }
}  // namespace
namespace qs {
int set_error(int code, const char* msg) { return fail(code, msg); }
}  // namespace qs
namespace {

// Carves named arrays out of one device buffer; used twice (size query with base == nullptr, then for real).
struct Carver {
  char* base;
  size_t off = 0;
  explicit Carver(void* b) : base(static_cast<char*>(b)) {}
  template <class T>
  T* take(size_t count) {
    off = align_up(off, 256);
    T* p = base ? reinterpret_cast<T*>(base + off) : nullptr;
    off += count * sizeof(T);
    return p;
  }
};

// Makes `dev` the current CUDA device for the lifetime of the guard (handles may live on different devices of one
// process; kernels, events and copies of a handle must be issued with its device current).
struct DeviceGuard {
  int prev = -1;
  bool switched = false;
  explicit DeviceGuard(int dev) {
    if (cudaGetDevice(&prev) == cudaSuccess && prev != dev) switched = cudaSetDevice(dev) == cudaSuccess;
  }
  ~DeviceGuard() {
    if (switched) cudaSetDevice(prev);
  }
  DeviceGuard(const DeviceGuard&) = delete;
  DeviceGuard& operator=(const DeviceGuard&) = delete;
};

}  // namespace

// cudaEvent pairs around kernel classes (qs_profile_*): recorded only while enabled
struct Profiler {
  struct Rec { int cls; int n; cudaEvent_t a, b; };
  bool on = false;
  std::vector<Rec> pending;
  std::vector<std::pair<cudaEvent_t, cudaEvent_t>> pool;
  double ms[QS_PROF_CLASSES] = {};
  long long launches[QS_PROF_CLASSES] = {};
  cudaEvent_t cur_a = nullptr, cur_b = nullptr;
  void begin(cudaStream_t st) {
    if (!on) return;
    if (pool.empty()) {
      cudaEvent_t a, b;
      cudaEventCreate(&a);
      cudaEventCreate(&b);
      pool.emplace_back(a, b);
    }
    cur_a = pool.back().first;
    cur_b = pool.back().second;
    pool.pop_back();
    cudaEventRecord(cur_a, st);
  }
  void end(cudaStream_t st, int cls, int n) {
    if (!on) return;
    cudaEventRecord(cur_b, st);
    pending.push_back({cls, n, cur_a, cur_b});
    if (pending.size() >= 4096) fold(st);
  }
  void fold(cudaStream_t st) {
    if (pending.empty()) return;
    cudaStreamSynchronize(st);
    for (const Rec& r : pending) {
      float t = 0.f;
      if (cudaEventElapsedTime(&t, r.a, r.b) == cudaSuccess) ms[r.cls] += t;
      launches[r.cls] += r.n;
      pool.emplace_back(r.a, r.b);
    }
    pending.clear();
  }
  void reset() {
    for (int k = 0; k < QS_PROF_CLASSES; ++k) ms[k] = 0.0, launches[k] = 0;
  }
  void destroy() {
    for (const Rec& r : pending) pool.emplace_back(r.a, r.b);
    pending.clear();
    for (auto& e : pool) {
      cudaEventDestroy(e.first);
      cudaEventDestroy(e.second);
    }
    pool.clear();
  }
};

struct qs_ctx {
  Profiler prof;
  // problem
  int N = 0, Np = 0, nb = 0, n_turns = 0;
  bool lattice = false, has_operator = true;
  bool tables = false;               // QS_GEO_LATTICE_TABLES: block-Toeplitz operator
  bool blockprec = false;            // free rings without constraints: block-Jacobi preconditioned CG in qs_solve
  double *TM = nullptr, *TBz = nullptr, *TBr = nullptr;   // [Nr][Nr][Nz]
  MaterialParams mp{};
  LatticeParams lp{};
  double theta = 1.0, cg_tol = 1e-10;
  int cg_maxit = 20000;
  double Bext0 = 0, Bext_rate = 0, Bext_max = 0;
  double soft_all = 0, soft_self = 0, minsep2 = 0, diag_d2 = 0;
  std::vector<int> perm;             // internal k -> caller index (empty = identity)
  // device
  cudaStream_t stream = nullptr;
  void* owned = nullptr;             // cudaMalloc'ed workspace (qs_init) or nullptr (qs_init_device)
  int sm_count = 148;
  int device = 0;                    // the CUDA device the handle lives on (current at qs_init)
  int inject = 0;                    // qs_debug_inject_failure: 1 = CUDA error in the heat stage, 2 = NaN in J after S5
  // transactional step: the derived fields (Br, Bz, E) and the per-turn event state (wire statistics, ebar_prev,
  // t_first, flags, count) are each one contiguous block with a backup block of the same size
  char *fld_begin = nullptr, *fld_backup = nullptr, *ev_begin = nullptr, *ev_backup = nullptr;
  size_t fld_bytes = 0, ev_bytes = 0;
  bool have_prev_E_old = false;
  bool backup_valid = false;         // the backups belong to the step in flight (restore_state copies them back only then)
  double *r, *z, *area, *jc0s, *selfcoef, *diagM;
  double *J, *Jold, *Ha, *Hb, *Hold, *Br, *Bz, *E, *dEdJ, *Q, *b, *shift, *Hd, *Jc, *rho;
  double *x, *xold, *cur, *p, *q, *rr, *g, *xp1, *Mxp1, *tmp, *tmp2, *zero;
  double* xprev2 = nullptr;          // I' of the step before the last (extrapolated CG start)
  int n_prev = 0;                    // how many consecutive previous solutions are stored (0..2)
  double last_dt = 0.0, last_ramp = 0.0;
  unsigned long long* counter;       // followed contiguously by yacc, bracc, bzacc (one memset)
  double *yacc, *bracc, *bzacc;
  size_t acc_bytes = 0;
  double *sw, *swM, *vw, *vsum, *tw, *defw, *ebar_prev, *t_first;
  double* wire = nullptr;            // [9][n_turns] per-wire statistics (f3)
  double* share = nullptr;           // [n_turns] transport-current share of each constraint group (C16)
  int *flags, *count, *turn_ptr, *turn_idx, *turn_id, *d_perm;
  int* rowturn = nullptr;            // [Nr] (ir / n) * turns_per_layer
  unsigned long long *xmax_bits = nullptr, *rmin_bits = nullptr;   // [n_turns] event observables of the material pass
  double4* rowtab = nullptr;         // [Nr] (r, selfcoef, diagM, area) per radial row of a lattice
  // CUDA graphs of two fused CG iterations (parities 0, 1), keyed by the vectors they were captured with
  struct CgGraph {
    const double *x = nullptr, *shift = nullptr, *Hd = nullptr, *sw = nullptr;
    bool patch = false;
    cudaGraphExec_t exec = nullptr;
    int launches = 0;
  } cg_graph[2];
  // CUDA graphs of the m explicit heat sub-steps of one step (launch-bound on lattices that live in L2), keyed by the
  // buffer the step starts from, m and the sub-step length
  struct HeatGraph {
    const double* H = nullptr;
    int m = 0;
    double sub = 0.0;
    cudaGraphExec_t exec = nullptr;
  } heat_graph[2];
  bool heat_force_blocked = false;   // QS_GEO_HEAT_BLOCKED: temporally blocked heat kernel at any lattice size (measurement)
  bool canonical_turns = false;      // turn_id[c] == (ir / n) * turns_per_layer + iz / n for every cell
  bool aux_on = false;               // qs_material_eval also writes dE/dJ (after the first qs_read_aux)
  double last_eval_dt = 0.0;
  double* adi[6] = {nullptr, nullptr, nullptr, nullptr, nullptr, nullptr};   // ADI scratch (lattice only)
  int adi_m = 0;                     // material.heat_adi_substeps
  double* heat_tab = nullptr;        // hr_p, hr_m, rb_r [Nr each], hz_p, hz_m, rb_z [Nz each]
  int tabNr = 0, tabNz = 0;
  double4* bbox;
  double* Lblk = nullptr;            // [nb][32][32] block-Jacobi factors of M (free rings: unconstrained solves)
  PatchPrec patch;                   // patch preconditioner of the lattice solves (pp = 0: off)
  int* pidx = nullptr;               // [N] patch slot -> cell
  int* pturn = nullptr;              // [N / pp] patch -> constraint group
  int* pid = nullptr;                // [N] cell -> patch (second level of the patch preconditioner)
  Scalars* sc;
  Scalars* h_sc = nullptr;           // pinned
  double* h_stage = nullptr;         // pinned staging, 2N doubles
  double* H = nullptr;               // current enthalpy (Ha or Hb)
  double* Halt = nullptr;
  // state
  double t = 0, I = 0;
  bool have_prev_E = false;
  long long launches = 0, pair_evals = 0;
  qs_stats_t st{};
  VecCtx v{};
};

namespace {

void carve(qs_ctx* c, void* base, size_t* total) {
  Carver k(base);
  const size_t N = c->N, Np = c->Np, nt = std::max(c->n_turns, 1);
  c->r = k.take<double>(Np);
  c->z = k.take<double>(Np);
  c->area = k.take<double>(N);
  c->jc0s = k.take<double>(N);
  c->selfcoef = k.take<double>(N);
  c->diagM = k.take<double>(N);
  c->J = k.take<double>(N);
  c->Jold = k.take<double>(N);
  c->Ha = k.take<double>(N);
  c->Hb = k.take<double>(N);
  c->Hold = k.take<double>(N);
  k.off = align_up(k.off, 256);
  const size_t fld0 = k.off;
  c->fld_begin = base ? static_cast<char*>(base) + fld0 : nullptr;
  c->Br = k.take<double>(N);
  c->Bz = k.take<double>(N);
  c->E = k.take<double>(N);
  c->fld_bytes = k.off - fld0;
  c->fld_backup = reinterpret_cast<char*>(k.take<char>(c->fld_bytes));
  c->dEdJ = k.take<double>(N);
  c->Q = k.take<double>(N);
  c->b = k.take<double>(N);
  c->shift = k.take<double>(N);
  c->Hd = k.take<double>(N);
  c->Jc = k.take<double>(N);
  c->rho = k.take<double>(N);
  c->x = k.take<double>(Np);
  c->xold = k.take<double>(Np);
  c->xprev2 = k.take<double>(Np);
  c->cur = k.take<double>(Np);
  c->p = k.take<double>(Np);
  c->q = k.take<double>(N);
  c->rr = k.take<double>(N);
  c->g = k.take<double>(N);
  c->xp1 = k.take<double>(N);
  c->Mxp1 = k.take<double>(N);
  c->tmp = k.take<double>(Np);
  c->tmp2 = k.take<double>(Np);
  c->zero = k.take<double>(N);
  // counter + accumulators: contiguous, zeroed by one memset per sweep
  k.off = align_up(k.off, 256);
  const size_t acc0 = k.off;
  c->counter = k.take<unsigned long long>(32);
  c->yacc = k.take<double>(Np);
  c->bracc = k.take<double>(Np);
  c->bzacc = k.take<double>(Np);
  c->acc_bytes = k.off - acc0;
  c->sw = k.take<double>(nt);
  c->swM = k.take<double>(nt);
  c->vw = k.take<double>(nt);
  c->vsum = k.take<double>(nt);
  c->tw = k.take<double>(nt);
  c->defw = k.take<double>(nt);
  c->share = k.take<double>(nt);
  k.off = align_up(k.off, 256);
  const size_t ev0 = k.off;
  c->ev_begin = base ? static_cast<char*>(base) + ev0 : nullptr;
  c->ebar_prev = k.take<double>(nt);
  c->t_first = k.take<double>(nt);
  c->wire = k.take<double>(9 * nt);
  c->flags = k.take<int>(nt);
  c->count = k.take<int>(nt);
  c->ev_bytes = k.off - ev0;
  c->ev_backup = reinterpret_cast<char*>(k.take<char>(c->ev_bytes));
  c->turn_ptr = k.take<int>(nt + 1);
  c->turn_idx = k.take<int>(N);
  c->turn_id = k.take<int>(N);
  c->d_perm = k.take<int>(N);
  c->bbox = k.take<double4>(std::max(c->nb, 1));
  if (c->blockprec) c->Lblk = k.take<double>(static_cast<size_t>(c->nb) * 1024);
  if (c->patch.pp > 0) {
    const size_t pp = c->patch.pp;
    c->pidx = k.take<int>(N);
    c->pturn = k.take<int>(N / pp);
    c->patch.Pm = k.take<double>(c->patch.big ? static_cast<size_t>(c->patch.layers) * c->patch.per * pp * pp : N * pp);
    c->patch.Pinv = k.take<double>(N * pp);
    if (c->patch.nc > 0) {
      const size_t nc = c->patch.nc;
      c->patch.C0m = k.take<double>(static_cast<size_t>(c->patch.layers) * nc * nc);
      c->patch.C0inv = k.take<double>(static_cast<size_t>(nt) * nc * nc);
      c->patch.rc = k.take<double>(N / pp);
      c->patch.yc = k.take<double>(N / pp);
      c->pid = k.take<int>(N);
    }
    c->patch.h1 = k.take<double>(N);
    c->patch.sw = k.take<double>(nt);
  }
  if (c->tables) {
    const size_t nt3 = static_cast<size_t>(c->tabNr) * c->tabNr * c->tabNz;
    c->TM = k.take<double>(nt3);
    c->TBz = k.take<double>(nt3);
    c->TBr = k.take<double>(nt3);
  }
  if (c->tabNr > 0)
    for (int q = 0; q < 6; ++q) c->adi[q] = k.take<double>(N);
  c->heat_tab = k.take<double>(3 * static_cast<size_t>(c->tabNr + c->tabNz) + 1);
  c->rowtab = k.take<double4>(static_cast<size_t>(c->tabNr) + 1);
  c->rowturn = k.take<int>(static_cast<size_t>(c->tabNr) + 1);
  c->xmax_bits = k.take<unsigned long long>(nt);   // xmax_bits and rmin_bits are contiguous: one reset
  c->rmin_bits = k.take<unsigned long long>(nt);
  c->sc = k.take<Scalars>(1);
  *total = align_up(k.off, 256);
}

int check_geometry(const qs_geometry* g) {
  if (!g || g->n_rings <= 0 || !g->r || !g->z || !g->area) return fail(QS_ERR_ARG, "geometry: NULL array or n_rings <= 0");
  if (g->n_turns < 0 || (g->n_turns > 0 && !g->turn_id)) return fail(QS_ERR_ARG, "geometry: n_turns without turn_id");
  if (!(g->softening > 0.0)) return fail(QS_ERR_ARG, "geometry: softening must be > 0");
  if (g->turn_share)
    for (int w = 0; w < g->n_turns; ++w)
      if (!std::isfinite(g->turn_share[w])) return fail(QS_ERR_ARG, "geometry: turn_share must be finite");
  if (g->lattice) {
    if (g->layers <= 0 || g->turns_per_layer <= 0 || g->cells_per_side <= 0 || !(g->wire_size > 0.0))
      return fail(QS_ERR_ARG, "geometry: bad lattice description");
    const long long n = g->cells_per_side, Nr = g->layers * n, Nz = g->turns_per_layer * n;
    if (Nr * Nz != g->n_rings) return fail(QS_ERR_ARG, "geometry: n_rings != Nr*Nz");
  }
  return QS_OK;
}

// Side p of the square patches of the patch preconditioner (0: not applicable): lattices whose constraint groups are
// the wires in canonical numbering.  p = the wire side up to 16 x 16 cells (configs 0, 2, 3: the patch is the wire, which
// is what halves the iterations); larger wires (config 1's 64 x 64) and QS_GEO_PATCH_SUBWIRE take the largest divisor
// <= 8 (16 x 16 patches of config 1 were measured: 50 against 57 iterations per step, and 9.6 against 4.2 ms per step
// for the inversions).
int patch_side(const qs_geometry* g) {
  if (!g->lattice || (g->flags & (QS_GEO_NO_OPERATOR | QS_GEO_NO_PATCH_PRECOND)) || g->n_turns <= 0) return 0;
  const int n = g->cells_per_side;
  if (n < 2 || g->n_turns != g->layers * g->turns_per_layer) return 0;
  const long long Nz = static_cast<long long>(g->turns_per_layer) * n;
  for (long long k = 0; k < g->n_rings; ++k)
    if (g->turn_id[k] != (k / Nz / n) * g->turns_per_layer + (k % Nz) / n) return 0;
  if (n <= 16 && !(g->flags & QS_GEO_PATCH_SUBWIRE)) return n;   // the whole wire
  int p = 1;
  for (int d = 2; d <= 8 && d <= n; ++d)
    if (n % d == 0) p = d;
  return p >= 2 ? p : 0;
}
void patch_setup(PatchPrec* pc, const qs_geometry* g, int N) {
  const int ps = patch_side(g);
  pc->pp = ps * ps;
  pc->n_patches = ps ? N / (ps * ps) : 0;
  pc->big = ps > 8;
  pc->per = ps ? g->cells_per_side / ps : 1;
  // second level for wires of several patches (at most 64 patches per wire), unless the plain patches are asked for
  pc->nc = (ps && pc->per > 1 && pc->per * pc->per <= 64 && !(g->flags & QS_GEO_PATCH_SUBWIRE)) ? pc->per * pc->per : 0;
  pc->layers = g->layers;
  pc->per_layer = g->turns_per_layer;
}

int sync_scalars(qs_ctx* c) {
  QS_CUDA(cudaMemcpyAsync(c->h_sc, c->sc, sizeof(Scalars), cudaMemcpyDeviceToHost, c->stream));
  QS_CUDA(cudaStreamSynchronize(c->stream));
  return QS_OK;
}

// y-accumulators <- sweep of (x [, cur]); consumer applies the scale factors.  prezeroed: the accumulators and the
// work counter were cleared by the previous CG iteration (fused path), no memset is enqueued.
int do_sweep(qs_ctx* c, const double* x, const double* cur, bool field, bool prezeroed = false, bool cg_guard = false) {
  if (!prezeroed) QS_CUDA(cudaMemsetAsync(c->counter, 0, c->acc_bytes, c->stream));
  if (c->tables) {   // lattice-aware operator: block-Toeplitz product with the tables built at init
    LatticeSweepParams lp;
    lp.Nr = c->lp.Nr;
    lp.Nz = c->lp.Nz;
    lp.jr_chunk = 0;
    lp.TM = c->TM;
    lp.TBz = c->TBz;
    lp.TBr = c->TBr;
    lp.x = x;
    lp.cur = cur ? cur : x;
    lp.yacc = c->yacc;
    lp.bracc = c->bracc;
    lp.bzacc = c->bzacc;
    lp.done = cg_guard ? &c->sc->done : nullptr;
    c->prof.begin(c->stream);
    QS_CUDA(launch_table_sweep(lp, field, c->sm_count, c->stream));
    c->prof.end(c->stream, field ? QS_PROF_SWEEP_FIELD : QS_PROF_SWEEP_M, 1);
    ++c->launches;
    ++c->st.sweeps;
    return QS_OK;
  }
  SweepParams prm;
  prm.r = c->r;
  prm.z = c->z;
  prm.x = x;
  prm.cur = cur ? cur : x;
  prm.bbox = c->bbox;
  prm.yacc = c->yacc;
  prm.bracc = c->bracc;
  prm.bzacc = c->bzacc;
  prm.counter = c->counter;
  prm.done = cg_guard ? &c->sc->done : nullptr;
  prm.nb = c->nb;
  prm.n_items = sweep_items(c->nb, field);
  prm.soft_all = c->soft_all;
  prm.soft_self = c->soft_self;
  prm.minsep2 = c->minsep2;
  prm.diag_d2 = c->diag_d2;
  const int wpc = sweep_warps_per_cta();
  int grid = sweep_grid(c->sm_count, field, c->nb);
  const long long need = (prm.n_items + wpc - 1) / wpc;
  if (need < grid) grid = static_cast<int>(need);
  const long long warps = static_cast<long long>(grid) * wpc;
  prm.chunk = static_cast<int>(std::max<long long>(1, std::min<long long>(32, prm.n_items / (warps * 8))));
  c->prof.begin(c->stream);
  QS_CUDA(launch_sweep(prm, field, grid, c->stream));
  c->prof.end(c->stream, field ? QS_PROF_SWEEP_FIELD : QS_PROF_SWEEP_M, 1);
  ++c->launches;
  c->pair_evals += (static_cast<long long>(c->nb) * (c->nb + 1) / 2) * 1024;   // every unordered block pair once
  ++c->st.sweeps;
  return QS_OK;
}

constexpr double kCM = 0.5 * kMu0 * kPi;   // yacc -> henry * ampere
constexpr long long kHeatBlockedMaxCells = 2000000;   // H, Q, H' of 2 M cells = 48 MB: well inside the 126 MB L2

// Projected CG (C8) on A = M + diag(shift), constraint C^T x = const kept by the projection.
// In: x satisfies the constraint; if yacc_has_Mx the accumulators hold the sweep of x.  nu < 0: nu = start norm.
// Iterations are enqueued in batches without a host round trip: the kernels stop themselves (Scalars::done) at the
// iteration where sqrt(r^T g) <= tol nu, so the result is the one of the iteration-by-iteration loop.
// prepared: r, g, p, rg[0], vsum and the reference norm (Scalars::nu2) were produced by k_turn_start (fused step path);
// nu_out receives the reference norm used.
int cg_core(qs_ctx* c, const Rhs& b, double* x, const double* shift, const double* Hd, const double* sw,
            bool yacc_has_Mx, double tol, int maxit, double nu, int* iters, double* relres, bool* hit_max,
            const double* Lblk = nullptr, bool prepared = false, double* nu_out = nullptr) {
  const VecCtx& v = c->v;
  int rc;
  if (!prepared) {
    if (!yacc_has_Mx && (rc = do_sweep(c, x, nullptr, false)) != QS_OK) return rc;
    k_residual(v, c->yacc, shift, x, b, c->rr, kCM);
    if (c->n_turns) QS_CUDA(cudaMemsetAsync(c->vsum, 0, sizeof(double) * c->n_turns, c->stream));
    k_turn_project(v, c->rr, Hd, sw, c->vw, c->vsum);
    if (Lblk) {   // block-Jacobi preconditioner: g = B^-1 r, rg[0] = r.g (rg[0] is zero on entry)
      QS_CUDA(launch_blockprec_apply(c->nb, c->N, Lblk, c->rr, c->g, &c->sc->rg[0], nullptr, c->stream));
      ++c->launches;
    } else {
      k_project_apply(v, 0, c->vw, Hd, c->rr, c->g);
    }
    k_direction(v, 0, true, c->g, c->p);
  }
  if ((rc = sync_scalars(c)) != QS_OK) return rc;
  double rg = c->h_sc->rg[0];
  if (prepared) nu = std::sqrt(std::max(c->h_sc->nu2, 0.0));
  if (nu < 0.0) nu = std::sqrt(std::max(rg, 0.0));
  if (nu_out) *nu_out = nu;
  *hit_max = false;
  *iters = 0;
  if (!(rg == rg)) return fail(QS_ERR_NONFINITE, "CG: r^T g is NaN");
  if (nu == 0.0 || std::sqrt(std::max(rg, 0.0)) <= tol * nu) {
    *relres = nu > 0.0 ? std::sqrt(std::max(rg, 0.0)) / nu : 0.0;
    return QS_OK;
  }
  if (maxit <= 0) {
    *hit_max = true;
    *relres = std::sqrt(std::max(rg, 0.0)) / nu;
    return QS_OK;
  }
  // fused iterations
  QS_CUDA(cudaMemsetAsync(c->counter, 0, c->acc_bytes, c->stream));
  if (c->n_turns) QS_CUDA(cudaMemsetAsync(c->tw, 0, sizeof(double) * c->n_turns, c->stream));
  k_cg_begin(v, (tol * nu) * (tol * nu));
  CgIter it;
  it.yacc_in = c->yacc;
  it.shift = shift;
  it.Hd = Hd;
  it.sw = sw;
  it.x = x;
  it.r = c->rr;
  it.g = c->g;
  it.p = c->p;
  it.q = c->q;
  it.tw = c->tw;
  it.vsum = c->vsum;
  it.yacc_zero = c->yacc;
  it.counter = c->counter;
  it.cM = kCM;
  it.Lblk = Lblk;
  it.nb = c->nb;
  // lattice solves with wires as constraint groups: patch (block-Jacobi) preconditioner, set up only now that the solve
  // really iterates - the block projection replaces the diagonal one from here on (the multipliers keep accumulating)
  const bool use_patch = c->patch.pp > 0 && c->n_turns > 0 && !Lblk;
  if (use_patch) {
    it.patch = c->patch;
    it.sw = c->patch.sw;
    it.par = 0;
    k_patch_start(v, it, shift);
  }
  // one iteration = sweep + four vector kernels; pairs of iterations are replayed from a CUDA graph (captured on
  // first use for this set of vectors) unless the event profiler is recording
  auto enqueue_iteration = [&](int par) -> int {
    it.par = par;
    int r2 = do_sweep(c, c->p, nullptr, false, true, true);
    if (r2 != QS_OK) return r2;
    c->prof.begin(c->stream);
    k_cg_Ap(v, it);
    k_cg_update(v, it);
    k_cg_project(v, it);
    k_cg_direction(v, it);
    c->prof.end(c->stream, QS_PROF_CG_VECTOR, 4);
    return QS_OK;
  };
  qs_ctx::CgGraph* graph = nullptr;
  if (!c->prof.on) {
    for (auto& gslot : c->cg_graph)
      if (gslot.exec && gslot.x == x && gslot.shift == shift && gslot.Hd == Hd && gslot.sw == sw && gslot.patch == use_patch)
        graph = &gslot;
    if (!graph) {
      qs_ctx::CgGraph& gslot = c->cg_graph[c->cg_graph[0].exec ? 1 : 0];
      if (gslot.exec) {
        cudaGraphExecDestroy(gslot.exec);
        gslot.exec = nullptr;
      }
      const long long l0 = c->launches, p0 = c->pair_evals;
      const int s0 = c->st.sweeps;
      cudaGraph_t gr = nullptr;
      if (cudaStreamBeginCapture(c->stream, cudaStreamCaptureModeRelaxed) == cudaSuccess) {
        const bool ok = enqueue_iteration(0) == QS_OK && enqueue_iteration(1) == QS_OK;
        const cudaError_t ec = cudaStreamEndCapture(c->stream, &gr);
        if (ok && ec == cudaSuccess && gr && cudaGraphInstantiate(&gslot.exec, gr, 0) == cudaSuccess) {
          gslot.x = x, gslot.shift = shift, gslot.Hd = Hd, gslot.sw = sw, gslot.patch = use_patch;
          gslot.launches = static_cast<int>(c->launches - l0);
          graph = &gslot;
        } else {
          gslot.exec = nullptr;
          cudaGetLastError();
        }
        if (gr) cudaGraphDestroy(gr);
      }
      c->launches = l0;        // capture enqueued nothing
      c->pair_evals = p0;
      c->st.sweeps = s0;
    }
  }
  const long long evals_per_sweep = c->tables ? 0 : (static_cast<long long>(c->nb) * (c->nb + 1) / 2) * 1024;
  int enq = 0, batch = 2;
  for (;;) {
    const int todo = std::min(batch, maxit - enq);
    int k = 0;
    while (k < todo) {
      if (graph && (enq & 1) == 0 && k + 2 <= todo) {
        QS_CUDA(cudaGraphLaunch(graph->exec, c->stream));
        c->launches += graph->launches;
        c->pair_evals += 2 * evals_per_sweep;
        c->st.sweeps += 2;
        k += 2, enq += 2;
      } else {
        if ((rc = enqueue_iteration(enq & 1)) != QS_OK) return rc;
        ++k, ++enq;
      }
    }
    if ((rc = sync_scalars(c)) != QS_OK) return rc;
    if (c->h_sc->done == 2) return fail(QS_ERR_CG, "CG breakdown: p^T A p <= 0 or NaN");
    if (c->h_sc->done == 1 || enq >= maxit) break;
    batch = std::min(16, batch * 2);
  }
  const int done_it = c->h_sc->iters;
  rg = use_patch ? c->h_sc->rd[done_it & 1] : c->h_sc->rg[done_it & 1];
  *iters = done_it;
  *hit_max = c->h_sc->done != 1;
  *relres = std::sqrt(std::max(rg, 0.0)) / nu;
  // no-op launches after convergence did not run; the sweep count reflects the enqueued ones: correct it
  c->st.sweeps -= (enq - done_it);
  if (!c->tables)
    c->pair_evals -= static_cast<long long>(enq - done_it) * (static_cast<long long>(c->nb) * (c->nb + 1) / 2) * 1024;
  return QS_OK;
}

double bext_at(const qs_ctx* c, double t) {
  if (c->Bext_rate == 0.0) return c->Bext0;
  return std::min(c->Bext0 + c->Bext_rate * t, c->Bext_max);
}

int heat_substeps_count(const qs_ctx* c, double dt) {
  const double alpha0 = c->mp.k_in / (c->mp.C3 * c->lp.T_bath * c->lp.T_bath + c->mp.C1);
  const double limit = 0.8 * c->lp.h * c->lp.h / (4.0 * alpha0);
  return std::max(1, static_cast<int>(std::ceil(dt / limit)));
}

int run_heat_adi(qs_ctx* c, double dt, int m) {
  const double delta = dt / m;
  c->prof.begin(c->stream);
  int launches = 0;
  for (int s = 0; s < m; ++s) {
    launches += k_heat_adi_substep(c->v, c->mp, c->lp, c->H, c->Q, c->Halt, delta, c->adi);
    std::swap(c->H, c->Halt);
  }
  c->prof.end(c->stream, QS_PROF_HEAT, launches);
  QS_CUDA(cudaGetLastError());
  return QS_OK;
}

int run_heat(qs_ctx* c, double dt, int* m_out) {
  if (c->adi_m > 0) {   // C15: the paper's ADI scheme instead of the explicit sub-steps
    *m_out = c->adi_m;
    return run_heat_adi(c, dt, c->adi_m);
  }
  const int m = heat_substeps_count(c, dt);
  const double sub = dt / m;
  c->prof.begin(c->stream);
  if (k_heat_all_substeps(c->v, c->mp, c->lp, m, c->H, c->Q, c->Halt, sub)) {   // small lattice: one in-SM launch
    std::swap(c->H, c->Halt);
    c->prof.end(c->stream, QS_PROF_HEAT, 1);
  } else {
    qs_ctx::HeatGraph* hg = nullptr;
    const int group = k_heat_block_max();   // sub-steps per temporally blocked launch
    // Temporal blocking pays where the lattice lives in L2 (every config: <= 6.9 MB per array) and the launches are
    // latency-bound: config 2, m = 28: 0.19 -> 0.074 ms per step.  On an HBM-resident lattice (4096 x 4096 cells) it
    // does cut the traffic to ~28 B per cell per 4 sub-steps but is slower than four marching launches (0.364 vs
    // 0.303 ms: 27 % halo recompute, one 1024-thread CTA per SM, FP64-bound), so those keep the marching kernel.
    const bool blocked = m > 1 && (c->heat_force_blocked || static_cast<long long>(c->N) <= kHeatBlockedMaxCells);
    if (blocked && !c->prof.on && m > 2 * group) {   // replay the m launches from a graph (captured on first use for this start buffer)
      for (auto& slot : c->heat_graph)
        if (slot.exec && slot.H == c->H && slot.m == m && slot.sub == sub) hg = &slot;
      if (!hg) {
        qs_ctx::HeatGraph& slot = c->heat_graph[c->heat_graph[0].exec && c->heat_graph[0].H != c->H ? 1 : 0];
        if (slot.exec) {
          cudaGraphExecDestroy(slot.exec);
          slot.exec = nullptr;
        }
        const long long l0 = c->launches;
        cudaGraph_t gr = nullptr;
        if (cudaStreamBeginCapture(c->stream, cudaStreamCaptureModeRelaxed) == cudaSuccess) {
          double *a = c->H, *b = c->Halt;
          for (int s = 0; s < m; s += group) {
            k_heat_block(c->v, c->mp, c->lp, std::min(group, m - s), a, c->Q, b, sub);
            std::swap(a, b);
          }
          const cudaError_t ec = cudaStreamEndCapture(c->stream, &gr);
          if (ec == cudaSuccess && gr && cudaGraphInstantiate(&slot.exec, gr, 0) == cudaSuccess) {
            slot.H = c->H, slot.m = m, slot.sub = sub;
            hg = &slot;
          } else {
            slot.exec = nullptr;
            cudaGetLastError();
          }
          if (gr) cudaGraphDestroy(gr);
        }
        c->launches = l0;   // capture enqueued nothing
      }
    }
    const int n_launch = (m + group - 1) / group;
    if (hg) {
      QS_CUDA(cudaGraphLaunch(hg->exec, c->stream));
      c->launches += n_launch;
      if (n_launch & 1) std::swap(c->H, c->Halt);
    } else if (!blocked) {   // one marching TMA kernel per sub-step (24 B per cell and sub-step, no halo re-reads)
      for (int s = 0; s < m; ++s) {
        k_heat_substep(c->v, c->mp, c->lp, c->H, c->Q, c->Halt, sub);
        std::swap(c->H, c->Halt);
      }
    } else {
      for (int s = 0; s < m; s += group) {
        k_heat_block(c->v, c->mp, c->lp, std::min(group, m - s), c->H, c->Q, c->Halt, sub);
        std::swap(c->H, c->Halt);
      }
    }
    c->prof.end(c->stream, QS_PROF_HEAT, blocked ? n_launch : m);
  }
  *m_out = m;
  QS_CUDA(cudaGetLastError());
  return QS_OK;
}

// per-wire statistics start: zeros, T_max = T_bath, t_q = -1
int reset_wire_stats(qs_ctx* c) {
  if (c->n_turns <= 0) return QS_OK;
  const size_t nt = c->n_turns;
  std::vector<double> w(9 * nt, 0.0);
  for (size_t k = 0; k < nt; ++k) w[3 * nt + k] = c->lp.T_bath, w[4 * nt + k] = -1.0;
  QS_CUDA(cudaMemcpyAsync(c->wire, w.data(), sizeof(double) * 9 * nt, cudaMemcpyHostToDevice, c->stream));
  QS_CUDA(cudaStreamSynchronize(c->stream));
  return QS_OK;
}

// presets of the per-turn event observables the material pass reduces into: max -> 0, min -> all ones
int reset_event_bits(qs_ctx* c) {
  if (!c->lattice || c->n_turns <= 0) return QS_OK;
  QS_CUDA(cudaMemsetAsync(c->xmax_bits, 0, sizeof(unsigned long long) * c->n_turns, c->stream));
  QS_CUDA(cudaMemsetAsync(c->rmin_bits, 0xff, sizeof(unsigned long long) * c->n_turns, c->stream));
  return QS_OK;
}

MaterialArgs material_args(qs_ctx* c, double Bext, double Bdot, double dt, bool from_acc, bool aux,
                           const double* Jsrc = nullptr) {
  MaterialArgs a;
  a.N = c->N;
  a.Nz = c->lattice ? c->lp.Nz : 0;
  a.J = Jsrc ? Jsrc : c->J;
  a.H = c->H;
  a.jc0_scale = c->jc0s;
  a.bracc = c->bracc;
  a.bzacc = c->bzacc;
  a.rowtab = c->rowtab;
  a.r = c->r;
  a.area = c->area;
  a.selfcoef = c->selfcoef;
  a.diagM = c->diagM;
  a.Br = c->Br;
  a.Bz = c->Bz;
  a.E = c->E;
  a.Q = c->Q;
  a.shift = c->shift;
  a.Hd = c->Hd;
  a.dEdJ = aux ? c->dEdJ : nullptr;
  a.Jc = aux ? c->Jc : nullptr;
  a.rho = aux ? c->rho : nullptr;
  const bool ev = c->lattice && c->n_turns > 0;
  a.rowturn = ev && c->canonical_turns ? c->rowturn : nullptr;
  a.turn_id = c->turn_id;
  a.cells_per_side = c->lp.n;
  a.xmax_bits = ev ? c->xmax_bits : nullptr;
  a.rmin_bits = ev ? c->rmin_bits : nullptr;
  a.Bext = Bext;
  a.Bdot = Bdot;
  a.dt = dt;
  a.inv_area = c->lattice ? 1.0 / (c->lp.h * c->lp.h) : 0.0;
  a.from_acc = from_acc;
  return a;
}

// Transactional step (include/qs.h: "negative = error (state unchanged)"): everything a step modifies that the caller
// can observe is copied aside first - J, H, I' and, as two contiguous blocks, the derived fields (Br, Bz, E) and the
// per-turn event state (wire statistics, mean-E history, first-event times, flag words, counters).
int backup_state(qs_ctx* c) {
  const size_t nb8 = sizeof(double) * c->N;
  c->backup_valid = false;
  QS_CUDA(cudaMemcpyAsync(c->Jold, c->J, nb8, cudaMemcpyDeviceToDevice, c->stream));
  QS_CUDA(cudaMemcpyAsync(c->Hold, c->H, nb8, cudaMemcpyDeviceToDevice, c->stream));
  QS_CUDA(cudaMemcpyAsync(c->xold, c->x, nb8, cudaMemcpyDeviceToDevice, c->stream));
  QS_CUDA(cudaMemcpyAsync(c->fld_backup, c->fld_begin, c->fld_bytes, cudaMemcpyDeviceToDevice, c->stream));
  if (c->n_turns) QS_CUDA(cudaMemcpyAsync(c->ev_backup, c->ev_begin, c->ev_bytes, cudaMemcpyDeviceToDevice, c->stream));
  c->have_prev_E_old = c->have_prev_E;
  c->backup_valid = true;
  return QS_OK;
}
// Called on every negative return after backup_state: puts the state back (best effort if the device itself failed).
// The stored previous solutions of the extrapolated CG start are dropped (a guess only).
void restore_state(qs_ctx* c) {
  const size_t nb8 = sizeof(double) * c->N;
  cudaGetLastError();
  c->n_prev = 0;
  if (!c->backup_valid) return;   // the backup itself never ran (launch failure): the state was not touched either
  c->backup_valid = false;
  cudaMemcpyAsync(c->J, c->Jold, nb8, cudaMemcpyDeviceToDevice, c->stream);
  cudaMemcpyAsync(c->H, c->Hold, nb8, cudaMemcpyDeviceToDevice, c->stream);
  cudaMemcpyAsync(c->x, c->xold, nb8, cudaMemcpyDeviceToDevice, c->stream);
  cudaMemcpyAsync(c->fld_begin, c->fld_backup, c->fld_bytes, cudaMemcpyDeviceToDevice, c->stream);
  if (c->n_turns) cudaMemcpyAsync(c->ev_begin, c->ev_backup, c->ev_bytes, cudaMemcpyDeviceToDevice, c->stream);
  cudaStreamSynchronize(c->stream);
  c->have_prev_E = c->have_prev_E_old;
  c->n_prev = 0;
}

// One electromagnetic stage (S1..S4) at the state Jsrc: field sweep fused with M x0, material law (diagonal shift
// theta dt_shift D), projected CG for I' (left in c->x, warm-started from its previous content), multipliers -> uterm.
int em_stage(qs_ctx* c, const double* Jsrc, double Bext, double Bdot, double dt_shift, double I_ramp, int* iters,
             double* relres, bool* hit_max) {
  const VecCtx& v = c->v;
  const size_t nb8 = sizeof(double) * c->N;
  int rc;
  *iters = 0;
  *relres = 0.0;
  *hit_max = false;
  // warm start I'_prev moved onto the constraint C^T x = I_ramp with the static diagonal of M
  k_turn_deficit(v, c->x, I_ramp, c->defw);
  k_apply_deficit(v, c->defw, c->diagM, c->swM, c->x);
  // S1 (+ M x0 in the same sweep): ring currents I = a J
  k_mul(v, c->area, Jsrc, c->cur);
  if ((rc = do_sweep(c, c->x, c->cur, true)) != QS_OK) return rc;
  // S2
  if ((rc = reset_event_bits(c)) != QS_OK) return rc;
  c->prof.begin(c->stream);
  k_material(v, c->mp, material_args(c, Bext, Bdot, dt_shift, true, false, Jsrc));
  c->prof.end(c->stream, QS_PROF_MATERIAL, 1);
  // S3/S4: the right-hand side b = -2 pi r (E + r Bdot / 2) is evaluated on the fly from E (C4)
  const Rhs rhs{nullptr, c->E, c->r, Bdot};
  double nu = -1.0;
  // the reference norm is accumulated into rg[0]: start from zero whatever an earlier stage of this step left there
  QS_CUDA(cudaMemsetAsync(c->sc->rg, 0, 2 * sizeof(double), c->stream));
  if (c->n_turns) {
    k_turn_schur(v, c->Hd, c->sw);
    k_nu_residual(v, I_ramp, c->Mxp1, c->shift, c->xp1, rhs, c->rr);
    k_turn_project(v, c->rr, c->Hd, c->sw, c->vw, nullptr);
    k_project_apply(v, 0, c->vw, c->Hd, c->rr, c->g);
    k_copy_rg_to_nu2(v, 0);
  } else {  // no constraint: nu^2 = b^T H^-1 b
    k_rhs_fill(v, rhs, c->rr);
    k_project_apply(v, 0, nullptr, c->Hd, c->rr, c->g);
    k_copy_rg_to_nu2(v, 0);
  }
  if ((rc = sync_scalars(c)) != QS_OK) return rc;
  nu = std::sqrt(std::max(c->h_sc->nu2, 0.0));
  if (nu > 0.0) {
    rc = cg_core(c, rhs, c->x, c->shift, c->Hd, c->sw, true, c->cg_tol, c->cg_maxit, nu, iters, relres, hit_max);
    if (rc != QS_OK) return rc;
  } else {
    // nu == 0: the cold start x_p = I_ramp xp1 already solves the projected system (e.g. one cell per turn, where the
    // constraint alone fixes I'; or b = 0 with no ramp, where x_p = 0); its projection multipliers are the V_w (C8)
    QS_CUDA(cudaMemsetAsync(c->x, 0, nb8, c->stream));
    if (c->n_turns) {
      k_axpy(v, I_ramp, c->xp1, c->x);
      QS_CUDA(cudaMemcpyAsync(c->vsum, c->vw, sizeof(double) * c->n_turns, cudaMemcpyDeviceToDevice, c->stream));
    }
  }
  k_sum_uterm(v, c->vsum);
  return QS_OK;
}

// The same stage for qs_step on geometries with constraint groups, in five launches and one host round trip before the
// CG iterates: step_begin (backups, CG start, I = a J, zeroing) -> turn_fix (start moved onto the constraint) -> fused
// sweep -> material -> turn_start (Schur scalars, reference norm, start residual, projection, first direction).
int em_stage_fused(qs_ctx* c, bool extrapolate, double Bext, double Bdot, double dt, double I_ramp, int* iters,
                   double* relres, bool* hit_max) {
  const VecCtx& v = c->v;
  int rc;
  *iters = 0;
  *relres = 0.0;
  *hit_max = false;
  StepBegin sb{};
  sb.N = c->N;
  sb.n_turns = c->n_turns;
  sb.extrapolate = extrapolate;
  sb.J = c->J; sb.H = c->H; sb.area = c->area;
  sb.Jold = c->Jold; sb.Hold = c->Hold; sb.x = c->x; sb.xold = c->xold; sb.xprev2 = c->xprev2; sb.cur = c->cur;
  sb.fld = reinterpret_cast<const unsigned long long*>(c->fld_begin);
  sb.fld_backup = reinterpret_cast<unsigned long long*>(c->fld_backup);
  sb.fld_words = c->fld_bytes / 8;
  sb.ev = reinterpret_cast<const unsigned long long*>(c->ev_begin);
  sb.ev_backup = reinterpret_cast<unsigned long long*>(c->ev_backup);
  sb.ev_words = c->ev_bytes / 8;
  sb.acc = reinterpret_cast<unsigned long long*>(c->counter);
  sb.acc_words = c->acc_bytes / 8;
  sb.vsum = c->vsum; sb.tw = c->tw;
  const bool ev = c->lattice && c->n_turns > 0;
  sb.xmax_bits = ev ? c->xmax_bits : nullptr;
  sb.rmin_bits = ev ? c->rmin_bits : nullptr;
  c->backup_valid = false;
  k_step_begin(v, sb);
  if (cudaPeekAtLastError() != cudaSuccess)
    return fail(QS_ERR_CUDA, std::string("step_begin launch failed: ") + cudaGetErrorString(cudaGetLastError()));
  c->backup_valid = true;
  c->have_prev_E_old = c->have_prev_E;
  k_turn_fix(v, I_ramp, c->diagM, c->swM, c->x);
  if ((rc = do_sweep(c, c->x, c->cur, true, /*prezeroed=*/true)) != QS_OK) return rc;
  c->prof.begin(c->stream);
  k_material(v, c->mp, material_args(c, Bext, Bdot, dt, true, false, c->J));
  c->prof.end(c->stream, QS_PROF_MATERIAL, 1);
  const Rhs rhs{nullptr, c->E, c->r, Bdot};
  TurnStart ts{};
  ts.ptr = c->turn_ptr; ts.idx = c->turn_idx;
  ts.I_ramp = I_ramp; ts.cM = kCM; ts.b = rhs;
  ts.Hd = c->Hd; ts.shift = c->shift; ts.x = c->x; ts.yacc = c->yacc; ts.xp1 = c->xp1; ts.Mxp1 = c->Mxp1;
  ts.r = c->rr; ts.g = c->g; ts.p = c->p; ts.sw = c->sw; ts.vnu = c->defw; ts.vsum = c->vsum;
  k_turn_start(v, ts);
  double nu = 0.0;
  rc = cg_core(c, rhs, c->x, c->shift, c->Hd, c->sw, true, c->cg_tol, c->cg_maxit, -1.0, iters, relres, hit_max, nullptr,
               /*prepared=*/true, &nu);
  if (rc != QS_OK) return rc;
  if (nu == 0.0) {
    // the cold start x_p = I_ramp xp1 already solves the projected system (see em_stage); its multipliers are the V_w
    QS_CUDA(cudaMemsetAsync(c->x, 0, sizeof(double) * c->N, c->stream));
    k_axpy(v, I_ramp, c->xp1, c->x);
    QS_CUDA(cudaMemcpyAsync(c->vsum, c->defw, sizeof(double) * c->n_turns, cudaMemcpyDeviceToDevice, c->stream));
  }
  return QS_OK;
}

// Common tail of qs_step / qs_step_rk once J^{k+1} has been written: S6 heat with the current Q, S7 events and step
// statistics, NaN/Inf check (state restored from the backups on failure), commit of t, I and the statistics.
// uterm_scale: factor applied to the accumulated multiplier sum (1, or 1/2 for the two stages of the RK pair);
// reset_scalars: the RK step has consumed the scalar block for its error estimate and needs it cleared first.
int finish_step(qs_ctx* c, double dt, double I_ramp, int iters, double relres, bool hit_max, double uterm_scale,
                bool reset_scalars) {
  const VecCtx& v = c->v;
  int rc, m = 0;
  double uterm = 0.0;
  if (reset_scalars) {
    uterm = uterm_scale * c->h_sc->uterm;        // read back by the caller's last sync_scalars
    k_set_scalars(v);
  }
  if (c->inject == 2) {   // test hook: a NaN in J after S5
    c->inject = 0;
    cudaMemsetAsync(c->J, 0xff, sizeof(double), c->stream);
  }
  rc = c->inject == 1 ? (c->inject = 0, fail(QS_ERR_CUDA, "injected failure in the heat stage (qs_debug_inject_failure)"))
                      : run_heat(c, dt, &m);
  if (rc != QS_OK) {
    restore_state(c);
    return rc;
  }
  EventArgs ev;
  ev.H = c->H; ev.E = c->E; ev.xmax_bits = c->xmax_bits; ev.rmin_bits = c->rmin_bits;
  ev.Q = c->Q; ev.r = c->r; ev.area = c->area; ev.wire = c->wire;
  ev.ebar_prev = c->ebar_prev; ev.flags = c->flags; ev.t_first = c->t_first; ev.count = c->count;
  ev.dt = dt; ev.t_new = c->t + dt; ev.have_prev = c->have_prev_E;
  c->prof.begin(c->stream);
  if (c->n_turns) {   // one pass: events, per-wire statistics and the step statistics
    ev.J = c->J;
    ev.Jold = c->Jold;
    k_events(v, c->mp, ev);
  } else {
    k_step_stats(v, c->mp, c->J, c->Jold, c->H, c->Q, c->r, c->area);
  }
  c->prof.end(c->stream, QS_PROF_EVENTS, 1);
  if ((rc = sync_scalars(c)) != QS_OK) {
    restore_state(c);
    return rc;
  }
  if (c->h_sc->nonfinite) {
    restore_state(c);
    return fail(QS_ERR_NONFINITE, "NaN/Inf in J or T after the step; state restored");
  }
  if (!reset_scalars) uterm = uterm_scale * c->h_sc->uterm;
  c->t += dt;
  c->I += dt * I_ramp;
  c->have_prev_E = true;
  const int ret = c->h_sc->event_or | (hit_max ? QS_EV_CG_MAXIT : 0);
  c->st.cg_iters = iters;
  c->st.cg_relres = relres;
  c->st.heat_substeps = m;
  c->st.event_word = ret;
  c->st.U_terminal = uterm;
  c->st.Tmax = c->h_sc->tmax;
  c->st.joule_power = c->h_sc->joule;
  c->st.dJ_max = c->h_sc->djmax;
  c->st.t = c->t;
  c->st.I = c->I;
  return ret;
}

// host arrays in caller order <-> device arrays in internal order
int upload(qs_ctx* c, const double* src, double* dst, int n_pad) {
  for (int k = 0; k < c->N; ++k) c->h_stage[k] = src[c->perm.empty() ? k : c->perm[k]];
  for (int k = c->N; k < n_pad; ++k) c->h_stage[k] = 0.0;
  QS_CUDA(cudaMemcpyAsync(dst, c->h_stage, sizeof(double) * n_pad, cudaMemcpyHostToDevice, c->stream));
  QS_CUDA(cudaStreamSynchronize(c->stream));
  return QS_OK;
}
int download(qs_ctx* c, const double* src, double* dst, double scale = 1.0) {
  QS_CUDA(cudaMemcpyAsync(c->h_stage, src, sizeof(double) * c->N, cudaMemcpyDeviceToHost, c->stream));
  QS_CUDA(cudaStreamSynchronize(c->stream));
  for (int k = 0; k < c->N; ++k) dst[c->perm.empty() ? k : c->perm[k]] = scale * c->h_stage[k];
  return QS_OK;
}

uint32_t morton16(uint32_t a, uint32_t b) {
  auto spread = [](uint32_t v) {
    v &= 0xffff;
    v = (v | (v << 8)) & 0x00ff00ff;
    v = (v | (v << 4)) & 0x0f0f0f0f;
    v = (v | (v << 2)) & 0x33333333;
    v = (v | (v << 1)) & 0x55555555;
    return v;
  };
  return spread(a) | (spread(b) << 1);
}

int init_common(const qs_geometry* geo, const qs_material* mat, void* workspace, size_t workspace_bytes, void* stream,
                bool own, qs_ctx** out) {
  int rc = check_geometry(geo);
  if (rc != QS_OK) return rc;
  if (!mat || !out) return fail(QS_ERR_ARG, "NULL material or out pointer");
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) return fail(QS_ERR_CUDA, "no CUDA device: libqs has no CPU path");
  qs_ctx* c = new (std::nothrow) qs_ctx();
  if (!c) return fail(QS_ERR_ARG, "out of host memory");
  auto bail = [&](int code) {
    qs_free(c);
    return code;
  };
  const int N = geo->n_rings;
  c->N = N;
  c->Np = (N + 31) / 32 * 32;
  c->nb = c->Np / 32;
  c->n_turns = geo->n_turns;
  c->lattice = geo->lattice != 0;
  c->has_operator = !(geo->flags & QS_GEO_NO_OPERATOR);
  c->tables = c->lattice && c->has_operator && (geo->flags & QS_GEO_LATTICE_TABLES);
  c->heat_force_blocked = (geo->flags & QS_GEO_HEAT_BLOCKED) != 0;
  c->blockprec = !c->lattice && c->has_operator && geo->n_turns == 0;
  patch_setup(&c->patch, geo, N);
  c->Bext0 = geo->Bext0;
  c->Bext_rate = geo->Bext_rate;
  c->Bext_max = geo->Bext_max;
  c->theta = mat->theta;
  c->cg_tol = mat->cg_tol > 0 ? mat->cg_tol : 1e-10;
  c->cg_maxit = mat->cg_maxit > 0 ? mat->cg_maxit : 20000;
  c->adi_m = mat->heat_adi_substeps > 0 ? mat->heat_adi_substeps : 0;
  MaterialParams& mp = c->mp;
  mp.Ec = mat->Ec; mp.n_exp = mat->n_exp; mp.Jc0 = mat->Jc0; mp.Tc = mat->Tc; mp.B0 = mat->B0;
  mp.eps_coef = mat->eps_coef; mp.eps_exp = mat->eps_exp; mp.Y = mat->Y; mp.rho_n = mat->rho_n;
  mp.C3 = mat->C3; mp.C1 = mat->C1; mp.k_in = mat->k_in; mp.k_between = mat->k_between; mp.theta = mat->theta;
  mp.T_fluxjump = mat->T_fluxjump; mp.dEdt_spike = mat->dEdt_spike;
  mp.n_int = (mat->n_exp == std::floor(mat->n_exp) && mat->n_exp >= 1 && mat->n_exp <= 200) ? static_cast<int>(mat->n_exp) : 0;
  if (!(mp.C3 > 0.0) || !(mp.rho_n > 0.0) || !(mp.Tc > 0.0)) return bail(fail(QS_ERR_ARG, "material: C3, rho_n, Tc must be > 0"));
  LatticeParams& lp = c->lp;
  lp = LatticeParams{};
  lp.T_bath = geo->T_bath;
  if (c->lattice) {
    lp.n = geo->cells_per_side;
    lp.Nr = geo->layers * lp.n;
    lp.Nz = geo->turns_per_layer * lp.n;
    lp.h = geo->wire_size / lp.n;
    lp.r_inner = geo->r_inner;
    for (int s = 0; s < 4; ++s) lp.h_conv[s] = geo->h_conv[s];
    c->tabNr = lp.Nr;
    c->tabNz = lp.Nz;
    // the lattice description must agree with the ring arrays (C1), ring by ring: the heat tables, the per-row
    // geometry, the block-Toeplitz tables and the separation bound minsep2 = h^2 behind the AGM evaluation classes
    // all come from the description, the pair sweep from the arrays
    for (int k = 0; k < N; ++k) {
      const int ir = k / lp.Nz, iz = k % lp.Nz;
      const double rr = lp.r_inner + (ir + 0.5) * lp.h, zz = (iz + 0.5) * lp.h - lp.Nz * lp.h / 2.0;
      if (std::fabs(geo->r[k] - rr) > 1e-9 * rr || std::fabs(geo->z[k] - zz) > 1e-9 * (std::fabs(zz) + lp.h))
        return bail(fail(QS_ERR_ARG, "geometry: r/z arrays do not match the lattice description (order c = ir*Nz + iz)"));
    }
  }
  const double g2 = geo->softening * geo->softening;
  c->soft_all = c->lattice ? 0.0 : g2;
  c->soft_self = c->lattice ? g2 : 0.0;
  c->minsep2 = c->lattice ? lp.h * lp.h * (1.0 - 1e-9) : 0.0;
  c->diag_d2 = std::min(c->soft_all + c->soft_self, c->minsep2 + c->soft_all);
  if (c->diag_d2 <= 0.0) c->diag_d2 = c->soft_all + c->soft_self;

  // validity domain of the squared-AGM recurrence: k'^2 <= 0.98 over the whole ring set
  double rmin = 1e300, rmax = 0, zmin = 1e300, zmax = -1e300;
  for (int k = 0; k < N; ++k) {
    if (!(geo->r[k] > 0.0) || !std::isfinite(geo->z[k]) || !(geo->area[k] > 0.0))
      return bail(fail(QS_ERR_ARG, "geometry: r, area must be > 0 and z finite"));
    rmin = std::min(rmin, geo->r[k]); rmax = std::max(rmax, geo->r[k]);
    zmin = std::min(zmin, geo->z[k]); zmax = std::max(zmax, geo->z[k]);
  }
  if (c->has_operator) {
    const double d2 = (rmax - rmin) * (rmax - rmin) + (zmax - zmin) * (zmax - zmin);
    if (d2 / (4.0 * rmin * rmin + d2) > 0.98)
      return bail(fail(QS_ERR_ARG, "geometry: ring set too spread out relative to its radius (k'^2 > 0.98)"));
  }
  if (geo->n_turns > 0)
    for (int k = 0; k < N; ++k)
      if (geo->turn_id[k] < 0 || geo->turn_id[k] >= geo->n_turns) return bail(fail(QS_ERR_ARG, "geometry: turn_id out of range"));

  // internal order: canonical for lattices (the heat stencil needs it); Morton order of (r, z) for free rings so
  // that blocks of 32 rings are compact and the per-item AGM depth bound is tight
  if (!c->lattice && c->has_operator) {
    std::vector<std::pair<uint32_t, int>> key(N);
    const double sr = rmax > rmin ? 65535.0 / (rmax - rmin) : 0.0, sz = zmax > zmin ? 65535.0 / (zmax - zmin) : 0.0;
    for (int k = 0; k < N; ++k)
      key[k] = {morton16(static_cast<uint32_t>((geo->r[k] - rmin) * sr), static_cast<uint32_t>((geo->z[k] - zmin) * sz)), k};
    std::sort(key.begin(), key.end());
    c->perm.resize(N);
    for (int k = 0; k < N; ++k) c->perm[k] = key[k].second;
  }
  const bool has_perm = !c->perm.empty();

  // device set-up
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) return bail(fail(QS_ERR_CUDA, "cudaGetDevice failed"));
  c->device = dev;
  cudaDeviceGetAttribute(&c->sm_count, cudaDevAttrMultiProcessorCount, dev);
  if (c->sm_count <= 0) c->sm_count = 148;
  pointwise_prepare_device();   // shared-memory opt-ins are per device
  size_t need = 0;
  carve(c, nullptr, &need);
  if (own) {
    if (cudaMalloc(&c->owned, need) != cudaSuccess) return bail(fail(QS_ERR_CUDA, "cudaMalloc of the workspace failed"));
    workspace = c->owned;
    if (cudaStreamCreateWithFlags(&c->stream, cudaStreamNonBlocking) != cudaSuccess) return bail(fail(QS_ERR_CUDA, "stream"));
  } else {
    if (!workspace || workspace_bytes < need || (reinterpret_cast<uintptr_t>(workspace) & 255))
      return bail(fail(QS_ERR_ARG, "workspace NULL, too small or not 256-byte aligned"));
    c->stream = static_cast<cudaStream_t>(stream);
  }
  carve(c, workspace, &need);
  if (cudaMallocHost(&c->h_sc, sizeof(Scalars)) != cudaSuccess ||
      cudaMallocHost(&c->h_stage, sizeof(double) * 2 * c->Np) != cudaSuccess)
    return bail(fail(QS_ERR_CUDA, "cudaMallocHost failed"));
  if (cudaMemsetAsync(workspace, 0, need, c->stream) != cudaSuccess) return bail(fail(QS_ERR_CUDA, "memset"));
  c->H = c->Ha;
  c->Halt = c->Hb;
  VecCtx& v = c->v;
  v.N = N; v.Np = c->Np; v.n_turns = c->n_turns;
  v.turn_id = c->turn_id; v.turn_ptr = c->turn_ptr; v.turn_idx = c->turn_idx; v.share = c->share;
  v.stream = c->stream; v.sc = c->sc; v.launches = &c->launches; v.sm_count = c->sm_count;

  // geometry arrays in internal order, padded with far-away dummy rings that carry no current
  std::vector<double> hr(c->Np), hz(c->Np), tmp(N);
  for (int k = 0; k < N; ++k) {
    const int o = c->perm.empty() ? k : c->perm[k];
    hr[k] = geo->r[o];
    hz[k] = geo->z[o];
  }
  for (int k = N; k < c->Np; ++k) {
    hr[k] = hr[0];
    hz[k] = zmax + 1.0 + 0.01 * (k - N);
  }
  auto put = [&](double* dst, const std::vector<double>& src, size_t n) {
    return cudaMemcpyAsync(dst, src.data(), sizeof(double) * n, cudaMemcpyHostToDevice, c->stream) == cudaSuccess &&
           cudaStreamSynchronize(c->stream) == cudaSuccess;
  };
  bool ok = put(c->r, hr, c->Np) && put(c->z, hz, c->Np);
  for (int k = 0; k < N; ++k) tmp[k] = geo->area[c->perm.empty() ? k : c->perm[k]];
  ok = ok && put(c->area, tmp, N);
  for (int k = 0; k < N; ++k) tmp[k] = mat->jc0_scale ? mat->jc0_scale[c->perm.empty() ? k : c->perm[k]] : 1.0;
  ok = ok && put(c->jc0s, tmp, N);
  for (int k = 0; k < N; ++k)   // C3 self field: mu0 [ln(8 r/g) - 1] / (4 pi r)
    tmp[k] = kMu0 * (std::log(8.0 * hr[k] / geo->softening) - 1.0) / (4.0 * kPi * hr[k]);
  ok = ok && put(c->selfcoef, tmp, N);
  if (!ok) return bail(fail(QS_ERR_CUDA, "upload of the geometry failed"));
  if (has_perm && (cudaMemcpyAsync(c->d_perm, c->perm.data(), sizeof(int) * N, cudaMemcpyHostToDevice, c->stream) != cudaSuccess ||
                   cudaStreamSynchronize(c->stream) != cudaSuccess))
    return bail(fail(QS_ERR_CUDA, "upload of the permutation failed"));
  // bounding boxes of the blocks of 32
  {
    std::vector<double4> bb(c->nb);
    for (int bidx = 0; bidx < c->nb; ++bidx) {
      double4 q = make_double4(1e300, -1e300, 1e300, -1e300);
      for (int l = 0; l < 32; ++l) {
        const int k = bidx * 32 + l;
        q.x = std::min(q.x, hr[k]); q.y = std::max(q.y, hr[k]);
        q.z = std::min(q.z, hz[k]); q.w = std::max(q.w, hz[k]);
      }
      bb[bidx] = q;
    }
    if (cudaMemcpyAsync(c->bbox, bb.data(), sizeof(double4) * c->nb, cudaMemcpyHostToDevice, c->stream) != cudaSuccess ||
        cudaStreamSynchronize(c->stream) != cudaSuccess)
      return bail(fail(QS_ERR_CUDA, "upload of the block boxes failed"));
  }
  // turns: ids in internal order + CSR
  if (c->n_turns) {
    std::vector<int> tid(N), ptr(c->n_turns + 1, 0), idx(N);
    for (int k = 0; k < N; ++k) tid[k] = geo->turn_id[c->perm.empty() ? k : c->perm[k]];
    for (int k = 0; k < N; ++k) ++ptr[tid[k] + 1];
    for (int w = 0; w < c->n_turns; ++w) {
      if (ptr[w + 1] == 0) return bail(fail(QS_ERR_ARG, "geometry: a turn has no cells"));
      ptr[w + 1] += ptr[w];
    }
    std::vector<int> fill(ptr.begin(), ptr.end() - 1);
    for (int k = 0; k < N; ++k) idx[fill[tid[k]]++] = k;
    std::vector<double> tf(c->n_turns, -1.0), sh(c->n_turns, 1.0);
    if (geo->turn_share) sh.assign(geo->turn_share, geo->turn_share + c->n_turns);
    if (cudaMemcpyAsync(c->share, sh.data(), sizeof(double) * c->n_turns, cudaMemcpyHostToDevice, c->stream) != cudaSuccess ||
        cudaMemcpyAsync(c->turn_id, tid.data(), sizeof(int) * N, cudaMemcpyHostToDevice, c->stream) != cudaSuccess ||
        cudaMemcpyAsync(c->turn_ptr, ptr.data(), sizeof(int) * (c->n_turns + 1), cudaMemcpyHostToDevice, c->stream) != cudaSuccess ||
        cudaMemcpyAsync(c->turn_idx, idx.data(), sizeof(int) * N, cudaMemcpyHostToDevice, c->stream) != cudaSuccess ||
        cudaMemcpyAsync(c->t_first, tf.data(), sizeof(double) * c->n_turns, cudaMemcpyHostToDevice, c->stream) != cudaSuccess ||
        cudaStreamSynchronize(c->stream) != cudaSuccess)
      return bail(fail(QS_ERR_CUDA, "upload of the turn tables failed"));
  }
  // heat-step coefficient tables (C9): conductivities, face areas and the cell volume folded per row / column
  if (c->lattice) {
    const int Nr = lp.Nr, Nz = lp.Nz, n = lp.n;
    const double h = lp.h;
    std::vector<double> tab(3 * static_cast<size_t>(Nr + Nz), 0.0);
    double *hr_p = tab.data(), *hr_m = hr_p + Nr, *rb_r = hr_m + Nr, *hz_p = rb_r + Nr, *hz_m = hz_p + Nz, *rb_z = hz_m + Nz;
    for (int ir = 0; ir < Nr; ++ir) {
      const double rc = lp.r_inner + (ir + 0.5) * h;
      if (ir + 1 < Nr) hr_p[ir] = ((ir / n == (ir + 1) / n) ? mp.k_in : mp.k_between) * (rc + 0.5 * h) / (2.0 * h * h * rc);
      if (ir > 0) hr_m[ir] = (((ir - 1) / n == ir / n) ? mp.k_in : mp.k_between) * (rc - 0.5 * h) / (2.0 * h * h * rc);
      if (ir == 0) rb_r[ir] += lp.h_conv[0] * (rc - 0.5 * h) / (rc * h);
      if (ir == Nr - 1) rb_r[ir] += lp.h_conv[1] * (rc + 0.5 * h) / (rc * h);
    }
    for (int iz = 0; iz < Nz; ++iz) {
      if (iz + 1 < Nz) hz_p[iz] = ((iz / n == (iz + 1) / n) ? mp.k_in : mp.k_between) / (2.0 * h * h);
      if (iz > 0) hz_m[iz] = (((iz - 1) / n == iz / n) ? mp.k_in : mp.k_between) / (2.0 * h * h);
      if (iz == 0) rb_z[iz] += lp.h_conv[2] / h;
      if (iz == Nz - 1) rb_z[iz] += lp.h_conv[3] / h;
    }
    if (!put(c->heat_tab, tab, tab.size())) return bail(fail(QS_ERR_CUDA, "upload of the heat tables failed"));
    std::vector<int> rt(Nr);
    for (int ir = 0; ir < Nr; ++ir) rt[ir] = (ir / n) * geo->turns_per_layer;
    c->canonical_turns = geo->n_turns == geo->layers * geo->turns_per_layer;
    for (int k = 0; k < N && c->canonical_turns; ++k)
      c->canonical_turns = geo->turn_id[k] == rt[k / Nz] + (k % Nz) / n;
    if (cudaMemcpyAsync(c->rowturn, rt.data(), sizeof(int) * Nr, cudaMemcpyHostToDevice, c->stream) != cudaSuccess ||
        cudaStreamSynchronize(c->stream) != cudaSuccess)
      return bail(fail(QS_ERR_CUDA, "upload of the row turn table failed"));
    lp.hr_p = c->heat_tab;
    lp.hr_m = lp.hr_p + Nr;
    lp.rb_r = lp.hr_m + Nr;
    lp.hz_p = lp.rb_r + Nr;
    lp.hz_m = lp.hz_p + Nz;
    lp.rb_z = lp.hz_m + Nz;
  }
  // initial state: J = 0 (memset), T = T_bath
  {
    std::vector<double> T0(N, geo->T_bath);
    if (!put(c->tmp, T0, N)) return bail(fail(QS_ERR_CUDA, "upload"));
    k_enthalpy_from_T(v, mp, c->tmp, c->H, N);
  }
  k_set_scalars(v);
  if (c->tables) {
    if (launch_table_build(lp.Nr, lp.Nz, lp.r_inner, lp.h, c->soft_self, c->TM, c->TBz, c->TBr, c->sm_count, c->stream) != cudaSuccess)
      return bail(fail(QS_ERR_CUDA, "table build kernel launch failed"));
    ++c->launches;
    c->pair_evals += static_cast<long long>(lp.Nr) * lp.Nr * lp.Nz;
  }
  if (c->has_operator) {
    if (launch_diag(N, c->r, c->soft_all + c->soft_self, c->diagM, c->stream) != cudaSuccess)
      return bail(fail(QS_ERR_CUDA, "diag kernel launch failed"));
    ++c->launches;
    if (cudaMemcpyAsync(c->Hd, c->diagM, sizeof(double) * N, cudaMemcpyDeviceToDevice, c->stream) != cudaSuccess)
      return bail(fail(QS_ERR_CUDA, "copy"));
    if (c->lattice) k_build_rowtab(v, lp.Nr, lp.Nz, c->r, c->selfcoef, c->diagM, c->area, c->rowtab);
    if (c->blockprec) {
      if (launch_blockprec_build(c->nb, c->r, c->z, c->soft_all, c->soft_self, c->Lblk, c->stream) != cudaSuccess)
        return bail(fail(QS_ERR_CUDA, "block preconditioner build failed"));
      ++c->launches;
    }
    if (c->patch.pp > 0) {   // patch preconditioner: slot -> cell map, patch -> wire map, constant part M_patch
      const int ps = static_cast<int>(std::lround(std::sqrt(static_cast<double>(c->patch.pp)))), pp = c->patch.pp;
      const int n = lp.n, per = n / ps;                 // patches per wire side
      std::vector<int> hidx(N), hturn(c->patch.n_patches);
      int pch = 0;
      for (int l = 0; l < geo->layers; ++l)
        for (int tq = 0; tq < geo->turns_per_layer; ++tq)
          for (int a = 0; a < per; ++a)
            for (int b = 0; b < per; ++b, ++pch) {
              hturn[pch] = l * geo->turns_per_layer + tq;
              for (int i = 0; i < ps; ++i)
                for (int j = 0; j < ps; ++j)
                  hidx[pch * pp + i * ps + j] = (l * n + a * ps + i) * lp.Nz + tq * n + b * ps + j;
            }
      if (cudaMemcpyAsync(c->pidx, hidx.data(), sizeof(int) * N, cudaMemcpyHostToDevice, c->stream) != cudaSuccess ||
          cudaMemcpyAsync(c->pturn, hturn.data(), sizeof(int) * hturn.size(), cudaMemcpyHostToDevice, c->stream) != cudaSuccess ||
          cudaStreamSynchronize(c->stream) != cudaSuccess)
        return bail(fail(QS_ERR_CUDA, "upload of the patch tables failed"));
      c->patch.pidx = c->pidx;
      c->patch.pturn = c->pturn;
      if (c->patch.nc > 0) {
        std::vector<int> hpid(N);
        for (int q = 0; q < c->patch.n_patches; ++q)
          for (int t = 0; t < pp; ++t) hpid[hidx[q * pp + t]] = q;
        if (cudaMemcpyAsync(c->pid, hpid.data(), sizeof(int) * N, cudaMemcpyHostToDevice, c->stream) != cudaSuccess ||
            cudaStreamSynchronize(c->stream) != cudaSuccess)
          return bail(fail(QS_ERR_CUDA, "upload of the patch tables failed"));
        c->patch.pid = c->pid;
      }
      k_patch_build(v, c->patch, c->r, c->z, c->soft_all, c->soft_self);
    }
    if (c->n_turns) {
      // unit-ramp particular solution x_p1 = H_M^-1 C (share/s_M) and M x_p1 (reference norm of the CG, C8, C16)
      k_turn_schur(v, c->diagM, c->swM);
      if (cudaMemcpyAsync(c->defw, c->share, sizeof(double) * c->n_turns, cudaMemcpyDeviceToDevice, c->stream) != cudaSuccess)
        return bail(fail(QS_ERR_CUDA, "copy"));
      k_apply_deficit(v, c->defw, c->diagM, c->swM, c->xp1);
      if (cudaMemcpyAsync(c->p, c->xp1, sizeof(double) * N, cudaMemcpyDeviceToDevice, c->stream) != cudaSuccess)
        return bail(fail(QS_ERR_CUDA, "copy"));
      if ((rc = do_sweep(c, c->p, nullptr, false)) != QS_OK) return bail(rc);
      k_scatter_scaled(v, c->yacc, nullptr, c->Mxp1, N, kCM);
    }
  }
  if (c->lattice && !c->has_operator) k_build_rowtab(v, lp.Nr, lp.Nz, c->r, c->selfcoef, c->diagM, c->area, c->rowtab);
  if (cudaStreamSynchronize(c->stream) != cudaSuccess || cudaGetLastError() != cudaSuccess)
    return bail(fail(QS_ERR_CUDA, std::string("initialisation kernels failed: ") + cudaGetErrorString(cudaGetLastError())));
  c->st = qs_stats_t{};
  c->st.Tmax = geo->T_bath;
  if ((rc = reset_wire_stats(c)) != QS_OK) return bail(rc);
  *out = c;
  return QS_OK;
}

}  // namespace

extern "C" {

const char* qs_last_error(void) { return g_err.c_str(); }

size_t qs_workspace_bytes(const qs_geometry* geo) {
  if (check_geometry(geo) != QS_OK) return 0;
  qs_ctx tmp;
  tmp.N = geo->n_rings;
  tmp.Np = (tmp.N + 31) / 32 * 32;
  tmp.nb = tmp.Np / 32;
  tmp.n_turns = geo->n_turns;
  if (geo->lattice) {
    tmp.tabNr = geo->layers * geo->cells_per_side;
    tmp.tabNz = geo->turns_per_layer * geo->cells_per_side;
    tmp.tables = (geo->flags & QS_GEO_LATTICE_TABLES) && !(geo->flags & QS_GEO_NO_OPERATOR);
  }
  tmp.blockprec = !geo->lattice && !(geo->flags & QS_GEO_NO_OPERATOR) && geo->n_turns == 0;
  patch_setup(&tmp.patch, geo, geo->n_rings);
  size_t need = 0;
  carve(&tmp, nullptr, &need);
  return need;
}

int qs_init(const qs_geometry* geo, const qs_material* mat, qs_ctx** out) {
  return init_common(geo, mat, nullptr, 0, nullptr, true, out);
}
int qs_init_device(const qs_geometry* geo, const qs_material* mat, void* workspace, size_t workspace_bytes, void* stream,
                   qs_ctx** out) {
  return init_common(geo, mat, workspace, workspace_bytes, stream, false, out);
}

void qs_free(qs_ctx* c) {
  if (!c) return;
  DeviceGuard guard(c->device);
  if (c->stream) cudaStreamSynchronize(c->stream);
  c->prof.destroy();
  for (auto& gslot : c->cg_graph)
    if (gslot.exec) cudaGraphExecDestroy(gslot.exec);
  for (auto& gslot : c->heat_graph)
    if (gslot.exec) cudaGraphExecDestroy(gslot.exec);
  if (c->h_sc) cudaFreeHost(c->h_sc);
  if (c->h_stage) cudaFreeHost(c->h_stage);
  if (c->owned) {
    cudaFree(c->owned);
    if (c->stream) cudaStreamDestroy(c->stream);
  }
  delete c;
}

int qs_sync(qs_ctx* c) {
  if (!c) return fail(QS_ERR_ARG, "NULL handle");
  DeviceGuard guard(c->device);
  QS_CUDA(cudaStreamSynchronize(c->stream));
  return QS_OK;
}

int qs_step(qs_ctx* c, double dt, double I_ramp) {
  if (!c) return fail(QS_ERR_ARG, "NULL handle");
  if (!c->lattice || !c->has_operator) return fail(QS_ERR_ARG, "qs_step needs a lattice geometry with the operator set up");
  DeviceGuard guard(c->device);
  if (!(dt > 0.0)) return fail(QS_ERR_DT, "dt <= 0");
  const VecCtx& v = c->v;
  const int N = c->N;
  int rc;
  c->st.sweeps = 0;
  const size_t nb8 = sizeof(double) * N;
  int iters = 0;
  double relres = 0.0;
  bool hit_max = false;
  auto restore = [&]() { restore_state(c); };
  const int n_prev_in = c->n_prev;
  const double B0 = bext_at(c, c->t), B1 = bext_at(c, c->t + dt);
  // CG start: linear extrapolation 2 I'_k - I'_{k-1} of the two previous solutions when the step is repeated with
  // the same dt and ramp (a guess only: the solution does not depend on it beyond cg_tol; config 1: 12 % fewer
  // iterations than the plain warm start, nothing changes where I' is constant)
  const bool extrapolate = c->n_prev >= 2 && dt == c->last_dt && I_ramp == c->last_ramp;
  if (c->n_turns > 0) {
    // fused path: backups, CG start and all zeroing in one launch (the step is transactional)
    rc = em_stage_fused(c, extrapolate, B0, (B1 - B0) / dt, dt, I_ramp, &iters, &relres, &hit_max);
    if (rc != QS_OK) {
      restore();
      return rc;
    }
    k_step_update(v, dt, c->x, c->area, c->J, c->vsum);   // S5 + terminal voltage
  } else {
    // backups: the step is transactional
    if ((rc = backup_state(c)) != QS_OK) return rc;
    k_set_scalars(v);
    if (extrapolate) {
      k_lincomb(v, 2.0, c->x, -1.0, c->xprev2);                                   // xprev2 <- extrapolated start
      QS_CUDA(cudaMemcpyAsync(c->tmp2, c->x, nb8, cudaMemcpyDeviceToDevice, c->stream));
      QS_CUDA(cudaMemcpyAsync(c->x, c->xprev2, nb8, cudaMemcpyDeviceToDevice, c->stream));
      QS_CUDA(cudaMemcpyAsync(c->xprev2, c->tmp2, nb8, cudaMemcpyDeviceToDevice, c->stream));   // xprev2 <- I'_k
    } else {
      QS_CUDA(cudaMemcpyAsync(c->xprev2, c->x, nb8, cudaMemcpyDeviceToDevice, c->stream));
    }
    if ((rc = em_stage(c, c->J, B0, (B1 - B0) / dt, dt, I_ramp, &iters, &relres, &hit_max)) != QS_OK) {
      restore();
      return rc;
    }
    // S5
    k_scale_div(v, dt, c->x, c->area, c->J);
  }
  // S6, S7, statistics, commit (restores the state itself on failure)
  rc = finish_step(c, dt, I_ramp, iters, relres, hit_max, 1.0, false);
  if (rc >= 0) {   // the history of the extrapolated start advances only with a committed step
    c->n_prev = (dt == c->last_dt && I_ramp == c->last_ramp) ? std::min(n_prev_in + 1, 2) : 1;
    c->last_dt = dt;
    c->last_ramp = I_ramp;
  }
  return rc;
}

// Embedded Heun-Euler step with error control (readings: DESIGN.md §3 C14).
int qs_step_rk(qs_ctx* c, double dt_try, double I_ramp, double rtol, double dt_min, double* dt_taken, double* dt_next,
               double* err_out) {
  if (!c) return fail(QS_ERR_ARG, "NULL handle");
  DeviceGuard guard(c->device);
  if (!c->lattice || !c->has_operator) return fail(QS_ERR_ARG, "qs_step_rk needs a lattice geometry with the operator set up");
  if (!(dt_try > 0.0) || !(dt_min > 0.0) || !(rtol > 0.0)) return fail(QS_ERR_DT, "dt_try, dt_min and rtol must be > 0");
  const VecCtx& v = c->v;
  const int N = c->N;
  const size_t nb8 = sizeof(double) * N;
  int rc;
  c->st.sweeps = 0;
  if ((rc = backup_state(c)) != QS_OK) return rc;
  auto restore = [&]() { restore_state(c); };
  const double Jref = c->mp.Jc0 * (1.0 - c->lp.T_bath / c->mp.Tc) * (1.0 - c->lp.T_bath / c->mp.Tc);
  double dt = dt_try, err = 0.0, fac = 2.0;
  int iters = 0, it1 = 0, it2 = 0;
  double rel1 = 0.0, rel2 = 0.0;
  bool hm1 = false, hm2 = false;
  double* I1 = c->tmp2;     // I' of stage 1
  double* Jstar = c->tmp;   // predictor J^k + dt I'_1 / a
  double* Q1 = c->b;        // Joule source of stage 1 (the explicit-rhs array is used by qs_solve only)
  for (;;) {
    k_set_scalars(v);
    const double B0 = bext_at(c, c->t), B1 = bext_at(c, c->t + dt), Bdot = (B1 - B0) / dt;
    // stage 1 at (J^k, t^k): explicit stage, no theta term (dt_shift = 0)
    if ((rc = em_stage(c, c->J, B0, Bdot, 0.0, I_ramp, &it1, &rel1, &hm1)) != QS_OK) {
      restore();
      return rc;
    }
    QS_CUDA(cudaMemcpyAsync(I1, c->x, nb8, cudaMemcpyDeviceToDevice, c->stream));
    QS_CUDA(cudaMemcpyAsync(Q1, c->Q, nb8, cudaMemcpyDeviceToDevice, c->stream));
    QS_CUDA(cudaMemcpyAsync(Jstar, c->J, nb8, cudaMemcpyDeviceToDevice, c->stream));
    k_scale_div(v, dt, I1, c->area, Jstar);
    // stage 2 at (J*, t^k + dt), warm-started from I'_1
    if ((rc = em_stage(c, Jstar, B1, Bdot, 0.0, I_ramp, &it2, &rel2, &hm2)) != QS_OK) {
      restore();
      return rc;
    }
    k_max_scaled_diff(v, 0.5 * dt, c->x, I1, c->area);
    if ((rc = sync_scalars(c)) != QS_OK) {
      restore();
      return rc;
    }
    err = c->h_sc->djmax / Jref;
    iters += it1 + it2;
    fac = err == 0.0 ? 2.0 : std::min(2.0, std::max(0.2, 0.9 * std::sqrt(rtol / err)));
    if (err <= rtol || dt <= dt_min) break;
    dt = std::max(dt_min, dt * fac);
    QS_CUDA(cudaMemcpyAsync(c->x, c->xold, nb8, cudaMemcpyDeviceToDevice, c->stream));   // retry from the same warm start
  }
  // accepted: J^{k+1} = J^k + dt (I'_1 + I'_2) / (2a); heat source = trapezoid of the stage powers
  k_scale_div(v, 0.5 * dt, I1, c->area, c->J);
  k_scale_div(v, 0.5 * dt, c->x, c->area, c->J);
  k_lincomb(v, 0.5, Q1, 0.5, c->Q);
  const int ret = finish_step(c, dt, I_ramp, iters, std::max(rel1, rel2), hm1 || hm2, 0.5, true);
  if (ret < 0) return ret;
  c->n_prev = 0;   // the stored solutions of qs_step's extrapolated start are stale after an RK step
  if (dt_taken) *dt_taken = dt;
  if (dt_next) *dt_next = dt * fac;
  if (err_out) *err_out = err;
  return ret;
}

int qs_read(qs_ctx* c, double* J, double* T, double* B, double* E) {
  if (!c) return fail(QS_ERR_ARG, "NULL handle");
  DeviceGuard guard(c->device);
  int rc;
  if (J && (rc = download(c, c->J, J)) != QS_OK) return rc;
  if (T) {
    k_T_from_enthalpy(c->v, c->mp, c->H, c->tmp, c->N);
    if ((rc = download(c, c->tmp, T)) != QS_OK) return rc;
  }
  if (B) {
    if ((rc = download(c, c->Br, B)) != QS_OK) return rc;
    if ((rc = download(c, c->Bz, B + c->N)) != QS_OK) return rc;
  }
  if (E && (rc = download(c, c->E, E)) != QS_OK) return rc;
  return QS_OK;
}

int qs_read_aux(qs_ctx* c, double* Q, double* dEdJ, double* Jc, double* rho) {
  if (!c) return fail(QS_ERR_ARG, "NULL handle");
  DeviceGuard guard(c->device);
  int rc;
  if (Q && (rc = download(c, c->Q, Q)) != QS_OK) return rc;
  if (dEdJ && (rc = download(c, c->dEdJ, dEdJ)) != QS_OK) return rc;
  if (Jc && (rc = download(c, c->Jc, Jc)) != QS_OK) return rc;
  if (rho && (rc = download(c, c->rho, rho)) != QS_OK) return rc;
  return QS_OK;
}

int qs_write(qs_ctx* c, const double* J, const double* T, double t, double I) {
  if (!c) return fail(QS_ERR_ARG, "NULL handle");
  DeviceGuard guard(c->device);
  int rc;
  if (J && (rc = upload(c, J, c->J, c->N)) != QS_OK) return rc;
  if (T) {
    for (int k = 0; k < c->N; ++k)
      if (!(T[k] > 0.0)) return fail(QS_ERR_ARG, "qs_write: T must be > 0");
    if ((rc = upload(c, T, c->tmp, c->N)) != QS_OK) return rc;
    k_enthalpy_from_T(c->v, c->mp, c->tmp, c->H, c->N);
  }
  // the previous I' stays as the CG's initial guess (a guess only: the solution does not depend on it)
  QS_CUDA(cudaStreamSynchronize(c->stream));
  c->t = t;
  c->I = I;
  c->have_prev_E = false;
  c->n_prev = 0;
  return reset_wire_stats(c);
}

int qs_read_rate(qs_ctx* c, double* Idot) {
  if (!c || !Idot) return fail(QS_ERR_ARG, "NULL argument");
  DeviceGuard guard(c->device);
  return download(c, c->x, Idot);
}

int qs_write_rate(qs_ctx* c, const double* Idot) {
  if (!c || !Idot) return fail(QS_ERR_ARG, "NULL argument");
  DeviceGuard guard(c->device);
  const int rc = upload(c, Idot, c->x, c->Np);
  c->n_prev = 0;
  return rc;
}

int qs_debug_inject_failure(qs_ctx* c, int32_t where) {
  if (!c || where < 0 || where > 2) return fail(QS_ERR_ARG, "qs_debug_inject_failure: handle and where in 0..2");
  c->inject = where;
  return QS_OK;
}

int qs_matvec_device(qs_ctx* c, const double* d_x, double* d_y) {
  if (!c || !d_x || !d_y) return fail(QS_ERR_ARG, "NULL argument");
  if (!c->has_operator) return fail(QS_ERR_ARG, "operator not set up (QS_GEO_NO_OPERATOR)");
  DeviceGuard guard(c->device);
  c->st.sweeps = 0;
  k_gather(c->v, d_x, c->perm.empty() ? nullptr : c->d_perm, c->p, c->N, c->Np);
  int rc = do_sweep(c, c->p, nullptr, false);
  if (rc != QS_OK) return rc;
  k_scatter_scaled(c->v, c->yacc, c->perm.empty() ? nullptr : c->d_perm, d_y, c->N, kCM);
  QS_CUDA(cudaGetLastError());
  return QS_OK;
}

int qs_matvec(qs_ctx* c, const double* x, double* y) {
  if (!c || !x || !y) return fail(QS_ERR_ARG, "NULL argument");
  if (!c->has_operator) return fail(QS_ERR_ARG, "operator not set up (QS_GEO_NO_OPERATOR)");
  DeviceGuard guard(c->device);
  int rc;
  c->st.sweeps = 0;
  if ((rc = upload(c, x, c->p, c->Np)) != QS_OK) return rc;
  if ((rc = do_sweep(c, c->p, nullptr, false)) != QS_OK) return rc;
  return download(c, c->yacc, y, kCM);
}

int qs_field(qs_ctx* c, const double* I, double* B) {
  if (!c || !I || !B) return fail(QS_ERR_ARG, "NULL argument");
  if (!c->lattice || !c->has_operator) return fail(QS_ERR_ARG, "qs_field needs a lattice geometry with the operator set up");
  DeviceGuard guard(c->device);
  int rc;
  c->st.sweeps = 0;
  if ((rc = upload(c, I, c->cur, c->Np)) != QS_OK) return rc;
  QS_CUDA(cudaMemsetAsync(c->p, 0, sizeof(double) * c->Np, c->stream));
  if ((rc = do_sweep(c, c->p, c->cur, true)) != QS_OK) return rc;
  // output scaling of the accumulators (the one the material kernel applies inside a step), on the device:
  // Br = mu0/(4 r) bracc ; Bz = mu0/4 bzacc + selfcoef I
  k_field_scale(c->v, c->bracc, c->bzacc, c->r, c->selfcoef, c->cur, c->tmp, c->tmp2);
  if ((rc = download(c, c->tmp, B)) != QS_OK) return rc;
  return download(c, c->tmp2, B + c->N);
}

int qs_solve_device(qs_ctx* c, const double* d_b, double* d_x, int32_t maxit_override, int32_t* iters, double* relres) {
  if (!c || !d_b || !d_x) return fail(QS_ERR_ARG, "NULL argument");
  if (!c->has_operator) return fail(QS_ERR_ARG, "operator not set up (QS_GEO_NO_OPERATOR)");
  DeviceGuard guard(c->device);
  const int* perm = c->perm.empty() ? nullptr : c->d_perm;
  c->st.sweeps = 0;
  k_set_scalars(c->v);
  k_gather(c->v, d_b, perm, c->b, c->N, c->N);
  QS_CUDA(cudaMemsetAsync(c->tmp, 0, sizeof(double) * c->Np, c->stream));   // x0 = 0 satisfies C^T x = 0
  QS_CUDA(cudaMemsetAsync(c->yacc, 0, sizeof(double) * c->Np, c->stream));  // M x0 = 0
  int it = 0;
  double rel = 0.0;
  bool hit = false;
  const Rhs rhs{c->b, nullptr, nullptr, 0.0};
  int rc = cg_core(c, rhs, c->tmp, c->zero, c->diagM, c->swM, true, c->cg_tol, maxit_override > 0 ? maxit_override : c->cg_maxit,
                   -1.0, &it, &rel, &hit, c->blockprec ? c->Lblk : nullptr);
  if (rc != QS_OK) return rc;
  k_scatter_scaled(c->v, c->tmp, perm, d_x, c->N, 1.0);
  QS_CUDA(cudaStreamSynchronize(c->stream));
  if (iters) *iters = it;
  if (relres) *relres = rel;
  c->st.cg_iters = it;
  c->st.cg_relres = rel;
  return hit ? QS_EV_CG_MAXIT : QS_OK;
}

int qs_solve(qs_ctx* c, const double* b, double* x, int32_t maxit_override, int32_t* iters, double* relres) {
  if (!c || !b || !x) return fail(QS_ERR_ARG, "NULL argument");
  if (!c->has_operator) return fail(QS_ERR_ARG, "operator not set up (QS_GEO_NO_OPERATOR)");
  DeviceGuard guard(c->device);
  // stage through tmp2 (caller order on the device), then the device variant
  QS_CUDA(cudaMemcpyAsync(c->tmp2, b, sizeof(double) * c->N, cudaMemcpyHostToDevice, c->stream));
  QS_CUDA(cudaStreamSynchronize(c->stream));
  int rc = qs_solve_device(c, c->tmp2, c->tmp2, maxit_override, iters, relres);
  if (rc < 0) return rc;
  QS_CUDA(cudaMemcpyAsync(x, c->tmp2, sizeof(double) * c->N, cudaMemcpyDeviceToHost, c->stream));
  QS_CUDA(cudaStreamSynchronize(c->stream));
  return rc;
}

int qs_set_fields(qs_ctx* c, const double* B, const double* Q) {
  if (!c) return fail(QS_ERR_ARG, "NULL handle");
  DeviceGuard guard(c->device);
  int rc;
  if (B) {
    if ((rc = upload(c, B, c->Br, c->N)) != QS_OK) return rc;
    if ((rc = upload(c, B + c->N, c->Bz, c->N)) != QS_OK) return rc;
  }
  if (Q && (rc = upload(c, Q, c->Q, c->N)) != QS_OK) return rc;
  return QS_OK;
}

int qs_material_eval(qs_ctx* c, double dt) {
  if (!c) return fail(QS_ERR_ARG, "NULL handle");
  DeviceGuard guard(c->device);
  const double B0 = bext_at(c, c->t), B1 = bext_at(c, c->t + dt);
  int rc = reset_event_bits(c);
  if (rc != QS_OK) return rc;
  c->prof.begin(c->stream);
  k_material(c->v, c->mp, material_args(c, B0, dt > 0 ? (B1 - B0) / dt : 0.0, dt, false, c->aux_on));
  c->prof.end(c->stream, QS_PROF_MATERIAL, 1);
  QS_CUDA(cudaGetLastError());
  return QS_OK;
}

int qs_set_aux(qs_ctx* c, int32_t on) {
  if (!c) return fail(QS_ERR_ARG, "NULL handle");
  c->aux_on = on != 0;
  return QS_OK;
}

int qs_heat(qs_ctx* c, double dt) {
  if (!c) return fail(QS_ERR_ARG, "NULL handle");
  if (!c->lattice) return fail(QS_ERR_ARG, "qs_heat needs a lattice geometry");
  DeviceGuard guard(c->device);
  if (!(dt > 0.0)) return fail(QS_ERR_DT, "dt <= 0");
  int m = 0;
  int rc = run_heat(c, dt, &m);
  return rc != QS_OK ? rc : m;
}

int qs_heat_adi(qs_ctx* c, double dt, int32_t m) {
  if (!c) return fail(QS_ERR_ARG, "NULL handle");
  if (!c->lattice) return fail(QS_ERR_ARG, "qs_heat_adi needs a lattice geometry");
  DeviceGuard guard(c->device);
  if (!(dt > 0.0) || m <= 0) return fail(QS_ERR_DT, "dt <= 0 or m <= 0");
  const int rc = run_heat_adi(c, dt, m);
  return rc != QS_OK ? rc : m;
}

int qs_stats(qs_ctx* c, qs_stats_t* out) {
  if (!c || !out) return fail(QS_ERR_ARG, "NULL argument");
  *out = c->st;
  out->launches = c->launches;
  out->pair_evals = c->pair_evals;
  out->t = c->t;
  out->I = c->I;
  return QS_OK;
}

int qs_profile_enable(qs_ctx* c, int32_t on) {
  if (!c) return fail(QS_ERR_ARG, "NULL handle");
  DeviceGuard guard(c->device);
  c->prof.fold(c->stream);
  c->prof.reset();
  c->prof.on = on != 0;
  return QS_OK;
}

int qs_profile_read(qs_ctx* c, qs_profile_t* out) {
  if (!c || !out) return fail(QS_ERR_ARG, "NULL argument");
  DeviceGuard guard(c->device);
  QS_CUDA(cudaStreamSynchronize(c->stream));
  c->prof.fold(c->stream);
  for (int k = 0; k < QS_PROF_CLASSES; ++k) {
    out->ms[k] = c->prof.ms[k];
    out->launches[k] = c->prof.launches[k];
  }
  c->prof.reset();
  return QS_OK;
}

int qs_issue_probe(int32_t mode, double* cycles_per_dfma) {
  if (!cycles_per_dfma || mode < 1 || mode > 3) return fail(QS_ERR_ARG, "qs_issue_probe: mode 1..3 and a result pointer");
  const cudaError_t e = issue_probe(mode, cycles_per_dfma);
  if (e != cudaSuccess) return fail(QS_ERR_CUDA, std::string("issue probe: ") + cudaGetErrorString(e));
  return QS_OK;
}

int qs_pair_eval(int32_t n, const double* A2, const double* B2, int32_t cls, double* M, double* K, double* E, int32_t* used) {
  if (n <= 0 || !A2 || !B2 || !M || !K || !E || !used) return fail(QS_ERR_ARG, "qs_pair_eval: bad argument");
  if (cls >= pair_num_classes()) return fail(QS_ERR_ARG, "qs_pair_eval: class out of range");
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) return fail(QS_ERR_CUDA, "no CUDA device: libqs has no CPU path");
  double* d = nullptr;
  const size_t nb8 = sizeof(double) * n;
  QS_CUDA(cudaMalloc(&d, 5 * nb8 + sizeof(int) * n));
  int* du = reinterpret_cast<int*>(d + 5 * static_cast<size_t>(n));
  cudaError_t e = cudaMemcpy(d, A2, nb8, cudaMemcpyHostToDevice);
  if (e == cudaSuccess) e = cudaMemcpy(d + n, B2, nb8, cudaMemcpyHostToDevice);
  if (e == cudaSuccess) e = launch_pair_eval(n, d, d + n, cls, d + 2 * n, d + 3 * n, d + 4 * n, du, nullptr);
  if (e == cudaSuccess) e = cudaMemcpy(M, d + 2 * n, nb8, cudaMemcpyDeviceToHost);
  if (e == cudaSuccess) e = cudaMemcpy(K, d + 3 * n, nb8, cudaMemcpyDeviceToHost);
  if (e == cudaSuccess) e = cudaMemcpy(E, d + 4 * n, nb8, cudaMemcpyDeviceToHost);
  if (e == cudaSuccess) e = cudaMemcpy(used, du, sizeof(int) * n, cudaMemcpyDeviceToHost);
  cudaFree(d);
  if (e != cudaSuccess) return fail(QS_ERR_CUDA, std::string("qs_pair_eval: ") + cudaGetErrorString(e));
  return QS_OK;
}

int qs_fp64_peak(double* tflops, double* sm_clock_mhz_effective) {
  if (!tflops) return fail(QS_ERR_ARG, "NULL argument");
  double tf = 0.0, mhz = 0.0;
  const cudaError_t e = fp64_peak_probe(&tf, &mhz);
  if (e != cudaSuccess) return fail(QS_ERR_CUDA, std::string("fp64 probe: ") + cudaGetErrorString(e));
  *tflops = tf;
  if (sm_clock_mhz_effective) *sm_clock_mhz_effective = mhz;
  return QS_OK;
}

int qs_wire_stats(qs_ctx* c, double* out) {
  if (!c || !out) return fail(QS_ERR_ARG, "NULL argument");
  if (!c->n_turns) return QS_OK;
  DeviceGuard guard(c->device);
  QS_CUDA(cudaMemcpyAsync(out, c->wire, sizeof(double) * 8 * c->n_turns, cudaMemcpyDeviceToHost, c->stream));
  QS_CUDA(cudaStreamSynchronize(c->stream));
  return QS_OK;
}

int qs_events(qs_ctx* c, int32_t* flags, double* t_first, int32_t* count) {
  if (!c) return fail(QS_ERR_ARG, "NULL handle");
  if (!c->n_turns) return QS_OK;
  DeviceGuard guard(c->device);
  const size_t nt = c->n_turns;
  if (flags) QS_CUDA(cudaMemcpyAsync(flags, c->flags, sizeof(int) * nt, cudaMemcpyDeviceToHost, c->stream));
  if (t_first) QS_CUDA(cudaMemcpyAsync(t_first, c->t_first, sizeof(double) * nt, cudaMemcpyDeviceToHost, c->stream));
  if (count) QS_CUDA(cudaMemcpyAsync(count, c->count, sizeof(int) * nt, cudaMemcpyDeviceToHost, c->stream));
  QS_CUDA(cudaStreamSynchronize(c->stream));
  return QS_OK;
}

}  // extern "C"
