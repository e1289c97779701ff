// qs_vector.cu — K3 (CG vector kernels: fused axpy / dot) and K4 (per-turn segmented reductions, Schur scalars).
//
// Projected CG with a per-turn constraint, SURVEY.md §8(c) C8.  All scalars (r^T g, p^T A p, alpha, beta) stay
// on the device in a Scalars block: a kernel reads the dot products its predecessor reduced, so an iteration
// needs no host round trip.  Reductions: warp shuffles -> one shared-memory stage -> one FP64 atomic per CTA.
// Streaming kernels use grid-stride loops over a grid that is a multiple of the SM count.
#include "qs_internal.h"
#include "qs_pair.cuh"

namespace qs {

namespace {
constexpr int kBlock = 256;
thread_local int g_sm_count = 0;   // SM count of the handle whose kernel is being launched (set by QS_LAUNCH)

inline int grid_for(int n) {
  if (g_sm_count == 0) {
    int dev = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&g_sm_count, cudaDevAttrMultiProcessorCount, dev);
    if (g_sm_count <= 0) g_sm_count = 148;
  }
  const int need = (n + kBlock - 1) / kBlock;
  const int cap = g_sm_count * 8;
  return need < cap ? (need > 0 ? need : 1) : cap;
}

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}
__device__ __forceinline__ double warp_max(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_xor_sync(0xffffffffu, v, o));
  return v;
}
__device__ __forceinline__ void block_atomic_sum(double v, double* dst) {
  __shared__ double part[kBlock / 32];
  v = warp_sum(v);
  if ((threadIdx.x & 31) == 0) part[threadIdx.x >> 5] = v;
  __syncthreads();
  if (threadIdx.x < 32) {
    double s = threadIdx.x < kBlock / 32 ? part[threadIdx.x] : 0.0;
    s = warp_sum(s);
    if (threadIdx.x == 0) atomicAdd(dst, s);
  }
}

__global__ void finish_Ap_kernel(int n, const double* __restrict__ yacc, const double* __restrict__ shift,
                                 const double* __restrict__ p, double* __restrict__ q, double cM, Scalars* sc) {
  double acc = 0.0;
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
    const double pi = p[i];
    const double qi = fma(shift[i], pi, cM * yacc[i]);
    q[i] = qi;
    acc = fma(pi, qi, acc);
  }
  block_atomic_sum(acc, &sc->pq[0]);
}

__device__ __forceinline__ double rhs_at(const Rhs& b, int i) {
  if (b.b) return b.b[i];
  const double r = b.radius[i];
  return -2.0 * kPi * r * (b.E[i] + 0.5 * r * b.Bdot);
}

__global__ void residual_kernel(int n, const double* __restrict__ yacc, const double* __restrict__ shift,
                                const double* __restrict__ x, Rhs b, double* __restrict__ r, double cM) {
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x)
    r[i] = fma(shift[i], x[i], cM * yacc[i]) - rhs_at(b, i);
}
__global__ void rhs_fill_kernel(int n, Rhs b, double* __restrict__ r) {
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) r[i] = rhs_at(b, i);
}

__global__ void update_xr_kernel(int n, int par, const double* __restrict__ p, const double* __restrict__ q,
                                 double* __restrict__ x, double* __restrict__ r, const Scalars* sc) {
  const double alpha = sc->rg[par] / sc->pq[0];
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
    x[i] = fma(alpha, p[i], x[i]);
    r[i] = fma(alpha, q[i], r[i]);
  }
}

// one warp per turn: CSR gather of the turn's cells
__global__ void turn_project_kernel(int n_turns, const int* __restrict__ ptr, const int* __restrict__ idx,
                                    const double* __restrict__ r, const double* __restrict__ Hd,
                                    const double* __restrict__ sw, double* __restrict__ vw, double* __restrict__ vsum) {
  const int w = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
  if (w >= n_turns) return;
  double acc = 0.0;
  for (int k = ptr[w] + lane; k < ptr[w + 1]; k += 32) {
    const int i = idx[k];
    acc += r[i] / Hd[i];
  }
  acc = warp_sum(acc);
  if (lane == 0) {
    const double v = acc / sw[w];
    vw[w] = v;
    if (vsum) vsum[w] += v;
  }
}

__global__ void turn_schur_kernel(int n_turns, const int* __restrict__ ptr, const int* __restrict__ idx,
                                  const double* __restrict__ Hd, double* __restrict__ sw) {
  const int w = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
  if (w >= n_turns) return;
  double acc = 0.0;
  for (int k = ptr[w] + lane; k < ptr[w + 1]; k += 32) acc += 1.0 / Hd[idx[k]];
  acc = warp_sum(acc);
  if (lane == 0) sw[w] = acc;
}

__global__ void turn_deficit_kernel(int n_turns, const int* __restrict__ ptr, const int* __restrict__ idx,
                                    const double* __restrict__ share, const double* __restrict__ x, double d,
                                    double* __restrict__ defw, Scalars* sc) {
  const int w = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
  if (w >= n_turns) return;
  double acc = 0.0;
  for (int k = ptr[w] + lane; k < ptr[w + 1]; k += 32) acc += x[idx[k]];
  acc = warp_sum(acc);
  if (lane == 0) defw[w] = fma(d, share[w], -acc);        // C16: group w carries share_w of the ramp
}

__global__ void apply_deficit_kernel(int n, const int* __restrict__ turn, const double* __restrict__ defw,
                                     const double* __restrict__ Hd, const double* __restrict__ sw,
                                     double* __restrict__ x) {
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
    const int w = turn[i];
    x[i] += defw[w] / (Hd[i] * sw[w]);
  }
}

__global__ void project_apply_kernel(int n, int par, const int* __restrict__ turn, const double* __restrict__ vw,
                                     const double* __restrict__ Hd, double* __restrict__ r, double* __restrict__ g,
                                     Scalars* sc) {
  double acc = 0.0;
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
    double ri = r[i];
    if (turn) {
      ri -= vw[turn[i]];
      r[i] = ri;
    }
    const double gi = ri / Hd[i];
    g[i] = gi;
    acc = fma(ri, gi, acc);
  }
  block_atomic_sum(acc, &sc->rg[par]);
}

__global__ void direction_kernel(int n, int par, int first, const double* __restrict__ g, double* __restrict__ p,
                                 Scalars* sc) {
  const double beta = first ? 0.0 : sc->rg[par] / sc->rg[par ^ 1];
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x)
    p[i] = first ? -g[i] : fma(beta, p[i], -g[i]);
}
// runs after direction_kernel (stream order): the scalars of the finished iteration are no longer needed
__global__ void recycle_scalars_kernel(int par, Scalars* sc) {
  sc->rg[par ^ 1] = 0.0;
  sc->pq[0] = 0.0;
}

__global__ void axpy_kernel(int n, double a, const double* __restrict__ x, double* __restrict__ y) {
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) y[i] = fma(a, x[i], y[i]);
}
__global__ void lincomb_kernel(int n, double a, const double* __restrict__ x, double b, double* __restrict__ y) {
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) y[i] = fma(a, x[i], b * y[i]);
}
__global__ void max_scaled_diff_kernel(int n, double s, const double* __restrict__ x1, const double* __restrict__ x2,
                                       const double* __restrict__ d, Scalars* sc) {
  double m = 0.0;
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x)
    m = fmax(m, fabs(s * (x1[i] - x2[i]) / d[i]));
  m = warp_max(m);
  if ((threadIdx.x & 31) == 0 && m > 0.0)   // non-negative doubles order like their bit patterns
    atomicMax(reinterpret_cast<unsigned long long*>(&sc->djmax), static_cast<unsigned long long>(__double_as_longlong(m)));
}
__global__ void scale_div_kernel(int n, double a, const double* __restrict__ x, const double* __restrict__ d,
                                 double* __restrict__ y) {
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) y[i] += a * x[i] / d[i];
}
__global__ void mul_kernel(int n, const double* __restrict__ a, const double* __restrict__ b, double* __restrict__ y) {
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) y[i] = a[i] * b[i];
}
__global__ void set_scalars_kernel(Scalars* sc) {
  sc->rg[0] = sc->rg[1] = sc->pq[0] = sc->pq[1] = sc->nu2 = 0.0;
  sc->rd[0] = sc->rd[1] = 0.0;
  sc->done = 0;
  sc->iters = 0;
  sc->blocks_done = 0u;
  sc->thresh2 = 0.0;
  sc->uterm = sc->joule = 0.0;
  sc->tmax = 0.0;
  sc->djmax = 0.0;
  sc->nonfinite = 0;
  sc->event_or = 0;
}
__global__ void copy_rg_to_nu2_kernel(int par, Scalars* sc) {
  sc->nu2 = sc->rg[par];
  sc->rg[par] = 0.0;
}
__global__ void nu_residual_kernel(int n, double I_ramp, const double* __restrict__ Mxp1,
                                   const double* __restrict__ shift, const double* __restrict__ xp1, Rhs b,
                                   double* __restrict__ r) {
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x)
    r[i] = I_ramp * fma(shift[i], xp1[i], Mxp1[i]) - rhs_at(b, i);
}
__global__ void field_scale_kernel(int n, const double* __restrict__ bracc, const double* __restrict__ bzacc,
                                   const double* __restrict__ r, const double* __restrict__ selfcoef,
                                   const double* __restrict__ cur, double* __restrict__ Br, double* __restrict__ Bz) {
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
    Br[i] = (0.25 * kMu0) * bracc[i] / r[i];
    Bz[i] = fma(0.25 * kMu0, bzacc[i], selfcoef[i] * cur[i]);
  }
}
__global__ void sum_uterm_kernel(int n, const double* __restrict__ share, const double* __restrict__ vsum, Scalars* sc) {
  double acc = 0.0;                                          // U_terminal = -sum_w share_w V_w (C16)
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) acc = fma(share[i], vsum[i], acc);
  block_atomic_sum(acc, &sc->uterm);
}
__global__ void gather_kernel(int n, int npad, const double* __restrict__ src, const int* __restrict__ perm,
                              double* __restrict__ dst) {
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < npad; i += gridDim.x * blockDim.x)
    dst[i] = i < n ? src[perm ? perm[i] : i] : 0.0;
}
__global__ void scatter_scaled_kernel(int n, const double* __restrict__ src, const int* __restrict__ perm,
                                      double* __restrict__ dst, double scale) {
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x)
    dst[perm ? perm[i] : i] = scale * src[i];
}

// ---- fused step kernels (qs_step with constraint groups): few launches per step, no host round trip before the CG's
// first convergence test ---------------------------------------------------------------------------------------------
__global__ void step_begin_kernel(StepBegin a, Scalars* sc) {
  const int tid = blockIdx.x * blockDim.x + threadIdx.x, nth = gridDim.x * blockDim.x;
  // state backups, CG start (plain warm start or the linear extrapolation 2 I'_k - I'_{k-1}), ring currents I = a J
  for (int i = tid; i < a.N; i += nth) {
    const double Ji = a.J[i];
    a.Jold[i] = Ji;
    a.Hold[i] = a.H[i];
    const double xi = a.x[i];
    a.xold[i] = xi;
    if (a.extrapolate) a.x[i] = fma(2.0, xi, -a.xprev2[i]);
    a.xprev2[i] = xi;
    a.cur[i] = a.area[i] * Ji;
  }
  // the two contiguous backup blocks (derived fields; per-turn event state), 8 bytes at a time
  for (size_t i = tid; i < a.fld_words; i += nth) a.fld_backup[i] = a.fld[i];
  for (size_t i = tid; i < a.ev_words; i += nth) a.ev_backup[i] = a.ev[i];
  // sweep accumulators + work counter, per-turn scratch, event observables of the material pass, solver scalars
  for (size_t i = tid; i < a.acc_words; i += nth) a.acc[i] = 0ull;
  for (int w = tid; w < a.n_turns; w += nth) {
    a.vsum[w] = 0.0;
    a.tw[w] = 0.0;
    if (a.xmax_bits) {
      a.xmax_bits[w] = 0ull;
      a.rmin_bits[w] = ~0ull;
    }
  }
  if (tid == 0) {
    sc->rg[0] = sc->rg[1] = sc->pq[0] = sc->pq[1] = sc->nu2 = 0.0;
    sc->rd[0] = sc->rd[1] = 0.0;
    sc->done = 0;
    sc->iters = 0;
    sc->blocks_done = 0u;
    sc->thresh2 = 0.0;
    sc->uterm = sc->joule = 0.0;
    sc->tmax = 0.0;
    sc->djmax = 0.0;
    sc->nonfinite = 0;
    sc->event_or = 0;
  }
}

constexpr int kTurnBlockMax = 1024;   // threads per constraint group: the power of two next to its cell count, 64..1024
__device__ __forceinline__ double turn_block_sum(double v, double* sh) {   // sum over the CTA, result in every thread
  v = warp_sum(v);
  __syncthreads();
  if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = v;
  __syncthreads();
  double s = 0.0;
  for (int k = 0; k < static_cast<int>(blockDim.x >> 5); ++k) s += sh[k];
  return s;
}
inline int turn_block(const VecCtx& v) {
  const int per = (v.N + v.n_turns - 1) / (v.n_turns > 0 ? v.n_turns : 1);
  int b = 64;
  while (b < per && b < kTurnBlockMax) b <<= 1;
  return b;
}

// one CTA per constraint group: deficit_w = d share_w - sum_{i in w} x_i ; x_i += deficit_w / (H_i s_w)  (C8: moves a
// warm start onto the constraint; H = diag(M), s_w its per-turn Schur scalar)
__global__ void __launch_bounds__(kTurnBlockMax) turn_fix_kernel(const int* __restrict__ ptr, const int* __restrict__ idx,
                                                              const double* __restrict__ share, double d,
                                                              const double* __restrict__ Hd, const double* __restrict__ sw,
                                                              double* __restrict__ x) {
  __shared__ double sh[kTurnBlockMax / 32];
  const int w = blockIdx.x, k0 = ptr[w], k1 = ptr[w + 1], nt = blockDim.x;
  double acc = 0.0;
  for (int k = k0 + threadIdx.x; k < k1; k += nt) acc += x[idx[k]];
  const double def = fma(d, share[w], -turn_block_sum(acc, sh)) / sw[w];
  for (int k = k0 + threadIdx.x; k < k1; k += nt) {
    const int i = idx[k];
    x[i] += def / Hd[i];
  }
}

// one CTA per constraint group, after the material pass: everything between the sweep and the first convergence test
// of the projected CG (C8), for BOTH residuals at once -
//   r1 = I_ramp (M xp1 + shift xp1) - b   (cold start: its projected norm is the reference norm nu)
//   r2 = M x + shift x - b                (the warm start x, already on the constraint)
// s_w = sum 1/H, v = (sum r/H)/s_w, r <- r - v, g = r/H, nu2 += r1.g1, rg[0] += r2.g2, p = -g2; the multipliers of the
// two projections go to vnu[w] and vsum[w].
__global__ void __launch_bounds__(kTurnBlockMax) turn_start_kernel(TurnStart a, Scalars* sc) {
  __shared__ double sh[kTurnBlockMax / 32];
  const int w = blockIdx.x, k0 = a.ptr[w], k1 = a.ptr[w + 1], kTurnBlock = blockDim.x;
  double s = 0.0, a1 = 0.0, a2 = 0.0;
  for (int k = k0 + threadIdx.x; k < k1; k += kTurnBlock) {
    const int i = a.idx[k];
    const double hinv = 1.0 / a.Hd[i], bi = rhs_at(a.b, i), sh_i = a.shift[i];
    const double r1 = a.I_ramp * fma(sh_i, a.xp1[i], a.Mxp1[i]) - bi;
    const double r2 = fma(sh_i, a.x[i], a.cM * a.yacc[i]) - bi;
    a.g[i] = r1;          // parked until the second pass
    a.r[i] = r2;
    s += hinv;
    a1 = fma(r1, hinv, a1);
    a2 = fma(r2, hinv, a2);
  }
  s = turn_block_sum(s, sh);
  const double v1 = turn_block_sum(a1, sh) / s, v2 = turn_block_sum(a2, sh) / s;
  double nu2 = 0.0, rg = 0.0;
  for (int k = k0 + threadIdx.x; k < k1; k += kTurnBlock) {
    const int i = a.idx[k];
    const double hinv = 1.0 / a.Hd[i];
    const double r1 = a.g[i] - v1, r2 = a.r[i] - v2;
    const double g2 = r2 * hinv;
    nu2 = fma(r1 * hinv, r1, nu2);
    rg = fma(r2, g2, rg);
    a.r[i] = r2;
    a.g[i] = g2;
    a.p[i] = -g2;
  }
  nu2 = turn_block_sum(nu2, sh);
  rg = turn_block_sum(rg, sh);
  if (threadIdx.x == 0) {
    a.sw[w] = s;
    a.vnu[w] = v1;
    a.vsum[w] = v2;
    atomicAdd(&sc->nu2, nu2);
    atomicAdd(&sc->rg[0], rg);
  }
}

// S5 (J += dt I'/a) and the terminal voltage sum_w share_w vsum_w in one launch
__global__ void step_update_kernel(int n, double dt, const double* __restrict__ x, const double* __restrict__ area,
                                   double* __restrict__ J, int n_turns, const double* __restrict__ share,
                                   const double* __restrict__ vsum, Scalars* sc) {
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) J[i] += dt * x[i] / area[i];
  if (blockIdx.x == 0) {
    double acc = 0.0;
    for (int w = threadIdx.x; w < n_turns; w += blockDim.x) acc = fma(share[w], vsum[w], acc);
    block_atomic_sum(acc, &sc->uterm);
  }
}

// ---- patch (block-Jacobi) constraint preconditioner of the lattice solves -------------------------------------------
// H = blockdiag over square patches of p x p cells inside one wire of (M_patch + diag(shift)); the projection of C8 with
// a block H:  t = H^-1 r,  s_w = sum_{i in w} (H^-1 1)_i,  v_w = (sum_{i in w} t_i)/s_w,  g = t - v_w H^-1 1,  r <- r - v_w.
// Patches never straddle a constraint group, so the per-turn Schur complement stays diagonal.
// Three shapes (qs_api.cu patch_setup): p <= 8 inverted in shared memory (patch_invert_kernel); the whole wire for wires
// of 9 x 9 to 16 x 16 cells, inverted by a blocked elimination in global memory (patch_invert_big_kernel); and for wires
// larger than that p <= 8 plus a second level of patch-wise constants per wire (coarse_* kernels).
constexpr int kPatchMax = 64;   // cells per patch (p <= 8)
constexpr int kWireMax = 256;   // cells per patch of the big patches (p <= 16: whole wires of up to 16 x 16 cells)

// once per qs_init: the constant part M_patch [H] of every patch, pair by pair with the sweeps' arithmetic
// (big patches: one matrix per (layer, radial slot) = blockIdx.x, evaluated on that slot's first patch of the layer)
__global__ void __launch_bounds__(kWireMax) patch_build_kernel(int pp, int per, int per_layer, const int* __restrict__ pidx,
                                                              const double* __restrict__ r, const double* __restrict__ z,
                                                              double soft_all, double soft_self, double* __restrict__ Pm) {
  const int pch = per > 0 ? ((blockIdx.x / per) * per_layer * per + blockIdx.x % per) * per : blockIdx.x;
  const int t = threadIdx.x;
  if (t >= pp) return;
  const int i = pidx[pch * pp + t];
  const double ri = r[i], zi = z[i];
  double* row = Pm + (static_cast<size_t>(blockIdx.x) * pp + t) * pp;
  for (int u = 0; u < pp; ++u) {
    const int j = pidx[pch * pp + u];
    const double rj = r[j], dz = zi - z[j];
    const double dz2 = fma(dz, dz, soft_all) + (u == t ? soft_self : 0.0);
    const double dif = ri - rj;
    const double B2 = fma(dif, dif, dz2), A2 = fma(4.0 * ri, rj, B2);
    const PairAGM a = agm_pair<7, 2, false>(A2, B2);
    row[u] = (0.5 * kMu0 * kPi) * a.S * a.yinf;
  }
}

// per solve: Pinv = (M_patch + diag(shift))^-1 by in-place Gauss-Jordan elimination in shared memory (SPD: no pivoting),
// h1 = Pinv 1, s_w += sum h1.  One CTA per patch, kPinvSplit threads per row (each owns every kPinvSplit-th column).
constexpr int kPinvSplit = 4;
// (H1_ATOMIC: h1 is accumulated, not stored - the coarse level of the same launch adds its part in any order)
template <bool H1_ATOMIC>
__device__ __forceinline__ void patch_invert_body(double (*A)[kPatchMax + 1], double* part, int pch, int pp,
                                                  const int* __restrict__ pidx, const int* __restrict__ pturn,
                                                  const double* __restrict__ Pm, const double* __restrict__ shift,
                                                  double* __restrict__ Pinv, double* __restrict__ h1,
                                                  double* __restrict__ sw) {
  const int nthr = pp * kPinvSplit;
  const int t = threadIdx.x / kPinvSplit, c = threadIdx.x % kPinvSplit;   // row, column phase
  const bool act = static_cast<int>(threadIdx.x) < nthr;
  const double* src = Pm + static_cast<size_t>(pch) * pp * pp;
  for (int e = threadIdx.x; e < pp * pp; e += blockDim.x) A[e / pp][e % pp] = src[e];
  __syncthreads();
  if (threadIdx.x < pp) A[threadIdx.x][threadIdx.x] += shift[pidx[pch * pp + threadIdx.x]];
  __syncthreads();
  for (int k = 0; k < pp; ++k) {
    const double piv = 1.0 / A[k][k];
    const double f = act ? A[t][k] : 0.0;
    __syncthreads();
    if (act && t == k) {
      for (int u = c; u < pp; u += kPinvSplit) A[k][u] = (u == k) ? piv : A[k][u] * piv;
    }
    __syncthreads();
    if (act && t != k) {
      for (int u = c; u < pp; u += kPinvSplit) A[t][u] = (u == k) ? -f * piv : fma(-f, A[k][u], A[t][u]);
    }
    __syncthreads();
  }
  double hs = 0.0;
  if (act) {
    double* row = Pinv + (static_cast<size_t>(pch) * pp + t) * pp;
    for (int u = c; u < pp; u += kPinvSplit) {
      // symmetrised on the way out (the elimination leaves rounding-level asymmetry)
      const double v = 0.5 * (A[t][u] + A[u][t]);
      row[u] = v;
      hs += v;
    }
  }
  // row sums: the kPinvSplit threads of a row are adjacent lanes
#pragma unroll
  for (int o = kPinvSplit / 2; o > 0; o >>= 1) hs += __shfl_xor_sync(0xffffffffu, hs, o);
  if (act && c == 0) {
    if (H1_ATOMIC) atomicAdd(h1 + pidx[pch * pp + t], hs);
    else h1[pidx[pch * pp + t]] = hs;
  }
  double tot = (act && c == 0) ? hs : 0.0;
  tot = warp_sum(tot);
  if ((threadIdx.x & 31) == 0) part[threadIdx.x >> 5] = tot;
  __syncthreads();
  if (threadIdx.x == 0) {
    double ssum = 0.0;
    for (int k = 0; k < static_cast<int>(blockDim.x >> 5); ++k) ssum += part[k];
    atomicAdd(sw + pturn[pch], ssum);
  }
}
__global__ void __launch_bounds__(kPatchMax * kPinvSplit) patch_invert_kernel(int pp, const int* __restrict__ pidx,
                                                                              const int* __restrict__ pturn,
                                                                              const double* __restrict__ Pm,
                                                                              const double* __restrict__ shift,
                                                                              double* __restrict__ Pinv, double* __restrict__ h1,
                                                                              double* __restrict__ sw) {
  __shared__ double A[kPatchMax][kPatchMax + 1];
  __shared__ double part[kPatchMax * kPinvSplit / 32];
  patch_invert_body<false>(A, part, blockIdx.x, pp, pidx, pturn, Pm, shift, Pinv, h1, sw);
}

// t = Pinv r over one patch; parks t in g and adds sum t to tw[turn].  UPDATE: first x += alpha p, r += alpha q
// (the fused CG iteration's update); else r is taken as it is (start of the solve).  SPLIT threads per row (adjacent
// lanes, each a part of the row product): 4 for the patches of <= 64 cells (few, small CTAs: the product is a latency
// chain), 1 for the big patches.
template <bool UPDATE, int SPLIT>
__global__ void __launch_bounds__(kWireMax) patch_apply_kernel(int pp, const int* __restrict__ pidx,
                                                              const int* __restrict__ pturn,
                                                              const double* __restrict__ Pinv, CgIter it, Scalars* sc) {
  __shared__ double rs[kWireMax];
  __shared__ double part[kWireMax / 32];
  if (UPDATE && sc->done) return;
  double alpha = 0.0;
  if (UPDATE) {
    const double pq = sc->pq[it.par];
    if (!(pq > 0.0)) {   // breakdown: every thread sees the same pq and leaves the state alone
      if (blockIdx.x == 0 && threadIdx.x == 0) sc->done = 2;
      return;
    }
    alpha = sc->rg[it.par] / pq;
  }
  const int pch = blockIdx.x, t = threadIdx.x / SPLIT, c = threadIdx.x % SPLIT;
  const bool act = t < pp;
  const int i = act ? pidx[pch * pp + t] : 0;
  if (act && c == 0) {
    double ri = it.r[i];
    if (UPDATE) {
      it.x[i] = fma(alpha, it.p[i], it.x[i]);
      ri = fma(alpha, it.q[i], ri);
      it.r[i] = ri;
    }
    rs[t] = ri;
  }
  __syncthreads();
  double acc = 0.0;
  if (act) {
    const double* col = Pinv + static_cast<size_t>(pch) * pp * pp + t;   // column t = row t (symmetric): coalesced
    for (int u = c; u < pp; u += SPLIT) acc = fma(col[static_cast<size_t>(u) * pp], rs[u], acc);
  }
#pragma unroll
  for (int o = SPLIT / 2; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
  if (act && c == 0) it.g[i] = acc;
  double tot = (act && c == 0) ? acc : 0.0;
  tot = warp_sum(tot);
  if ((threadIdx.x & 31) == 0) part[threadIdx.x >> 5] = tot;
  __syncthreads();
  if (threadIdx.x == 0) {
    double s = 0.0;
    for (int k = 0; k < static_cast<int>((blockDim.x + 31) >> 5); ++k) s += part[k];
    atomicAdd(it.tw + pturn[pch], s);
    if (it.patch.nc > 0) {             // second level: restricted residual of this patch
      double rsum = 0.0;
      for (int u = 0; u < pp; ++u) rsum += rs[u];
      it.patch.rc[pch] = rsum;
    }
  }
}

// ---- second level: piecewise constants per patch (wires larger than one patch: config 1) -----------------------------
// Host experiment (single wire of 32 x 32 cells in a fast field ramp, surface at Jc, warm start): 8 x 8 patches alone 85
// iterations, 16 x 16 patches 50, 8 x 8 patches + this coarse space 45 (4 x 4 + coarse: 46): what the patches miss are
// the wire-scale screening-current modes, and patch-wise constants carry them.
// once per qs_init: C0m[layer][P][Q] = sum_{i in P, j in Q} M_ij on the first wire of the layer, one CTA per (layer, P, Q)
__global__ void __launch_bounds__(kPatchMax) coarse_build_kernel(PatchPrec pc, const double* __restrict__ r,
                                                                const double* __restrict__ z, double soft_all,
                                                                double soft_self) {
  __shared__ double part[kPatchMax / 32];
  const int nc = pc.nc, pp = pc.pp, t = threadIdx.x;
  const int Q = blockIdx.x % nc, P = (blockIdx.x / nc) % nc, layer = blockIdx.x / (nc * nc);
  const int w0 = layer * pc.per_layer;                            // first wire of the layer
  const int* iP = pc.pidx + (static_cast<size_t>(w0) * nc + P) * pp;
  const int* iQ = pc.pidx + (static_cast<size_t>(w0) * nc + Q) * pp;
  double acc = 0.0;
  if (t < pp) {
    const int i = iP[t];
    const double ri = r[i], zi = z[i];
    for (int u = 0; u < pp; ++u) {
      const int j = iQ[u];
      const double rj = r[j], dz = zi - z[j];
      const double dz2 = fma(dz, dz, soft_all) + (i == j ? soft_self : 0.0);
      const double dif = ri - rj;
      const double B2 = fma(dif, dif, dz2), A2 = fma(4.0 * ri, rj, B2);
      const PairAGM a = agm_pair<7, 2, false>(A2, B2);
      acc += (0.5 * kMu0 * kPi) * a.S * a.yinf;
    }
  }
  acc = warp_sum(acc);
  if ((t & 31) == 0) part[t >> 5] = acc;
  __syncthreads();
  if (t == 0) {
    double s = 0.0;
    for (int k = 0; k < static_cast<int>(blockDim.x >> 5); ++k) s += part[k];
    pc.C0m[blockIdx.x] = s;
  }
}

// per solve, after the patch inverses: C0inv[w] = (C0m[layer] + diag(sum of the shift over each patch))^-1 by the same
// elimination in shared memory; h1 += Z C Z^T 1, s_w += its sum.  One CTA per wire, kPinvSplit threads per coarse
// unknown (each owns every kPinvSplit-th column; a single wire is a single CTA, so the row work is spread).
__device__ __forceinline__ void coarse_invert_body(double (*A)[kPatchMax + 1], double* hc, int w, const PatchPrec& pc,
                                                   const double* __restrict__ shift) {
  const int nc = pc.nc, pp = pc.pp;
  const int t = threadIdx.x / kPinvSplit, c = threadIdx.x % kPinvSplit;   // row, column phase
  const bool act = t < nc;
  const double* src = pc.C0m + static_cast<size_t>(w / pc.per_layer) * nc * nc;
  for (int e = threadIdx.x; e < nc * nc; e += blockDim.x) A[e / nc][e % nc] = src[e];
  __syncthreads();
  double ssum = 0.0;
  if (act) {
    const int* idx = pc.pidx + (static_cast<size_t>(w) * nc + t) * pp;
    for (int u = c; u < pp; u += kPinvSplit) ssum += shift[idx[u]];
  }
#pragma unroll
  for (int o = kPinvSplit / 2; o > 0; o >>= 1) ssum += __shfl_xor_sync(0xffffffffu, ssum, o);
  if (act && c == 0) A[t][t] += ssum;
  __syncthreads();
  for (int k = 0; k < nc; ++k) {
    const double piv = 1.0 / A[k][k];
    const double f = act ? A[t][k] : 0.0;
    __syncthreads();
    if (act && t == k)
      for (int u = c; u < nc; u += kPinvSplit) A[k][u] = (u == k) ? piv : A[k][u] * piv;
    __syncthreads();
    if (act && t != k)
      for (int u = c; u < nc; u += kPinvSplit) A[t][u] = (u == k) ? -f * piv : fma(-f, A[k][u], A[t][u]);
    __syncthreads();
  }
  double h = 0.0;
  if (act) {
    double* row = pc.C0inv + (static_cast<size_t>(w) * nc + t) * nc;
    for (int u = c; u < nc; u += kPinvSplit) {
      const double v = 0.5 * (A[t][u] + A[u][t]);                 // symmetrised on the way out
      row[u] = v;
      h += v;
    }
  }
#pragma unroll
  for (int o = kPinvSplit / 2; o > 0; o >>= 1) h += __shfl_xor_sync(0xffffffffu, h, o);
  if (act && c == 0) hc[t] = h * pp;                               // (C Z^T 1)_t : Z^T 1 = pp on every patch
  __syncthreads();
  for (int e = threadIdx.x; e < nc * pp; e += blockDim.x) {        // h1 += Z hc over the cells of the wire
    const int q = e / pp;
    atomicAdd(pc.h1 + pc.pidx[(static_cast<size_t>(w) * nc + q) * pp + (e - q * pp)], hc[q]);
  }
  if (threadIdx.x == 0) {
    double s = 0.0;
    for (int q = 0; q < nc; ++q) s += hc[q];
    atomicAdd(pc.sw + w, s * pp);
  }
}
// both levels in ONE launch (CTAs 0 .. n_patches-1: the patches, the rest: one per wire); h1 and s_w are accumulated with
// atomics into zeroed arrays, so the two levels need no order (config 1: the single coarse CTA of 0.13 ms hides behind
// the 64 patch CTAs instead of following them)
__global__ void __launch_bounds__(kPatchMax * kPinvSplit) two_level_invert_kernel(PatchPrec pc, const double* __restrict__ shift) {
  __shared__ double A[kPatchMax][kPatchMax + 1];
  __shared__ double part[kPatchMax * kPinvSplit / 32];
  __shared__ double hc[kPatchMax];
  if (static_cast<int>(blockIdx.x) < pc.n_patches)
    patch_invert_body<true>(A, part, blockIdx.x, pc.pp, pc.pidx, pc.pturn, pc.Pm, shift, pc.Pinv, pc.h1, pc.sw);
  else
    coarse_invert_body(A, hc, static_cast<int>(blockIdx.x) - pc.n_patches, pc, shift);
}

// per iteration, after the patch products: yc = C0inv (Z^T r) per wire, tw[w] += sum of Z yc.  kPinvSplit threads per
// coarse unknown (adjacent lanes, each a quarter of the row product).
template <bool UPDATE>
__global__ void __launch_bounds__(kPatchMax * kPinvSplit) coarse_apply_kernel(PatchPrec pc, double* __restrict__ tw, Scalars* sc) {
  __shared__ double rs[kPatchMax];
  __shared__ double part[kPatchMax * kPinvSplit / 32];
  if (UPDATE && sc->done) return;
  const int nc = pc.nc, w = blockIdx.x;
  const int t = threadIdx.x / kPinvSplit, c = threadIdx.x % kPinvSplit;
  if (threadIdx.x < nc) rs[threadIdx.x] = pc.rc[static_cast<size_t>(w) * nc + threadIdx.x];
  __syncthreads();
  double acc = 0.0;
  if (t < nc) {
    const double* row = pc.C0inv + (static_cast<size_t>(w) * nc + t) * nc;
    for (int u = c; u < nc; u += kPinvSplit) acc = fma(row[u], rs[u], acc);
  }
#pragma unroll
  for (int o = kPinvSplit / 2; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
  if (t < nc && c == 0) pc.yc[static_cast<size_t>(w) * nc + t] = acc;
  double tot = (t < nc && c == 0) ? acc : 0.0;
  tot = warp_sum(tot);
  if ((threadIdx.x & 31) == 0) part[threadIdx.x >> 5] = tot;
  __syncthreads();
  if (threadIdx.x == 0) {
    double s = 0.0;
    for (int k = 0; k < static_cast<int>(blockDim.x >> 5); ++k) s += part[k];
    atomicAdd(tw + w, s * pc.pp);
  }
}

// ---- patches of more than 64 cells (p = 9..16: whole wires of configs 2 and 3, 16 x 16 sub-wire patches of config 1) ----
// A 256 x 256 block does not fit shared memory, so the per-solve inverse is formed by a Gauss-Jordan elimination IN GLOBAL
// MEMORY (the block stays in L2 while its CTA works on it).  The constant part is shared: patches in the same layer and
// radial slot of their wire are translates of each other along z, so Pm holds one matrix per (layer, radial slot).
// Why whole wires: measured on the host on mid-trajectory systems of shrunk configs 2 / 3 with the surface cells at Jc
// (warm start), 2 x 2 ... 8 x 8 sub-wire patches all need 87-97 iterations, the whole wire 41 / 44: only the full block
// carries the wire's screening-current modes.  A fixed inverse of M_wire with a diagonal scaling for the shift (no
// per-solve inversion) does as well there (43 / 44) but not when the shift is comparable to diag(M) (single wire of
// 32 x 32 cells under a fast field ramp, shift / diag(M) up to 3: 165 iterations against 50), so the inverse is exact.
__device__ __forceinline__ int patch_pm_index(const PatchPrec& pc, int pch) {
  return (pch / (pc.per_layer * pc.per * pc.per)) * pc.per + (pch / pc.per) % pc.per;   // (layer, radial slot)
}
// BLOCKED elimination with block size p (the wire side: pp = p blocks of p): per block step K the pivot block is inverted
// in shared memory, the row panel P^-1 A[K, :] and the column panel A[:, K] are staged in shared memory, and every
// other element takes ONE rank-p update from them (4 x 4 register tiles), so the block is read and written p times
// instead of p^2 times (element-wise elimination in global memory: 45 ms per solve at config 2, L2-bandwidth bound):
//   A[K,K] <- P^-1;  A[K,j] <- P^-1 A[K,j];  A[i,j] <- A[i,j] - A[i,K] (P^-1 A[K,j]);  A[i,K] <- -A[i,K] P^-1   (i, j != K)
constexpr int kBigThreads = 512;
__host__ __device__ inline int big_ldr(int pp) { return (pp + 3) / 4 * 4; }
static size_t big_invert_smem(int p) {
  const int pp = p * p, ldr = big_ldr(pp);
  return sizeof(double) * (static_cast<size_t>(p) * (p + 1) + static_cast<size_t>(p) * ldr + static_cast<size_t>(ldr) * (p + 1));
}
__global__ void __launch_bounds__(kBigThreads, 2) patch_invert_big_kernel(PatchPrec pc, int p, const double* __restrict__ shift) {
  extern __shared__ __align__(16) double bsm[];
  __shared__ double part[kBigThreads / 32];
  const int pp = pc.pp, pch = blockIdx.x, nthr = blockDim.x, tid = threadIdx.x;
  const int ldr = big_ldr(pp), ldc = p + 1;
  double* Pb = bsm;                    // [p][p + 1]   pivot block, then its inverse
  double* R = Pb + p * (p + 1);        // [p][ldr]     row panel (columns past pp: zero)
  double* Cp = R + p * ldr;            // [ldr][p + 1] column panel (rows past pp: zero)
  const double* src = pc.Pm + static_cast<size_t>(patch_pm_index(pc, pch)) * pp * pp;
  double* A = pc.Pinv + static_cast<size_t>(pch) * pp * pp;
  const int* idx = pc.pidx + static_cast<size_t>(pch) * pp;
  for (int e = tid; e < pp * pp; e += nthr) {                      // A = M_patch + diag(shift)
    const int i = e / pp, u = e - i * pp;
    A[e] = src[e] + (i == u ? shift[idx[i]] : 0.0);
  }
  for (int e = tid; e < p * ldr; e += nthr) R[e] = 0.0;
  for (int e = tid; e < ldr * ldc; e += nthr) Cp[e] = 0.0;
  __syncthreads();
  const int ri = tid / p, ci = tid % p;                            // element of the pivot block (tid < p * p)
  const bool inP = tid < p * p;
  const int ntile = ldr / 4;
  for (int K = 0; K < p; ++K) {
    const int k0 = K * p;
    if (inP) Pb[ri * ldc + ci] = A[(k0 + ri) * pp + k0 + ci];
    for (int e = tid; e < p * pp; e += nthr) {
      const int m = e / pp, j = e - m * pp;
      R[m * ldr + j] = A[(k0 + m) * pp + j];
    }
    for (int e = tid; e < pp * p; e += nthr) {
      const int i = e / p, m = e - i * p;
      Cp[i * ldc + m] = A[i * pp + k0 + m];
    }
    __syncthreads();
    for (int k = 0; k < p; ++k) {                                  // pivot block: element-wise elimination in shared memory
      double v = 0.0;
      if (inP) {
        const double piv = 1.0 / Pb[k * ldc + k];
        const double f = Pb[ri * ldc + k], rv = Pb[k * ldc + ci];
        if (ri == k) v = (ci == k) ? piv : rv * piv;
        else if (ci == k) v = -f * piv;
        else v = fma(-f * piv, rv, Pb[ri * ldc + ci]);
      }
      __syncthreads();
      if (inP) Pb[ri * ldc + ci] = v;
      __syncthreads();
    }
    if (tid < pp) {                                                // row panel in place, one column per thread
      const int j = tid;
      if (j >= k0 && j < k0 + p) {
        for (int m = 0; m < p; ++m) R[m * ldr + j] = Pb[m * ldc + (j - k0)];
      } else {
        double col[16];
#pragma unroll
        for (int q = 0; q < 16; ++q) col[q] = q < p ? R[q * ldr + j] : 0.0;
        for (int m = 0; m < p; ++m) {
          double acc = 0.0;
#pragma unroll
          for (int q = 0; q < 16; ++q)
            if (q < p) acc = fma(Pb[m * ldc + q], col[q], acc);
          R[m * ldr + j] = acc;
        }
      }
    }
    __syncthreads();
    for (int tile = tid; tile < ntile * ntile; tile += nthr) {     // rank-p update, 4 x 4 elements per tile
      const int i0 = (tile / ntile) * 4, j0 = (tile % ntile) * 4;
      double acc[4][4];
#pragma unroll
      for (int a = 0; a < 4; ++a)
#pragma unroll
        for (int b = 0; b < 4; ++b) acc[a][b] = 0.0;
      for (int m = 0; m < p; ++m) {
        const double2 r01 = *reinterpret_cast<const double2*>(R + m * ldr + j0);
        const double2 r23 = *reinterpret_cast<const double2*>(R + m * ldr + j0 + 2);
        const double rr[4] = {r01.x, r01.y, r23.x, r23.y};
#pragma unroll
        for (int a = 0; a < 4; ++a) {
          const double c = Cp[(i0 + a) * ldc + m];
#pragma unroll
          for (int b = 0; b < 4; ++b) acc[a][b] = fma(c, rr[b], acc[a][b]);
        }
      }
#pragma unroll
      for (int a = 0; a < 4; ++a) {
        const int i = i0 + a;
        if (i >= pp) continue;
        const bool rowK = i >= k0 && i < k0 + p;
#pragma unroll
        for (int b = 0; b < 4; ++b) {
          const int j = j0 + b;
          if (j >= pp) continue;
          const bool colK = j >= k0 && j < k0 + p;
          double v;
          if (rowK) v = R[(i - k0) * ldr + j];
          else v = (colK ? 0.0 : A[i * pp + j]) - acc[a][b];
          A[i * pp + j] = v;
        }
      }
    }
    __syncthreads();
  }
  for (int e = threadIdx.x; e < pp * pp; e += nthr) {             // symmetrise (rounding-level asymmetry of the elimination)
    const int i = e / pp, u = e - i * pp;
    if (u > i) {
      const double v = 0.5 * (A[e] + A[u * pp + i]);
      A[e] = v;
      A[u * pp + i] = v;
    }
  }
  __syncthreads();
  // h1 = Pinv 1 (one warp per row), s_w += sum h1
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarps = nthr >> 5;
  double tot = 0.0;
  for (int i = warp; i < pp; i += nwarps) {
    double hs = 0.0;
    for (int u = lane; u < pp; u += 32) hs += A[i * pp + u];
    hs = warp_sum(hs);
    if (lane == 0) pc.h1[idx[i]] = hs, tot += hs;
  }
  if (lane == 0) part[warp] = tot;
  __syncthreads();
  if (threadIdx.x == 0) {
    double ssum = 0.0;
    for (int k = 0; k < nwarps; ++k) ssum += part[k];
    atomicAdd(pc.sw + pc.pturn[pch], ssum);
  }
}

// r -= v_w ; g = t - v_w h1 ; rg[slot] += r.g ; FIRST: p = -g (start of the solve)
template <bool FIRST>
__global__ void patch_project_kernel(int n, CgIter it, const int* __restrict__ turn, const double* __restrict__ h1,
                                     Scalars* sc) {
  if (!FIRST && sc->done) return;
  double acc = 0.0, accd = 0.0;
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
    const int w = turn[i];
    const double v = it.tw[w] / it.sw[w];
    const double ri = it.r[i] - v;
    const double ti = it.patch.nc > 0 ? it.g[i] + it.patch.yc[it.patch.pid[i]] : it.g[i];   // t = B r + Z yc
    const double gi = fma(-v, h1[i], ti);
    it.r[i] = ri;
    it.g[i] = gi;
    if (FIRST) it.p[i] = -gi;
    acc = fma(ri, gi, acc);
    accd = fma(ri / it.Hd[i], ri, accd);          // the stopping rule's norm: r^T diag(A)^-1 r
  }
  block_atomic_sum(acc, &sc->rg[FIRST ? 0 : it.par ^ 1]);
  __syncthreads();
  block_atomic_sum(accd, &sc->rd[FIRST ? 0 : it.par ^ 1]);
}
// vsum += tw/sw ; tw = 0  (the multipliers of the start projection; later ones are booked by the direction kernel)
__global__ void turn_book_kernel(int n_turns, double* __restrict__ tw, const double* __restrict__ sw,
                                 double* __restrict__ vsum) {
  for (int w = blockIdx.x * blockDim.x + threadIdx.x; w < n_turns; w += gridDim.x * blockDim.x) {
    vsum[w] += tw[w] / sw[w];
    tw[w] = 0.0;
  }
}

// ---- fused CG iteration ---------------------------------------------------------------------------------------------
__global__ void cg_begin_kernel(Scalars* sc, double thresh2) {
  sc->done = 0;
  sc->iters = 0;
  sc->pq[0] = sc->pq[1] = 0.0;
  sc->rd[0] = sc->rd[1] = 0.0;
  sc->blocks_done = 0u;
  sc->thresh2 = thresh2;
}

__global__ void cg_Ap_kernel(int n, CgIter it, Scalars* sc) {
  if (sc->done) return;
  double acc = 0.0;
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
    const double pi = it.p[i];
    const double qi = fma(it.shift[i], pi, it.cM * it.yacc_in[i]);
    it.q[i] = qi;
    acc = fma(pi, qi, acc);
  }
  block_atomic_sum(acc, &sc->pq[it.par]);
}

__global__ void cg_update_kernel(int n, CgIter it, const int* __restrict__ turn, Scalars* sc) {
  if (sc->done) return;
  const double pq = sc->pq[it.par];
  if (!(pq > 0.0)) {   // breakdown: every thread sees the same pq and leaves the state alone
    if (blockIdx.x == 0 && threadIdx.x == 0) sc->done = 2;
    return;
  }
  const double alpha = sc->rg[it.par] / pq;
  for (int base = blockIdx.x * blockDim.x; base < n; base += gridDim.x * blockDim.x) {
    const int i = base + threadIdx.x;
    const bool ok = i < n;
    double t = 0.0;
    int w = -1;
    if (ok) {
      it.x[i] = fma(alpha, it.p[i], it.x[i]);
      const double ri = fma(alpha, it.q[i], it.r[i]);
      it.r[i] = ri;
      if (turn) {
        t = ri / it.Hd[i];
        w = turn[i];
      }
    }
    if (turn) {   // per-turn sums: one atomic per warp when the warp lies inside one turn, else one per lane
      const int w0 = __shfl_sync(0xffffffffu, w, 0);
      if (__all_sync(0xffffffffu, w == w0 || !ok)) {
        t = warp_sum(t);
        if ((threadIdx.x & 31) == 0 && w0 >= 0) atomicAdd(it.tw + w0, t);
      } else if (ok) {
        atomicAdd(it.tw + w, t);
      }
    }
  }
}

__global__ void cg_project_kernel(int n, CgIter it, const int* __restrict__ turn, Scalars* sc) {
  if (sc->done) return;
  double acc = 0.0;
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
    double ri = it.r[i];
    if (turn) {
      const int w = turn[i];
      ri -= it.tw[w] / it.sw[w];
      it.r[i] = ri;
    }
    const double gi = ri / it.Hd[i];
    it.g[i] = gi;
    acc = fma(ri, gi, acc);
  }
  block_atomic_sum(acc, &sc->rg[it.par ^ 1]);
}

__global__ void cg_direction_kernel(int n, int npad, int n_turns, CgIter it, Scalars* sc) {
  if (sc->done) return;
  const double rg_new = sc->rg[it.par ^ 1];
  const double beta = rg_new / sc->rg[it.par];
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < npad; i += gridDim.x * blockDim.x) {
    if (i < n) it.p[i] = fma(beta, it.p[i], -it.g[i]);
    it.yacc_zero[i] = 0.0;
  }
  // the last block to finish does the bookkeeping of the iteration: every block has read the scalars by then
  __shared__ bool last;
  __threadfence();
  __syncthreads();
  if (threadIdx.x == 0) last = atomicAdd(&sc->blocks_done, 1u) == gridDim.x - 1;
  __syncthreads();
  if (!last) return;
  for (int w = threadIdx.x; w < n_turns; w += blockDim.x) {   // multipliers (C8): V = -sum of the subtracted v
    it.vsum[w] += it.tw[w] / it.sw[w];
    it.tw[w] = 0.0;
  }
  if (threadIdx.x == 0) {
    const double test = it.patch.pp > 0 ? sc->rd[it.par ^ 1] : rg_new;   // same stopping rule with either preconditioner
    sc->rg[it.par] = 0.0;
    sc->rd[it.par] = 0.0;
    sc->pq[it.par] = 0.0;
    sc->blocks_done = 0u;
    *it.counter = 0ull;
    sc->iters += 1;
    if (!(rg_new == rg_new)) sc->done = 2;
    else if (test <= sc->thresh2) sc->done = 1;
  }
}
}  // namespace

#define QS_LAUNCH(v) (g_sm_count = (v).sm_count, ++*(v).launches)

void k_finish_Ap(const VecCtx& v, const double* yacc, const double* shift, const double* p, double* q, double cM) {
  QS_LAUNCH(v);
  finish_Ap_kernel<<<grid_for(v.N), kBlock, 0, v.stream>>>(v.N, yacc, shift, p, q, cM, v.sc);
}
void k_rhs_fill(const VecCtx& v, const Rhs& b, double* r) {
  QS_LAUNCH(v);
  rhs_fill_kernel<<<grid_for(v.N), kBlock, 0, v.stream>>>(v.N, b, r);
}
void k_residual(const VecCtx& v, const double* yacc, const double* shift, const double* x, const Rhs& b, double* r,
                double cM) {
  QS_LAUNCH(v);
  residual_kernel<<<grid_for(v.N), kBlock, 0, v.stream>>>(v.N, yacc, shift, x, b, r, cM);
}
void k_update_xr(const VecCtx& v, int par, const double* p, const double* q, double* x, double* r) {
  QS_LAUNCH(v);
  update_xr_kernel<<<grid_for(v.N), kBlock, 0, v.stream>>>(v.N, par, p, q, x, r, v.sc);
}
void k_turn_project(const VecCtx& v, const double* r, const double* Hd, const double* sw, double* vw, double* vsum) {
  if (!v.n_turns) return;
  QS_LAUNCH(v);
  turn_project_kernel<<<(v.n_turns * 32 + kBlock - 1) / kBlock, kBlock, 0, v.stream>>>(v.n_turns, v.turn_ptr,
                                                                                      v.turn_idx, r, Hd, sw, vw, vsum);
}
void k_turn_schur(const VecCtx& v, const double* Hd, double* sw) {
  if (!v.n_turns) return;
  QS_LAUNCH(v);
  turn_schur_kernel<<<(v.n_turns * 32 + kBlock - 1) / kBlock, kBlock, 0, v.stream>>>(v.n_turns, v.turn_ptr, v.turn_idx,
                                                                                    Hd, sw);
}
void k_turn_deficit(const VecCtx& v, const double* x, double d, double* defw) {
  if (!v.n_turns) return;
  QS_LAUNCH(v);
  turn_deficit_kernel<<<(v.n_turns * 32 + kBlock - 1) / kBlock, kBlock, 0, v.stream>>>(v.n_turns, v.turn_ptr,
                                                                                      v.turn_idx, v.share, x, d, defw,
                                                                                      v.sc);
}
void k_apply_deficit(const VecCtx& v, const double* defw, const double* Hd, const double* sw, double* x) {
  if (!v.n_turns) return;
  QS_LAUNCH(v);
  apply_deficit_kernel<<<grid_for(v.N), kBlock, 0, v.stream>>>(v.N, v.turn_id, defw, Hd, sw, x);
}
void k_project_apply(const VecCtx& v, int par, const double* vw, const double* Hd, double* r, double* g) {
  QS_LAUNCH(v);
  project_apply_kernel<<<grid_for(v.N), kBlock, 0, v.stream>>>(v.N, par, v.n_turns ? v.turn_id : nullptr, vw, Hd, r, g,
                                                              v.sc);
}
void k_direction(const VecCtx& v, int par, bool first, const double* g, double* p) {
  QS_LAUNCH(v);
  direction_kernel<<<grid_for(v.N), kBlock, 0, v.stream>>>(v.N, par, first ? 1 : 0, g, p, v.sc);
  QS_LAUNCH(v);
  recycle_scalars_kernel<<<1, 1, 0, v.stream>>>(par, v.sc);
}
void k_cg_begin(const VecCtx& v, double thresh2) {
  QS_LAUNCH(v);
  cg_begin_kernel<<<1, 1, 0, v.stream>>>(v.sc, thresh2);
}
void k_cg_Ap(const VecCtx& v, const CgIter& it) {
  QS_LAUNCH(v);
  cg_Ap_kernel<<<grid_for(v.N), kBlock, 0, v.stream>>>(v.N, it, v.sc);
}
static int patch_threads(const PatchPrec& pc) { return pc.big ? (pc.pp + 31) / 32 * 32 : (pc.pp * kPinvSplit + 31) / 32 * 32; }
void k_cg_update(const VecCtx& v, const CgIter& it) {
  QS_LAUNCH(v);
  if (it.patch.pp > 0) {   // patch preconditioner: update fused with t = Pinv r
    if (it.patch.big)
      patch_apply_kernel<true, 1><<<it.patch.n_patches, patch_threads(it.patch), 0, v.stream>>>(it.patch.pp, it.patch.pidx,
                                                                                             it.patch.pturn, it.patch.Pinv, it, v.sc);
    else
      patch_apply_kernel<true, kPinvSplit><<<it.patch.n_patches, patch_threads(it.patch), 0, v.stream>>>(
          it.patch.pp, it.patch.pidx, it.patch.pturn, it.patch.Pinv, it, v.sc);
    if (it.patch.nc > 0) {
      QS_LAUNCH(v);
      coarse_apply_kernel<true><<<v.n_turns, kPatchMax * kPinvSplit, 0, v.stream>>>(it.patch, it.tw, v.sc);
    }
    return;
  }
  cg_update_kernel<<<grid_for(v.N), kBlock, 0, v.stream>>>(v.N, it, v.n_turns ? v.turn_id : nullptr, v.sc);
}
void k_patch_build(const VecCtx& v, const PatchPrec& pc, const double* r, const double* z, double soft_all,
                   double soft_self) {
  QS_LAUNCH(v);
  if (pc.big) {   // one matrix per (layer, radial slot)
    patch_build_kernel<<<pc.layers * pc.per, patch_threads(pc), 0, v.stream>>>(pc.pp, pc.per, pc.per_layer, pc.pidx, r, z,
                                                                              soft_all, soft_self, pc.Pm);
    return;
  }
  patch_build_kernel<<<pc.n_patches, kPatchMax, 0, v.stream>>>(pc.pp, 0, 0, pc.pidx, r, z, soft_all, soft_self, pc.Pm);
  if (pc.nc > 0) {
    QS_LAUNCH(v);
    coarse_build_kernel<<<pc.layers * pc.nc * pc.nc, kPatchMax, 0, v.stream>>>(pc, r, z, soft_all, soft_self);
  }
}
// start of a solve in patch mode: Pinv for this shift, then the block projection of the current (refined) residual
void k_patch_start(const VecCtx& v, const CgIter& it, const double* shift) {
  const PatchPrec& pc = it.patch;
  cudaMemsetAsync(pc.sw, 0, sizeof(double) * v.n_turns, v.stream);
  cudaMemsetAsync(&v.sc->rg[0], 0, sizeof(double), v.stream);
  cudaMemsetAsync(&v.sc->rd[0], 0, 2 * sizeof(double), v.stream);
  QS_LAUNCH(v);
  if (pc.big) {
    const int p = static_cast<int>(std::lround(std::sqrt(static_cast<double>(pc.pp))));
    const size_t smem = big_invert_smem(p);
    cudaFuncSetAttribute(patch_invert_big_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, static_cast<int>(smem));
    patch_invert_big_kernel<<<pc.n_patches, kBigThreads, smem, v.stream>>>(pc, p, shift);
  }
  else if (pc.nc > 0) {   // patches and coarse level in one launch
    cudaMemsetAsync(pc.h1, 0, sizeof(double) * v.N, v.stream);
    two_level_invert_kernel<<<pc.n_patches + v.n_turns, kPatchMax * kPinvSplit, 0, v.stream>>>(pc, shift);
  }
  else patch_invert_kernel<<<pc.n_patches, kPatchMax * kPinvSplit, 0, v.stream>>>(pc.pp, pc.pidx, pc.pturn, pc.Pm, shift, pc.Pinv, pc.h1, pc.sw);
  QS_LAUNCH(v);
  if (pc.big) patch_apply_kernel<false, 1><<<pc.n_patches, patch_threads(pc), 0, v.stream>>>(pc.pp, pc.pidx, pc.pturn, pc.Pinv, it, v.sc);
  else patch_apply_kernel<false, kPinvSplit><<<pc.n_patches, patch_threads(pc), 0, v.stream>>>(pc.pp, pc.pidx, pc.pturn, pc.Pinv, it, v.sc);
  if (pc.nc > 0) {
    QS_LAUNCH(v);
    coarse_apply_kernel<false><<<v.n_turns, kPatchMax * kPinvSplit, 0, v.stream>>>(pc, it.tw, v.sc);
  }
  QS_LAUNCH(v);
  patch_project_kernel<true><<<grid_for(v.N), kBlock, 0, v.stream>>>(v.N, it, v.turn_id, pc.h1, v.sc);
  QS_LAUNCH(v);
  turn_book_kernel<<<(v.n_turns + kBlock - 1) / kBlock, kBlock, 0, v.stream>>>(v.n_turns, it.tw, it.sw, it.vsum);
}
void k_cg_project(const VecCtx& v, const CgIter& it) {
  QS_LAUNCH(v);
  if (it.patch.pp > 0) {
    patch_project_kernel<false><<<grid_for(v.N), kBlock, 0, v.stream>>>(v.N, it, v.turn_id, it.patch.h1, v.sc);
    return;
  }
  if (it.Lblk) {   // block-Jacobi preconditioner (unconstrained solves): g = B^-1 r, rg[par^1] += r.g
    launch_blockprec_apply(it.nb, v.N, it.Lblk, it.r, it.g, &v.sc->rg[it.par ^ 1], &v.sc->done, v.stream);
    return;
  }
  cg_project_kernel<<<grid_for(v.N), kBlock, 0, v.stream>>>(v.N, it, v.n_turns ? v.turn_id : nullptr, v.sc);
}
void k_cg_direction(const VecCtx& v, const CgIter& it) {
  QS_LAUNCH(v);
  cg_direction_kernel<<<grid_for(v.Np), kBlock, 0, v.stream>>>(v.N, v.Np, v.n_turns, it, v.sc);
}
void k_step_begin(const VecCtx& v, const StepBegin& a) {
  QS_LAUNCH(v);
  const size_t most = a.acc_words > static_cast<size_t>(a.N) ? a.acc_words : static_cast<size_t>(a.N);
  step_begin_kernel<<<grid_for(static_cast<int>(most < (1u << 30) ? most : (1u << 30))), kBlock, 0, v.stream>>>(a, v.sc);
}
void k_turn_fix(const VecCtx& v, double d, const double* Hd, const double* sw, double* x) {
  if (!v.n_turns) return;
  QS_LAUNCH(v);
  turn_fix_kernel<<<v.n_turns, turn_block(v), 0, v.stream>>>(v.turn_ptr, v.turn_idx, v.share, d, Hd, sw, x);
}
void k_turn_start(const VecCtx& v, const TurnStart& a) {
  QS_LAUNCH(v);
  turn_start_kernel<<<v.n_turns, turn_block(v), 0, v.stream>>>(a, v.sc);
}
void k_step_update(const VecCtx& v, double dt, const double* x, const double* area, double* J, const double* vsum) {
  QS_LAUNCH(v);
  step_update_kernel<<<grid_for(v.N), kBlock, 0, v.stream>>>(v.N, dt, x, area, J, v.n_turns, v.share, vsum, v.sc);
}
void k_axpy(const VecCtx& v, double a, const double* x, double* y) {
  QS_LAUNCH(v);
  axpy_kernel<<<grid_for(v.N), kBlock, 0, v.stream>>>(v.N, a, x, y);
}
void k_lincomb(const VecCtx& v, double a, const double* x, double b, double* y) {
  QS_LAUNCH(v);
  lincomb_kernel<<<grid_for(v.N), kBlock, 0, v.stream>>>(v.N, a, x, b, y);
}
void k_max_scaled_diff(const VecCtx& v, double s, const double* x1, const double* x2, const double* d) {
  QS_LAUNCH(v);
  max_scaled_diff_kernel<<<grid_for(v.N), kBlock, 0, v.stream>>>(v.N, s, x1, x2, d, v.sc);
}
void k_scale_div(const VecCtx& v, double a, const double* x, const double* d, double* y) {
  QS_LAUNCH(v);
  scale_div_kernel<<<grid_for(v.N), kBlock, 0, v.stream>>>(v.N, a, x, d, y);
}
void k_mul(const VecCtx& v, const double* a, const double* b, double* y) {
  QS_LAUNCH(v);
  mul_kernel<<<grid_for(v.N), kBlock, 0, v.stream>>>(v.N, a, b, y);
}
void k_set_scalars(const VecCtx& v) {
  QS_LAUNCH(v);
  set_scalars_kernel<<<1, 1, 0, v.stream>>>(v.sc);
}
void k_copy_rg_to_nu2(const VecCtx& v, int par) {
  QS_LAUNCH(v);
  copy_rg_to_nu2_kernel<<<1, 1, 0, v.stream>>>(par, v.sc);
}
void k_nu_residual(const VecCtx& v, double I_ramp, const double* Mxp1, const double* shift, const double* xp1,
                   const Rhs& b, double* r) {
  QS_LAUNCH(v);
  nu_residual_kernel<<<grid_for(v.N), kBlock, 0, v.stream>>>(v.N, I_ramp, Mxp1, shift, xp1, b, r);
}
void k_field_scale(const VecCtx& v, const double* bracc, const double* bzacc, const double* r, const double* selfcoef,
                   const double* cur, double* Br, double* Bz) {
  QS_LAUNCH(v);
  field_scale_kernel<<<grid_for(v.N), kBlock, 0, v.stream>>>(v.N, bracc, bzacc, r, selfcoef, cur, Br, Bz);
}
void k_sum_uterm(const VecCtx& v, const double* vsum) {
  if (!v.n_turns) return;
  QS_LAUNCH(v);
  sum_uterm_kernel<<<1, kBlock, 0, v.stream>>>(v.n_turns, v.share, vsum, v.sc);
}
void k_gather(const VecCtx& v, const double* src, const int* perm, double* dst, int n, int npad) {
  QS_LAUNCH(v);
  gather_kernel<<<grid_for(npad), kBlock, 0, v.stream>>>(n, npad, src, perm, dst);
}
void k_scatter_scaled(const VecCtx& v, const double* src, const int* perm, double* dst, int n, double scale) {
  QS_LAUNCH(v);
  scatter_scaled_kernel<<<grid_for(n), kBlock, 0, v.stream>>>(n, src, perm, dst, scale);
}

}  // namespace qs
