// qs_operator.cu — the all-pairs ring operator sweeps K1 (y = M x) and K2 (y = M x fused with Br, Bz = G_B I).
//
// Decomposition (B200-first, not the paper's): rings are grouped in blocks of 32 (one per lane).  The
// symmetric kernel is evaluated ONCE per unordered pair: a work item is a pair of ring blocks
// (bi <= bj); lane l owns target i = 32 bi + l and walks the 32 sources of block bj in a rotated order
// j = 32 bj + ((l + s) & 31), s = 0..31.  The contribution to y_i stays in a register; the
// contribution to y_j rides in a register that is passed to the neighbouring lane after every step
// (one 64-bit shuffle), so that after 32 steps lane l holds the finished partial sum for source
// 32 bj + l.  Partial sums go to FP64 accumulators in L2 with RED.ADD.F64 (256-byte coalesced).
// Source blocks (r, z, x[, I]: 3-4 x 256 B) are staged in per-warp shared memory with TMA bulk copies
// (cp.async.bulk + mbarrier), double buffered one item ahead.  Items are handed out in contiguous
// chunks from an atomic counter to a persistent grid (a multiple of the SM count).
// The evaluation class (AGM depth + series order, qs_pair.cuh) is chosen per item from the bounding boxes of the two
// blocks (a lower bound on k'^2 over the 1024 pairs), so the 32-step loops are branch-free and fully unrolled in the
// depth; items whose two blocks each sit on one radius (rows of a lattice) take a variant with the radial terms hoisted.
// What bounds the kernel is the issue port (an FP64 instruction holds it for two cycles), so the loops
// are written for instruction count: source arrays staged twice (no index wrap), unroll 2, no divisions, no roots.
#include "qs_internal.h"
#include "qs_pair.cuh"
#include "qs_tma.cuh"

namespace qs {

// Evaluation classes, cheapest first: (AGM iterations NIT, series order HI) and the smallest k'^2 = B2/A2 for which
// the truncated evaluation is exact to < 1e-16 relative in M, K and E (60-digit evaluation of the truncated
// recurrence against K, E, plus 2 % margin).  FP64 operations per pair:
// 8 + 10 NIT + 16 (lo) or 20 (hi).
constexpr int kNumClasses = 10;
__device__ __constant__ double kClassKp2Min[kNumClasses] = {0.3965,   0.1394,   0.01529,   1.374e-3, 1.453e-5,
                                                            1.157e-7, 1.293e-11, 8.2e-16,  1.03e-23, 0.0};
//                                                class:      0       1       2       3       4       5       6       7       8       9
//                                                (NIT,HI): (2,lo)  (2,hi)  (3,lo)  (3,hi)  (4,lo)  (4,hi)  (5,lo)  (5,hi)  (6,lo)  (7,lo)

#ifndef QS_SW_WARPS
#define QS_SW_WARPS 4          // warps per CTA of the pair sweeps (small CTAs: finer register-budget steps)
#endif
#ifndef QS_SW_MINB_FIELD
#define QS_SW_MINB_FIELD 5     // resident CTAs per SM the register budget of the fused sweep is sized for: 20 warps
                               // at <= 102 registers (96 used).  Measured on config 2: 8x2 (112 regs) 108.8 ms,
                               // 4x5 102.7 ms, 8x3 (80 regs) 103.9 ms, 4x6 (80 regs) 104.2 ms
#endif
#ifndef QS_SW_MINB_M
#define QS_SW_MINB_M 7         // the same for the M-only sweep: 28 warps at 72 registers.  N = 262,144: 4x6 / 8x3
                               // (80 regs) 113.1 ms, 4x7 112.1 ms, 8x4 (64 regs) 114.8 ms, 4x5 (96 regs) 117.4 ms
#endif
#ifndef QS_SW_UNROLL
#define QS_SW_UNROLL 2         // source steps unrolled in the off-diagonal item loop (1: +3 %, 4: +17 % on K2)
#endif
constexpr int kSweepUnroll = QS_SW_UNROLL;
constexpr int kWarpsPerCta = QS_SW_WARPS;
constexpr int kThreads = kWarpsPerCta * 32;
constexpr int kMaxArrays = 4;

__device__ __forceinline__ void red_add(double* addr, double v) {
  asm volatile("red.global.add.f64 [%0], %1;" ::"l"(addr), "d"(v) : "memory");
}

struct TargetRegs {
  double r, z, x, cur;
};
struct Accum {
  double y, br, bz;
};

// ---- one off-diagonal item: all 32 x 32 pairs, both directions -----------------------------------
// UNI: every ring of the source block has the same radius rju and so has the target block (blocks of a lattice row,
// the common case on winding packs whose Nz is a multiple of 32): (ri - rj)^2, 4 ri rj and rj^2 - ri^2 are item
// constants, the source radii are not read.
template <int NIT, bool HI, bool FIELD, bool UNI>
__device__ __forceinline__ void item_offdiag(const TargetRegs& t, const double* __restrict__ sr,
                                             const double* __restrict__ sz, const double* __restrict__ sx,
                                             const double* __restrict__ sc, double soft_all, double rju, int lane,
                                             Accum& acc, Accum& trav) {
  const unsigned full = 0xffffffffu;
  const int next = (lane + 1) & 31;
  const double ri2 = t.r * t.r, ri4 = 4.0 * t.r;
  const double difu = t.r - rju, dif2u = difu * difu, c4u = ri4 * rju, eu = fma(rju, rju, -ri2);
  const double dif2s = dif2u + soft_all;
  sr += lane, sz += lane, sx += lane, sc += lane;   // arrays are stored twice: entry lane + s = source (lane + s) & 31
#pragma unroll kSweepUnroll
  for (int s = 0; s < 32; ++s) {
    const int jl = s;
    const double zj = sz[jl], xj = sx[jl];
    const double dz = t.z - zj;
    double dz2 = 0.0, A2, B2, rj = rju;
    if (UNI) {
      if (FIELD) {
        dz2 = fma(dz, dz, soft_all);
        B2 = dz2 + dif2u;
      } else {
        B2 = fma(dz, dz, dif2s);
      }
      A2 = B2 + c4u;
    } else {
      rj = sr[jl];
      dz2 = fma(dz, dz, soft_all);
      const double dif = t.r - rj;
      B2 = fma(dif, dif, dz2);
      A2 = fma(ri4, rj, B2);                               // (ri+rj)^2 = (ri-rj)^2 + 4 ri rj
    }
    const PairAGM a = agm_pair<NIT, HI, FIELD>(A2, B2);
    const double mt = a.S * a.yinf;
    acc.y = fma(mt, xj, acc.y);
    trav.y = fma(mt, t.x, trav.y);
    if (FIELD) {
      const double cj = sc[jl];
      const double qt = a.yinf * (a.mid - a.S) * a.y0sq;
      const double e = UNI ? eu : fma(rj, rj, -ri2);       // rj^2 - ri^2
      const double bz_ij = fma(e - dz2, qt, a.yinf);       // Kt + (rj^2 - ri^2 - dz^2) Qt
      const double bz_ji = fma(-e - dz2, qt, a.yinf);
      const double ur = dz * fma(a.mid, qt, -a.yinf);      // dz (-Kt + (ri^2 + rj^2 + dz^2) Qt)
      acc.bz = fma(bz_ij, cj, acc.bz);
      acc.br = fma(ur, cj, acc.br);
      trav.bz = fma(bz_ji, t.cur, trav.bz);
      trav.br = fma(-ur, t.cur, trav.br);
      trav.bz = __shfl_sync(full, trav.bz, next);
      trav.br = __shfl_sync(full, trav.br, next);
    }
    trav.y = __shfl_sync(full, trav.y, next);
  }
}

// ---- one diagonal item (bi == bj): every ordered pair appears once in the rotation -----------------
template <int NIT, bool HI, bool FIELD>
__device__ __forceinline__ void item_diag(const TargetRegs& t, const double* __restrict__ sr,
                                          const double* __restrict__ sz, const double* __restrict__ sx,
                                          const double* __restrict__ sc, double soft_all, double soft_self, int lane,
                                          Accum& acc) {
  const double ri2 = t.r * t.r;
  {  // s = 0: the self pair; M_ii = M(ri, ri, dz^2 = soft_all + soft_self); no field term (C3 self field is analytic)
    const double dz2 = soft_all + soft_self;
    const double sum = t.r + t.r;
    const PairAGM a = agm_pair<NIT, HI, false>(fma(sum, sum, dz2), dz2);
    acc.y = fma(a.S * a.yinf, t.x, acc.y);
  }
  sr += lane, sz += lane, sx += lane, sc += lane;
#pragma unroll 1
  for (int s = 1; s < 32; ++s) {
    const int jl = s;
    const double rj = sr[jl], zj = sz[jl], xj = sx[jl];
    const double dz = t.z - zj;
    const double dz2 = fma(dz, dz, soft_all);
    const double sum = t.r + rj, dif = t.r - rj;
    const PairAGM a = agm_pair<NIT, HI, FIELD>(fma(sum, sum, dz2), fma(dif, dif, dz2));
    acc.y = fma(a.S * a.yinf, xj, acc.y);
    if (FIELD) {
      const double cj = sc[jl];
      const double qt = a.yinf * (a.mid - a.S) * a.y0sq;
      const double e = fma(rj, rj, -ri2);
      acc.bz = fma(fma(e - dz2, qt, a.yinf), cj, acc.bz);
      acc.br = fma(dz * fma(a.mid, qt, -a.yinf), cj, acc.br);
    }
  }
}

__device__ __forceinline__ int classify(const double4& bi, const double4& bj, bool diag, const SweepParams& prm) {
  // double4 = (rmin, rmax, zmin, zmax) of the ring centres of a block
  const double dr = fmax(0.0, fmax(bi.x - bj.y, bj.x - bi.y));
  const double dzg = fmax(0.0, fmax(bi.z - bj.w, bj.z - bi.w));
  const double smax = bi.y + bj.y;
  const double d2 = diag ? prm.diag_d2 : fmax(fma(dr, dr, dzg * dzg), prm.minsep2) + prm.soft_all;
  const double kp2 = d2 / (fma(smax, smax, d2));
  int cls = kNumClasses - 1;
#pragma unroll
  for (int k = kNumClasses - 2; k >= 0; --k)
    if (kp2 >= kClassKp2Min[k]) cls = k;
  return cls;
}

// row-major enumeration of the upper triangle (bi <= bj) of an nb x nb block matrix
__device__ __forceinline__ void unrank(long long k, int nb, int& bi, int& bj) {
  const double t = 2.0 * nb + 1.0;
  int i = static_cast<int>(floor(0.5 * (t - sqrt(t * t - 8.0 * static_cast<double>(k)))));
  i = max(0, min(i, nb - 1));
  auto row_start = [nb](int r) { return static_cast<long long>(r) * nb - static_cast<long long>(r) * (r - 1) / 2; };
  while (i > 0 && row_start(i) > k) --i;
  while (i + 1 < nb && row_start(i + 1) <= k) ++i;
  bi = i;
  bj = i + static_cast<int>(k - row_start(i));
}

template <bool FIELD>
__global__ void __launch_bounds__(kThreads, FIELD ? QS_SW_MINB_FIELD : QS_SW_MINB_M) sweep_kernel(SweepParams prm) {
  constexpr int NA = FIELD ? 4 : 3;
  __shared__ __align__(128) double sbuf[kWarpsPerCta][2][kMaxArrays][64];   // every array twice: no wrap of lane + s
  __shared__ __align__(8) uint64_t sbar[kWarpsPerCta][2];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const unsigned full = 0xffffffffu;
  if (prm.done != nullptr && *prm.done != 0) return;   // a converged CG batch: nothing left to do
  if (threadIdx.x < kWarpsPerCta * 2) mbar_init(&sbar[threadIdx.x >> 1][threadIdx.x & 1], 1);
  asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  __syncthreads();

  uint32_t phase = 0u;   // bit b = parity to wait for on buffer b
  const double* src[kMaxArrays] = {prm.r, prm.z, prm.x, prm.cur};

  auto issue = [&](int buf, int bj) {
    if (lane == 0) {
      mbar_expect_tx(&sbar[warp][buf], NA * 512u);
#pragma unroll
      for (int a = 0; a < NA; ++a) {
        bulk_g2s(&sbuf[warp][buf][a][0], src[a] + 32ll * bj, 256u, &sbar[warp][buf]);
        bulk_g2s(&sbuf[warp][buf][a][32], src[a] + 32ll * bj, 256u, &sbar[warp][buf]);
      }
    }
  };

  for (;;) {
    long long k0 = 0;
    if (lane == 0) k0 = static_cast<long long>(atomicAdd(prm.counter, static_cast<unsigned long long>(prm.chunk)));
    k0 = __shfl_sync(full, k0, 0);
    if (k0 >= prm.n_items) break;
    const int cnt = static_cast<int>(min(static_cast<long long>(prm.chunk), prm.n_items - k0));
    int bi, bj;
    unrank(k0, prm.nb, bi, bj);
    issue(0, bj);

    TargetRegs t;
    Accum acc = {0.0, 0.0, 0.0};
    double4 bbi;
    int cur_bi = -1;
    for (int it = 0; it < cnt; ++it) {
      const int buf = it & 1;
      if (bi != cur_bi) {  // new target block: flush the old accumulators, load the new targets
        if (cur_bi >= 0) {
          red_add(prm.yacc + 32ll * cur_bi + lane, acc.y);
          if (FIELD) {
            red_add(prm.bracc + 32ll * cur_bi + lane, acc.br);
            red_add(prm.bzacc + 32ll * cur_bi + lane, acc.bz);
          }
        }
        acc = {0.0, 0.0, 0.0};
        cur_bi = bi;
        const long long i = 32ll * bi + lane;
        t.r = prm.r[i];
        t.z = prm.z[i];
        t.x = prm.x[i];
        t.cur = FIELD ? prm.cur[i] : 0.0;
        bbi = prm.bbox[bi];
      }
      // next item of this chunk (row-major walk), prefetched into the other buffer
      int nbi = bi, nbj = bj + 1;
      if (nbj == prm.nb) {
        nbi = bi + 1;
        nbj = nbi;
      }
      if (it + 1 < cnt) issue(buf ^ 1, nbj);

      const double4 bbj = prm.bbox[bj];
      const bool uni = bbi.x == bbi.y && bbj.x == bbj.y;   // both blocks on one radius each (lattice rows)
      const int nit = classify(bbi, bbj, bi == bj, prm);
      mbar_wait(&sbar[warp][buf], (phase >> buf) & 1u);
      phase ^= 1u << buf;
      const double* sr = sbuf[warp][buf][0];
      const double* sz = sbuf[warp][buf][1];
      const double* sx = sbuf[warp][buf][2];
      const double* sc = sbuf[warp][buf][3];
      if (bi == bj) {
#define QS_DIAG(N_, HI_) item_diag<N_, HI_, FIELD>(t, sr, sz, sx, sc, prm.soft_all, prm.soft_self, lane, acc); break
        switch (nit) {   // diagonal items are rare: the four cheapest classes share (4, lo)
          case 0: case 1: case 2: case 3: case 4: QS_DIAG(4, false);
          case 5: QS_DIAG(4, true);
          case 6: QS_DIAG(5, false);
          case 7: QS_DIAG(5, true);
          case 8: QS_DIAG(6, false);
          default: QS_DIAG(7, false);
        }
#undef QS_DIAG
      } else {
        Accum trav = {0.0, 0.0, 0.0};
#define QS_OFF(N_, HI_)                                                                              \
  if (uni)                                                                                           \
    item_offdiag<N_, HI_, FIELD, true>(t, sr, sz, sx, sc, prm.soft_all, bbj.x, lane, acc, trav);     \
  else                                                                                               \
    item_offdiag<N_, HI_, FIELD, false>(t, sr, sz, sx, sc, prm.soft_all, 0.0, lane, acc, trav);      \
  break
        switch (nit) {
          case 0: QS_OFF(2, false);
          case 1: QS_OFF(2, true);
          case 2: QS_OFF(3, false);
          case 3: QS_OFF(3, true);
          case 4: QS_OFF(4, false);
          case 5: QS_OFF(4, true);
          case 6: QS_OFF(5, false);
          case 7: QS_OFF(5, true);
          case 8: QS_OFF(6, false);
          default: QS_OFF(7, false);
        }
#undef QS_OFF
        red_add(prm.yacc + 32ll * bj + lane, trav.y);
        if (FIELD) {
          red_add(prm.bracc + 32ll * bj + lane, trav.br);
          red_add(prm.bzacc + 32ll * bj + lane, trav.bz);
        }
      }
      __syncwarp();  // every lane is done reading sbuf[buf] before it is refilled two items later
      bi = nbi;
      bj = nbj;
    }
    red_add(prm.yacc + 32ll * cur_bi + lane, acc.y);
    if (FIELD) {
      red_add(prm.bracc + 32ll * cur_bi + lane, acc.br);
      red_add(prm.bzacc + 32ll * cur_bi + lane, acc.bz);
    }
  }
}

__global__ void diag_kernel(int n, const double* __restrict__ r, double d2self, double* __restrict__ diagM) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const double s = r[i] + r[i];
  const PairAGM a = agm_pair<7, false, false>(fma(s, s, d2self), d2self);
  diagM[i] = (0.5 * kMu0 * kPi) * a.S * a.yinf;
}
// ---- test hook: one pair per thread through a chosen evaluation class (cls < 0: chosen from k'^2 like the sweep) ----
template <int NIT, bool HI>
__device__ __forceinline__ void pair_out(double A2, double B2, double* M, double* K, double* E) {
  const PairAGM a = agm_pair<NIT, HI, true>(A2, B2);
  *M = (0.5 * kMu0 * kPi) * a.S * a.yinf;
  const double sa = sqrt(A2);
  *K = (0.5 * kPi) * a.yinf * sa;
  *E = (0.5 * kPi) * a.yinf * (a.mid - a.S) / sa;
}
__global__ void pair_eval_kernel(int n, const double* __restrict__ A2, const double* __restrict__ B2, int cls,
                                 double* __restrict__ M, double* __restrict__ K, double* __restrict__ E,
                                 int* __restrict__ used) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  int c = cls;
  if (c < 0) {
    const double kp2 = B2[i] / A2[i];
    c = kNumClasses - 1;
    for (int k = kNumClasses - 2; k >= 0; --k)
      if (kp2 >= kClassKp2Min[k]) c = k;
  }
  used[i] = c;
  switch (c) {
    case 0: pair_out<2, false>(A2[i], B2[i], M + i, K + i, E + i); break;
    case 1: pair_out<2, true>(A2[i], B2[i], M + i, K + i, E + i); break;
    case 2: pair_out<3, false>(A2[i], B2[i], M + i, K + i, E + i); break;
    case 3: pair_out<3, true>(A2[i], B2[i], M + i, K + i, E + i); break;
    case 4: pair_out<4, false>(A2[i], B2[i], M + i, K + i, E + i); break;
    case 5: pair_out<4, true>(A2[i], B2[i], M + i, K + i, E + i); break;
    case 6: pair_out<5, false>(A2[i], B2[i], M + i, K + i, E + i); break;
    case 7: pair_out<5, true>(A2[i], B2[i], M + i, K + i, E + i); break;
    case 8: pair_out<6, false>(A2[i], B2[i], M + i, K + i, E + i); break;
    default: pair_out<7, false>(A2[i], B2[i], M + i, K + i, E + i); break;
  }
}
cudaError_t launch_pair_eval(int n, const double* A2, const double* B2, int cls, double* M, double* K, double* E,
                             int* used, cudaStream_t stream) {
  pair_eval_kernel<<<(n + 127) / 128, 128, 0, stream>>>(n, A2, B2, cls, M, K, E, used);
  return cudaGetLastError();
}
int pair_num_classes() { return kNumClasses; }

// ---- block-Jacobi preconditioner of the unconstrained solve (free rings, config 4): the 32 x 32 diagonal blocks of M
// (the sweep's diagonal items, same pair arithmetic) are Cholesky-factored once, one warp per block; applying
// B^-1 = blockdiag(L L^T)^-1 is a forward and a backward substitution per block.  On the Morton-ordered random rings
// the near pairs that make M ill-conditioned (cond ~ 1e7) mostly fall inside a block: 7.4e3 -> 5.8e2 CG iterations
// at N = 4096.
constexpr int kBpWarps = 4;
__global__ void __launch_bounds__(kBpWarps * 32) blockprec_build_kernel(int nb, const double* __restrict__ r,
                                                                        const double* __restrict__ z, double soft_all,
                                                                        double soft_self, double* __restrict__ L) {
  __shared__ double A[kBpWarps][32][33];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int b = blockIdx.x * kBpWarps + warp;
  if (b >= nb) return;
  double(*At)[33] = A[warp];
  const double ri = r[32 * b + lane], zi = z[32 * b + lane];
  for (int j = 0; j < 32; ++j) {
    const double rj = r[32 * b + j], zj = z[32 * b + j];
    const double dz = zi - zj;
    const double dz2 = fma(dz, dz, soft_all) + (j == lane ? soft_self : 0.0);
    const double dif = ri - rj;
    const double B2 = fma(dif, dif, dz2), A2 = fma(4.0 * ri, rj, B2);
    const PairAGM a = agm_pair<7, false, false>(A2, B2);
    At[lane][j] = (0.5 * kMu0 * kPi) * a.S * a.yinf;
  }
  __syncwarp();
  for (int k = 0; k < 32; ++k) {                     // right-looking Cholesky, lane = row
    if (lane == k) At[k][k] = sqrt(At[k][k]);
    __syncwarp();
    if (lane > k) At[lane][k] /= At[k][k];
    __syncwarp();
    if (lane > k)
      for (int j = k + 1; j <= lane; ++j) At[lane][j] -= At[lane][k] * At[j][k];
    __syncwarp();
  }
  double* Lb = L + static_cast<size_t>(b) * 1024;
  for (int i = 0; i < 32; ++i) Lb[i * 32 + lane] = lane <= i ? (lane == i ? 1.0 / At[i][i] : At[i][lane]) : 0.0;
}

// g = B^-1 r (blocks of 32), rg += r.g ; the diagonal of the stored factor holds 1 / L_ii
__global__ void __launch_bounds__(kBpWarps * 32) blockprec_apply_kernel(int nb, int n, const double* __restrict__ L,
                                                                        const double* __restrict__ rvec,
                                                                        double* __restrict__ g, double* rg_out,
                                                                        const int* done) {
  __shared__ double A[kBpWarps][32][33];
  if (done != nullptr && *done != 0) return;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int b = blockIdx.x * kBpWarps + warp;
  double dot = 0.0;
  if (b < nb) {
    double(*At)[33] = A[warp];
    const double* Lb = L + static_cast<size_t>(b) * 1024;
    for (int i = 0; i < 32; ++i) At[i][lane] = Lb[i * 32 + lane];
    __syncwarp();
    const int idx = 32 * b + lane;
    const double ri = idx < n ? rvec[idx] : 0.0;
    double acc = ri, y = 0.0;
    for (int k = 0; k < 32; ++k) {                   // L y = r
      const double yk = __shfl_sync(0xffffffffu, acc * At[k][k], k);   // lane k's value is the finished one
      if (lane == k) y = yk;
      if (lane > k) acc = fma(-At[lane][k], yk, acc);
    }
    acc = y;
    double x = 0.0;
    for (int k = 31; k >= 0; --k) {                  // L^T x = y
      const double xk = __shfl_sync(0xffffffffu, acc * At[k][k], k);
      if (lane == k) x = xk;
      if (lane < k) acc = fma(-At[k][lane], xk, acc);
    }
    if (idx < n) g[idx] = x;
    dot = ri * x;
  }
  dot = [&] {
    double v = dot;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
  }();
  if (lane == 0 && dot != 0.0) atomicAdd(rg_out, dot);
}

cudaError_t launch_blockprec_build(int nb, const double* r, const double* z, double soft_all, double soft_self, double* L,
                                   cudaStream_t stream) {
  blockprec_build_kernel<<<(nb + kBpWarps - 1) / kBpWarps, kBpWarps * 32, 0, stream>>>(nb, r, z, soft_all, soft_self, L);
  return cudaGetLastError();
}
cudaError_t launch_blockprec_apply(int nb, int n, const double* L, const double* rvec, double* g, double* rg_out,
                                   const int* done, cudaStream_t stream) {
  blockprec_apply_kernel<<<(nb + kBpWarps - 1) / kBpWarps, kBpWarps * 32, 0, stream>>>(nb, n, L, rvec, g, rg_out, done);
  return cudaGetLastError();
}

cudaError_t launch_diag(int n, const double* r, double d2self, double* diagM, cudaStream_t stream) {
  diag_kernel<<<(n + 255) / 256, 256, 0, stream>>>(n, r, d2self, diagM);
  return cudaGetLastError();
}

// ---- FP64 FMA roofline probe: 16 independent chains per thread, 1024 threads x 2 CTAs per SM ----------------
__global__ void __launch_bounds__(512) dfma_probe_kernel(int iters, double seed, double* sink, long long* cycles) {
  double a[16];
#pragma unroll
  for (int k = 0; k < 16; ++k) a[k] = seed + 1e-3 * (threadIdx.x + k);
  const double m = 1.0 - 1e-9 * seed, c = 1e-9;
  const long long t0 = clock64();
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int k = 0; k < 16; ++k) a[k] = fma(a[k], m, c);
  }
  const long long t1 = clock64();
  double s = 0.0;
#pragma unroll
  for (int k = 0; k < 16; ++k) s += a[k];
  if (s == 123.456) sink[0] = s;   // keeps the chains alive
  if (threadIdx.x == 0 && blockIdx.x == 0) cycles[0] = t1 - t0;
}

cudaError_t fp64_peak_probe(double* tflops, double* sm_mhz) {
  int dev = 0, sms = 0;
  cudaError_t e;
  if ((e = cudaGetDevice(&dev)) != cudaSuccess) return e;
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  double* sink = nullptr;
  long long* cyc = nullptr;
  if ((e = cudaMalloc(&sink, 64)) != cudaSuccess) return e;
  cyc = reinterpret_cast<long long*>(sink + 1);
  cudaEvent_t a, b;
  cudaEventCreate(&a);
  cudaEventCreate(&b);
  const int iters = 20000, grid = sms * 4, threads = 512;
  double best_ms = 1e300, best_mhz = 0.0;
  for (int rep = 0; rep < 6; ++rep) {
    cudaEventRecord(a, 0);
    dfma_probe_kernel<<<grid, threads>>>(iters, 1.0 + rep, sink, cyc);
    cudaEventRecord(b, 0);
    if ((e = cudaEventSynchronize(b)) != cudaSuccess) break;
    float ms = 0.f;
    cudaEventElapsedTime(&ms, a, b);
    long long hc = 0;
    cudaMemcpy(&hc, cyc, sizeof(hc), cudaMemcpyDeviceToHost);
    if (rep > 0 && ms < best_ms) {   // rep 0 warms up
      best_ms = ms;
      best_mhz = static_cast<double>(hc) / (ms * 1e-3) / 1e6;
    }
  }
  if (e == cudaSuccess) e = cudaGetLastError();
  cudaEventDestroy(a);
  cudaEventDestroy(b);
  cudaFree(sink);
  if (e != cudaSuccess) return e;
  *tflops = 2.0 * 16.0 * iters * static_cast<double>(grid) * threads / (best_ms * 1e-3) / 1e12;
  *sm_mhz = best_mhz;
  return cudaSuccess;
}

// Issue-model probes behind DESIGN.md §6 (what bounds the sweeps): 8 independent DFMA chains per thread with
//   mode 1: three distinct register operands per DFMA            (register-file read port: 3 cycles per warp-instr)
//   mode 2: two register operands + immediate                     (2 cycles per warp-instr: the pipe rate)
//   mode 3: mode 2 plus 8 integer ALU instructions per 8 DFMAs    (an FP64 instruction holds the issue port: the
//                                                                   integer work does not co-issue for free)
template <int MODE>
__global__ void __launch_bounds__(256) issue_probe_kernel(int iters, const double* __restrict__ in, double* __restrict__ out,
                                                          int sh) {
  double a[8], b[8], c[8];
  int q[4] = {static_cast<int>(threadIdx.x), static_cast<int>(threadIdx.x) * 3, static_cast<int>(threadIdx.x) * 5,
              static_cast<int>(threadIdx.x) * 7};
#pragma unroll
  for (int i = 0; i < 8; ++i) {
    a[i] = in[threadIdx.x + 32 * i];
    b[i] = in[threadIdx.x + 32 * i + 1000];
    c[i] = in[threadIdx.x + 32 * i + 2000];
  }
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int i = 0; i < 8; ++i) a[i] = MODE == 1 ? fma(a[i], b[i], c[i]) : fma(a[i], b[i], 0.5);
    if (MODE == 3) {
#pragma unroll
      for (int j = 0; j < 4; ++j) q[j] = (q[j] + sh) ^ it;
    }
  }
  double s = q[0] + q[1] + q[2] + q[3];
#pragma unroll
  for (int i = 0; i < 8; ++i) s += a[i] + b[i] + c[i];
  out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

cudaError_t issue_probe(int mode, double* cycles_per_dfma) {
  int dev = 0, sms = 0, khz = 0;
  cudaError_t e;
  if ((e = cudaGetDevice(&dev)) != cudaSuccess) return e;
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  cudaDeviceGetAttribute(&khz, cudaDevAttrClockRate, dev);
  const int iters = 20000, grid = sms * 4, threads = 256;
  double* buf = nullptr;
  if ((e = cudaMalloc(&buf, sizeof(double) * (4096 + static_cast<size_t>(grid) * threads))) != cudaSuccess) return e;
  cudaMemset(buf, 0, sizeof(double) * 4096);
  cudaEvent_t a, b;
  cudaEventCreate(&a);
  cudaEventCreate(&b);
  float best = 1e30f;
  for (int rep = 0; rep < 4 && e == cudaSuccess; ++rep) {
    cudaEventRecord(a, 0);
    if (mode == 1) issue_probe_kernel<1><<<grid, threads>>>(iters, buf, buf + 4096, 3);
    else if (mode == 2) issue_probe_kernel<2><<<grid, threads>>>(iters, buf, buf + 4096, 3);
    else issue_probe_kernel<3><<<grid, threads>>>(iters, buf, buf + 4096, 3);
    cudaEventRecord(b, 0);
    e = cudaEventSynchronize(b);
    float ms = 0.f;
    cudaEventElapsedTime(&ms, a, b);
    if (rep > 0 && ms < best) best = ms;
  }
  if (e == cudaSuccess) e = cudaGetLastError();
  cudaEventDestroy(a);
  cudaEventDestroy(b);
  cudaFree(buf);
  if (e != cudaSuccess) return e;
  // cycles per DFMA warp-instruction per SM sub-partition at the maximum SM clock: 8 warps x 8 DFMA x iters per SMSP... per CTA
  const double warp_instr_per_smsp = static_cast<double>(iters) * 8.0 * (static_cast<double>(grid) * threads / 32.0) / (sms * 4.0);
  *cycles_per_dfma = best * 1e-3 * (khz * 1e3) / warp_instr_per_smsp;
  return cudaSuccess;
}

int sweep_grid(int sm_count, bool field) { return sm_count * (field ? QS_SW_MINB_FIELD : QS_SW_MINB_M); }

cudaError_t launch_sweep(const SweepParams& prm, bool field, int grid, cudaStream_t stream) {
  if (field)
    sweep_kernel<true><<<grid, kThreads, 0, stream>>>(prm);
  else
    sweep_kernel<false><<<grid, kThreads, 0, stream>>>(prm);
  return cudaGetLastError();
}

int sweep_warps_per_cta() { return kWarpsPerCta; }

}  // namespace qs
