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

// Evaluation classes, cheapest first: (AGM iterations NIT, series order ORD) and the smallest k'^2 = B2/A2 for which
// the truncated evaluation is exact to < 1e-16 relative in M, K and E (60-digit evaluation of the truncated
// recurrence against K, E, plus 2 % margin).  FP64 operations per pair (M only):
// 7 + 10 NIT + 11 + 2 ORD.  A finer ladder (orders 3, 5, 6 in between: 14 classes) saves ~1.2 operations per pair on
// the coil configs but lost on the clock (config 2 fused sweep 96.3 vs 94.8 ms, N = 262,144 matvec 131 vs 103 ms):
// more distinct loops are hot at the same time and the instruction caches thrash.
constexpr int kNumClasses = 10;
__device__ __constant__ double kClassKp2Min[kNumClasses] = {0.3965,   0.1394,   0.01529,   1.374e-3, 1.453e-5,
                                                            1.157e-7, 1.293e-11, 8.2e-16,  1.03e-23, 0.0};
//  class:        0      1      2      3      4      5      6      7      8      9
//  (NIT,ORD):  (2,2)  (2,4)  (3,2)  (3,4)  (4,2)  (4,4)  (5,2)  (5,4)  (6,2)  (7,2)
// QS_CLASS_SWITCH(cls, M) expands M(NIT, ORD) for the class
#define QS_CLASS_SWITCH(cls_, M_) \
  switch (cls_) {                 \
    case 0: M_(2, 2); break;      \
    case 1: M_(2, 4); break;      \
    case 2: M_(3, 2); break;      \
    case 3: M_(3, 4); break;      \
    case 4: M_(4, 2); break;      \
    case 5: M_(4, 4); break;      \
    case 6: M_(5, 2); break;      \
    case 7: M_(5, 4); break;      \
    case 8: M_(6, 2); break;      \
    default: M_(7, 2); break;     \
  }

#ifndef QS_SW_WARPS
#define QS_SW_WARPS 4          // warps per CTA of the pair sweeps (small CTAs: finer register-budget steps)
#endif
#ifndef QS_SW_MINB_FIELD
#define QS_SW_MINB_FIELD 5     // resident CTAs per SM the register budget of the fused sweep is sized for: 20 warps
                               // at <= 102 registers (96 used).  Measured on config 2 (T = target blocks per item):
                               // T=1: 104.6 ms; T=2 at 5 CTAs (96 regs) 98.5 ms, at 4 CTAs (128 regs) 99.6 ms;
                               // T=3 at 4 CTAs 100.7 ms; T=4 at 4 CTAs (128 regs, spills) 100.8 ms, at 3 CTAs (168 regs) 110.6 ms
#endif
#ifndef QS_SW_MINB_M
#define QS_SW_MINB_M 4         // the same for the M-only sweep: 16 warps at 128 registers.  N = 262,144: T=1 113.9 ms;
                               // T=2 at 7 CTAs (72 regs) 108.6 ms, at 6 CTAs 110.1 ms; T=3 at 5 CTAs 107.7 ms;
                               // T=4 at 5 CTAs (96 regs, spills) 107.7 ms, at 4 CTAs (128 regs) 105.0 ms
#endif
#ifndef QS_SW_MINB_M12
#define QS_SW_MINB_M12 7       // M-only sweep at T = 1, 2: 28 warps at 72 registers
#endif
#ifndef QS_SW_UNROLL
#define QS_SW_UNROLL 2         // source steps unrolled in the off-diagonal item loop (1: +3 %, 4: +17 % on K2)
#endif
constexpr int kSweepUnroll = QS_SW_UNROLL;
#ifndef QS_SW_NB_T2
#define QS_SW_NB_T2 1024       // blocks of 32 rings from which items hold T = 2 target blocks (both sweeps)
#endif
#ifndef QS_SW_NB_T4
#define QS_SW_NB_T4 4096       // ... and T = 4 (M-only sweep)
#endif
#ifndef QS_SW_MULTI_UNROLL
#define QS_SW_MULTI_UNROLL 1   // source steps unrolled in the multi-target loop (each step already holds T pair chains)
#endif
constexpr int kMultiUnroll = QS_SW_MULTI_UNROLL;
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
template <int NIT, int ORD, bool FIELD, bool UNI>
__device__ __forceinline__ void item_offdiag(const TargetRegs& t, const double* __restrict__ sr,
                                             const double* __restrict__ sz, const double* __restrict__ sx,
                                             const double* __restrict__ sc, double soft_all, double rju, int lane,
                                             Accum& acc, Accum& trav) {
  const unsigned full = 0xffffffffu;
  const int next = (lane + 1) & 31;
  const double ri2 = t.r * t.r, ri4 = 4.0 * t.r;
  const double difu = t.r - rju, dif2u = difu * difu, c4u = ri4 * rju, eu = fma(rju, rju, -ri2), sigu = fma(rju, rju, ri2);
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
    const PairAGM a = agm_pair<NIT, ORD, FIELD>(A2, B2);
    const double mt = a.S * a.yinf;
    acc.y = fma(mt, xj, acc.y);
    trav.y = fma(mt, t.x, trav.y);
    if (FIELD) {
      const double cj = sc[jl];
      const double qt = a.yinf * a.emS * a.y0sq;
      const double sig = UNI ? sigu : fma(rj, rj, ri2);    // ri^2 + rj^2
      const double e = UNI ? eu : fma(-2.0, ri2, sig);     // rj^2 - ri^2
      const double P = fma(-dz2, qt, a.yinf);              // Kt - dz^2 Qt
      const double R = e * qt;
      const double bz_ij = P + R;                          // Kt + (rj^2 - ri^2 - dz^2) Qt
      const double bz_ji = P - R;
      const double ur = dz * fma(sig, qt, -P);             // dz (-Kt + (ri^2 + rj^2 + dz^2) Qt)
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
template <int NIT, int ORD, bool FIELD>
__device__ __forceinline__ void item_diag(const TargetRegs& t, const double* __restrict__ sr,
                                          const double* __restrict__ sz, const double* __restrict__ sx,
                                          const double* __restrict__ sc, double soft_all, double soft_self, int lane,
                                          Accum& acc) {
  const double ri2 = t.r * t.r;
  {  // s = 0: the self pair; M_ii = M(ri, ri, dz^2 = soft_all + soft_self); no field term (C3 self field is analytic)
    const double dz2 = soft_all + soft_self;
    const double sum = t.r + t.r;
    const PairAGM a = agm_pair<NIT, ORD, false>(fma(sum, sum, dz2), dz2);
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
    const PairAGM a = agm_pair<NIT, ORD, FIELD>(fma(sum, sum, dz2), fma(dif, dif, dz2));
    acc.y = fma(a.S * a.yinf, xj, acc.y);
    if (FIELD) {
      const double cj = sc[jl];
      const double qt = a.yinf * a.emS * a.y0sq;
      const double sig = fma(rj, rj, ri2), e = fma(rj, rj, -ri2);
      const double P = fma(-dz2, qt, a.yinf);
      acc.bz = fma(fma(e, qt, P), cj, acc.bz);
      acc.br = fma(dz * fma(sig, qt, -P), cj, acc.br);
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

// ---- one multi-target item: T target blocks (32 T rings, T targets per lane) against one source block --------------
// Every staged source value (LDS) and every hop of the travelling sums (SHFL) serves T pair evaluations instead of one:
// the sweep is issue-bound and every non-FP64 instruction costs an issue slot.  UNI: every one of the
// T target blocks and the source block sit on one radius each (rows of a lattice).
template <int NIT, int ORD, bool FIELD, bool UNI, int T>
__device__ __forceinline__ void item_multi(const TargetRegs (&t)[T], const double* __restrict__ sr,
                                           const double* __restrict__ sz, const double* __restrict__ sx,
                                           const double* __restrict__ sc, double soft_all, double rju, int lane,
                                           Accum (&acc)[T], Accum& trav) {
  const unsigned full = 0xffffffffu;
  const int next = (lane + 1) & 31;
  double ri2[T], ri4[T], dif2u[T], c4u[T], eu[T], sigu[T];
#pragma unroll
  for (int k = 0; k < T; ++k) {
    ri2[k] = t[k].r * t[k].r;
    ri4[k] = 4.0 * t[k].r;
    const double difu = t[k].r - rju;
    dif2u[k] = FIELD ? difu * difu : fma(difu, difu, soft_all);
    c4u[k] = ri4[k] * rju;
    eu[k] = fma(rju, rju, -ri2[k]);
    sigu[k] = fma(rju, rju, ri2[k]);
  }
  sr += lane, sz += lane, sx += lane, sc += lane;   // arrays are stored twice: entry lane + s = source (lane + s) & 31
#pragma unroll kMultiUnroll
  for (int s = 0; s < 32; ++s) {
    const double zj = sz[s], xj = sx[s];
    const double rj = UNI ? rju : sr[s];
    const double cj = FIELD ? sc[s] : 0.0;
#pragma unroll
    for (int k = 0; k < T; ++k) {
      const double dz = t[k].z - zj;
      double dz2 = 0.0, A2, B2;
      if (UNI) {
        if (FIELD) {
          dz2 = fma(dz, dz, soft_all);
          B2 = dz2 + dif2u[k];
        } else {
          B2 = fma(dz, dz, dif2u[k]);
        }
        A2 = B2 + c4u[k];
      } else {
        dz2 = fma(dz, dz, soft_all);
        const double dif = t[k].r - rj;
        B2 = fma(dif, dif, dz2);
        A2 = fma(ri4[k], rj, B2);                            // (ri+rj)^2 = (ri-rj)^2 + 4 ri rj
      }
      const PairAGM a = agm_pair<NIT, ORD, FIELD>(A2, B2);
      const double mt = a.S * a.yinf;
      acc[k].y = fma(mt, xj, acc[k].y);
      trav.y = fma(mt, t[k].x, trav.y);
      if (FIELD) {
        const double qt = a.yinf * a.emS * a.y0sq;
        const double sig = UNI ? sigu[k] : fma(rj, rj, ri2[k]);   // ri^2 + rj^2
        const double e = UNI ? eu[k] : fma(-2.0, ri2[k], sig);    // rj^2 - ri^2
        const double P = fma(-dz2, qt, a.yinf);                   // Kt - dz^2 Qt
        const double R = e * qt;
        const double bz_ij = P + R;                               // Kt + (rj^2 - ri^2 - dz^2) Qt
        const double bz_ji = P - R;
        const double ur = dz * fma(sig, qt, -P);                  // dz (-Kt + (ri^2 + rj^2 + dz^2) Qt)
        acc[k].bz = fma(bz_ij, cj, acc[k].bz);
        acc[k].br = fma(ur, cj, acc[k].br);
        trav.bz = fma(bz_ji, t[k].cur, trav.bz);
        trav.br = fma(-ur, t[k].cur, trav.br);
      }
    }
    if (FIELD) {
      trav.bz = __shfl_sync(full, trav.bz, next);
      trav.br = __shfl_sync(full, trav.br, next);
    }
    trav.y = __shfl_sync(full, trav.y, next);
  }
}

// Work list.  Blocks of 32 rings are grouped T at a time into super-blocks I = 0 .. ceil(nb/T)-1 (the last one may hold
// fewer, Ta < T).  Row I of the list: first the "triangle" of the super-block with itself - for a = 0..Ta-1 the diagonal
// item (a, a) followed by the single-target items (a, b), b = a+1..Ta-1 - then the multi-target items (I, bj) for every
// source block bj >= T (I + 1).  Every unordered block pair appears exactly once.
template <int T>
struct WorkList {
  int nb, nbF, rem;
  __host__ __device__ explicit WorkList(int nb_) : nb(nb_), nbF(nb_ / T), rem(nb_ % T) {}
  static __host__ __device__ constexpr int tri(int n) { return n * (n + 1) / 2; }
  __host__ __device__ long long row_start(int I) const {   // I <= nbF
    return static_cast<long long>(I) * (tri(T) + nb) - static_cast<long long>(T) * I * (I + 1) / 2;
  }
  __host__ __device__ long long total() const { return row_start(nbF) + tri(rem); }
  __host__ __device__ int blocks_in(int I) const { return I < nbF ? T : rem; }
  __host__ __device__ int row_count(int I) const { return I < nbF ? tri(T) + nb - T * (I + 1) : tri(rem); }
  __device__ void unrank(long long k, int& I, int& loc) const {
    const double B = tri(T) + nb - 0.5 * T;
    const double disc = fmax(B * B - 2.0 * T * static_cast<double>(k), 0.0);
    int i = static_cast<int>(floor((B - sqrt(disc)) / T));
    i = max(0, min(i, nbF));
    while (i > 0 && row_start(i) > k) --i;
    while (i < nbF && row_start(i + 1) <= k) ++i;
    I = i;
    loc = static_cast<int>(k - row_start(i));
  }
  // item (I, loc) -> a, b (target / source block inside the super-block; a == b: diagonal; a < 0: multi item) and the
  // source block index bj
  __device__ void decode(int I, int loc, int& a, int& b, int& bj) const {
    const int Ta = blocks_in(I), ntri = tri(Ta);
    if (loc < ntri) {
      int aa = 0, l = loc;
      while (l >= Ta - aa) {
        l -= Ta - aa;
        ++aa;
      }
      a = aa;
      b = aa + l;
      bj = T * I + b;
    } else {
      a = -1;
      b = -1;
      bj = T * (I + 1) + (loc - ntri);
    }
  }
};

// resident CTAs per SM the register budget is sized for (measured, see QS_SW_MINB_*): fused 5 (96 registers);
// M-only 7 at T <= 2 (72 registers), 4 at T = 4 (128 registers)
constexpr int sweep_minb(bool field, int T) { return field ? QS_SW_MINB_FIELD : (T >= 4 ? QS_SW_MINB_M : QS_SW_MINB_M12); }
template <bool FIELD, int T>
__global__ void __launch_bounds__(kThreads, sweep_minb(FIELD, T)) sweep_kernel(SweepParams prm) {
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
  const WorkList<T> wl(prm.nb);

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
  auto add_into = [](Accum& dst, const Accum& v) {
    dst.y += v.y;
    if (FIELD) dst.br += v.br, dst.bz += v.bz;
  };

  for (;;) {
    long long k0 = 0;
    if (lane == 0) k0 = static_cast<long long>(atomicAdd(prm.counter, static_cast<unsigned long long>(prm.chunk)));
    k0 = __shfl_sync(full, k0, 0);
    if (k0 >= prm.n_items) break;
    const int cnt = static_cast<int>(min(static_cast<long long>(prm.chunk), prm.n_items - k0));
    int I, loc, a, b, bj;
    wl.unrank(k0, I, loc);
    wl.decode(I, loc, a, b, bj);
    issue(0, bj);

    TargetRegs t[T];
    Accum acc[T];
    double4 bbU = make_double4(0.0, 0.0, 0.0, 0.0);   // union of the boxes of the super-block's target blocks
    bool uniT = false;
    int cur_I = -1, Ta = 0;
    auto flush = [&]() {
#pragma unroll
      for (int k = 0; k < T; ++k)
        if (k < Ta) {
          const long long i = 32ll * (T * cur_I + k) + lane;
          red_add(prm.yacc + i, acc[k].y);
          if (FIELD) {
            red_add(prm.bracc + i, acc[k].br);
            red_add(prm.bzacc + i, acc[k].bz);
          }
        }
    };
    for (int it = 0; it < cnt; ++it) {
      const int buf = it & 1;
      if (I != cur_I) {  // new target super-block: flush the old accumulators, load the new targets
        if (cur_I >= 0) flush();
        cur_I = I;
        Ta = wl.blocks_in(I);
        uniT = true;
#pragma unroll
        for (int k = 0; k < T; ++k) {
          acc[k] = {0.0, 0.0, 0.0};
          const int blk = T * I + (k < Ta ? k : 0);
          const long long i = 32ll * blk + lane;
          t[k].r = prm.r[i];
          t[k].z = prm.z[i];
          t[k].x = prm.x[i];
          t[k].cur = FIELD ? prm.cur[i] : 0.0;
          const double4 bk = prm.bbox[blk];
          uniT = uniT && bk.x == bk.y;
          if (k == 0) {
            bbU = bk;
          } else {
            bbU.x = fmin(bbU.x, bk.x), bbU.y = fmax(bbU.y, bk.y);
            bbU.z = fmin(bbU.z, bk.z), bbU.w = fmax(bbU.w, bk.w);
          }
        }
      }
      // next item of this chunk, prefetched into the other buffer
      int nI = I, nloc = loc + 1, na = 0, nbb = 0, nbj = 0;
      if (nloc == wl.row_count(I)) {
        nI = I + 1;
        nloc = 0;
      }
      if (it + 1 < cnt) {
        wl.decode(nI, nloc, na, nbb, nbj);
        issue(buf ^ 1, nbj);
      }

      const double4 bbj = prm.bbox[bj];
      mbar_wait(&sbar[warp][buf], (phase >> buf) & 1u);
      phase ^= 1u << buf;
      const double* sr = sbuf[warp][buf][0];
      const double* sz = sbuf[warp][buf][1];
      const double* sx = sbuf[warp][buf][2];
      const double* sc = sbuf[warp][buf][3];
      if (a >= 0 && a == b) {   // diagonal item of target block a
        const int nit = classify(bbj, bbj, true, prm);
#pragma unroll
        for (int k = 0; k < T; ++k)
          if (k == a) {
#define QS_DIAG(N_, O_) item_diag<N_, O_, FIELD>(t[k], sr, sz, sx, sc, prm.soft_all, prm.soft_self, lane, acc[k])
            if (nit <= 4) {   // diagonal items are rare: every class up to (4, 2) shares (4, 2)
              QS_DIAG(4, 2);
            } else {
              switch (nit) {
                case 5: QS_DIAG(4, 4); break;
                case 6: QS_DIAG(5, 2); break;
                case 7: QS_DIAG(5, 4); break;
                case 8: QS_DIAG(6, 2); break;
                default: QS_DIAG(7, 2); break;
              }
            }
#undef QS_DIAG
          }
      } else if (a >= 0) {      // single-target item inside the super-block's triangle: rare, deepest class (always valid)
        Accum trav = {0.0, 0.0, 0.0};
#pragma unroll
        for (int k = 0; k < T - 1; ++k)
          if (k == a) item_offdiag<7, 2, FIELD, false>(t[k], sr, sz, sx, sc, prm.soft_all, 0.0, lane, acc[k], trav);
#pragma unroll
        for (int k = 1; k < T; ++k)
          if (k == b) add_into(acc[k], trav);   // lane l of trav = source ring l of block b = target l of acc[b]
      } else {
        const bool uni = uniT && bbj.x == bbj.y;   // every block on one radius (lattice rows)
        const int nit = classify(bbU, bbj, false, prm);
        Accum trav = {0.0, 0.0, 0.0};
#define QS_OFF(N_, O_)                                                                              \
  if (uni)                                                                                          \
    item_multi<N_, O_, FIELD, true, T>(t, sr, sz, sx, sc, prm.soft_all, bbj.x, lane, acc, trav);    \
  else                                                                                              \
    item_multi<N_, O_, FIELD, false, T>(t, sr, sz, sx, sc, prm.soft_all, 0.0, lane, acc, trav)
        QS_CLASS_SWITCH(nit, QS_OFF)
#undef QS_OFF
        red_add(prm.yacc + 32ll * bj + lane, trav.y);
        if (FIELD) {
          red_add(prm.bracc + 32ll * bj + lane, trav.br);
          red_add(prm.bzacc + 32ll * bj + lane, trav.bz);
        }
      }
      __syncwarp();  // every lane is done reading sbuf[buf] before it is refilled two items later
      I = nI, loc = nloc, a = na, b = nbb, bj = nbj;
    }
    flush();
  }
}

__global__ void diag_kernel(int n, const double* __restrict__ r, double d2self, double* __restrict__ diagM) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const double s = r[i] + r[i];
  const PairAGM a = agm_pair<7, 2, false>(fma(s, s, d2self), d2self);
  diagM[i] = (0.5 * kMu0 * kPi) * a.S * a.yinf;
}
// ---- test hook: one pair per thread through a chosen evaluation class (cls < 0: chosen from k'^2 like the sweep) ----
template <int NIT, int ORD>
__device__ __forceinline__ void pair_out(double A2, double B2, double* M, double* K, double* E) {
  const PairAGM a = agm_pair<NIT, ORD, true>(A2, B2);
  *M = (0.5 * kMu0 * kPi) * a.S * a.yinf;
  const double sa = sqrt(A2);
  *K = (0.5 * kPi) * a.yinf * sa;
  *E = (0.5 * kPi) * a.yinf * a.emS / sa;
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
#define QS_PAIR_OUT(N_, O_) pair_out<N_, O_>(A2[i], B2[i], M + i, K + i, E + i)
  QS_CLASS_SWITCH(c, QS_PAIR_OUT)
#undef QS_PAIR_OUT
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
    const PairAGM a = agm_pair<7, 2, false>(A2, B2);
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


// Target blocks per multi-target item, by problem size: small ring sets have too few items for big ones, large ones
// gain from the shared source loads and shuffles.  Measured, T = 1 / 2 / 4 (ms): matvec on free
// rings N = 4,096: 0.054 / 0.060 / 0.070; 16,384: 0.500 / 0.498 / 0.637; 65,536: 7.32 / 7.16 / 7.43; 262,144: 112.2 /
// 106.9 / 104.1; lattice matvec config 0: 0.024 / 0.032 / 0.040, config 1: 0.058 / 0.064 / 0.069, N = 34,560:
// 2.38 / 2.28 / 3.04; fused sweep config 0: 0.019 / 0.029, config 1: 0.065 / 0.066.  QS_SW_T_FORCE_* pin the choice.
int sweep_T(int nb, bool field) {
#ifdef QS_SW_T_FORCE_FIELD
  if (field) return QS_SW_T_FORCE_FIELD;
#endif
#ifdef QS_SW_T_FORCE_M
  if (!field) return QS_SW_T_FORCE_M;
#endif
  if (field) return nb >= QS_SW_NB_T2 ? 2 : 1;
  return nb >= QS_SW_NB_T4 ? 4 : (nb >= QS_SW_NB_T2 ? 2 : 1);
}

int sweep_grid(int sm_count, bool field, int nb) { return sm_count * sweep_minb(field, sweep_T(nb, field)); }

long long sweep_items(int nb, bool field) {
  switch (sweep_T(nb, field)) {
    case 1: return WorkList<1>(nb).total();
    case 2: return WorkList<2>(nb).total();
    default: return WorkList<4>(nb).total();
  }
}

cudaError_t launch_sweep(const SweepParams& prm, bool field, int grid, cudaStream_t stream) {
  const int T = sweep_T(prm.nb, field);
  if (field) {
    if (T == 1) sweep_kernel<true, 1><<<grid, kThreads, 0, stream>>>(prm);
    else sweep_kernel<true, 2><<<grid, kThreads, 0, stream>>>(prm);
  } else {
    if (T == 1) sweep_kernel<false, 1><<<grid, kThreads, 0, stream>>>(prm);
    else if (T == 2) sweep_kernel<false, 2><<<grid, kThreads, 0, stream>>>(prm);
    else sweep_kernel<false, 4><<<grid, kThreads, 0, stream>>>(prm);
  }
  return cudaGetLastError();
}

int sweep_warps_per_cta() { return kWarpsPerCta; }

}  // namespace qs
