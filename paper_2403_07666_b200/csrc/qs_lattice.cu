// qs_lattice.cu — lattice-aware operator (geometry: the square array of wires).
//
// On a regular winding pack the pair kernels depend only on (ir, jr, iz - jz): M, G_Bz are even and G_Br is odd in
// iz - jz.  At init every unique value is evaluated ONCE with the same per-pair arithmetic as the on-the-fly sweeps
// (qs_pair.cuh, deepest evaluation class) into tables T[ir][jr][d], d = |iz - jz| = 0..Nz-1; a sweep is then a
// block-Toeplitz product
//     y[ir][iz] = sum_jr sum_jz T[ir][jr][|iz - jz|] x[jr][jz]
// — N^2 FP64 multiply-adds instead of N^2/2 AGM evaluations (~60 FP64 operations each).  The tables hold the same
// unscaled quantities the pair sweeps accumulate, and the kernel adds into the same accumulators (yacc, bracc, bzacc),
// so everything downstream (scaling, material law, CG) is unchanged and either operator can serve a handle.
//
// Kernel: a CTA owns one target row ir, a chunk of source rows jr and a tile of T*R outputs; thread t owns R ADJACENT
// outputs (R odd: the stride-R shared-memory reads of the table window are bank-conflict free).  Per source row the
// table row is mirrored into shared memory as t_ext[e], e = iz - jz in (-Nz, Nz), next to the source row x; the thread
// then slides over jz with a register window W[k] = t_ext[iz0 + k - jz]: one broadcast read of x[jz] and ONE new
// window element per jz feed R multiply-adds (register rotation by unrolling, no moves).  Partial sums over the
// jr chunks are combined with FP64 red.add in L2.
#include <algorithm>

#include "qs_internal.h"
#include "qs_pair.cuh"

namespace qs {

namespace {

// ---- table construction: one thread per (ir, jr, d) ---------------------------------------------------------------
__global__ void table_build_kernel(int Nr, int Nz, double r_inner, double h, double soft_self2, double* __restrict__ TM,
                                   double* __restrict__ TBz, double* __restrict__ TBr) {
  const long long total = static_cast<long long>(Nr) * Nr * Nz;
  for (long long id = blockIdx.x * static_cast<long long>(blockDim.x) + threadIdx.x; id < total;
       id += static_cast<long long>(gridDim.x) * blockDim.x) {
    const int d = static_cast<int>(id % Nz);
    const long long rr = id / Nz;
    const int jr = static_cast<int>(rr % Nr), ir = static_cast<int>(rr / Nr);
    const double ri = r_inner + (ir + 0.5) * h, rj = r_inner + (jr + 0.5) * h;
    const double dz = d * h;                                   // target above source: dz = z_i - z_j >= 0
    const bool self = (ir == jr) && d == 0;
    const double dz2 = self ? soft_self2 : dz * dz;            // C2: M_ii = M(r_i, r_i, dz = g)
    const double dif = ri - rj;
    const double B2 = fma(dif, dif, dz2), A2 = fma(4.0 * ri, rj, B2);
    const PairAGM a = agm_pair<7, 2, true>(A2, B2);
    TM[id] = a.S * a.yinf;
    if (TBz) {
      if (self) {                                              // C3: the self field is analytic (material pass)
        TBz[id] = 0.0;
        TBr[id] = 0.0;
      } else {
        const double qt = a.yinf * a.emS * a.y0sq;
        const double e = fma(rj, rj, -ri * ri), sig = fma(rj, rj, ri * ri);
        const double P = fma(-dz2, qt, a.yinf);                // Kt - dz^2 Qt
        TBz[id] = fma(e, qt, P);                               // Kt + (rj^2 - ri^2 - dz^2) Qt
        TBr[id] = dz * fma(sig, qt, -P);                       // dz (-Kt + (ri^2 + rj^2 + dz^2) Qt), odd in dz
      }
    }
  }
}

// ---- block-Toeplitz sweep -----------------------------------------------------------------------------------------
template <int R, bool FIELD>
__global__ void __launch_bounds__(256) table_sweep_kernel(LatticeSweepParams prm) {
  extern __shared__ __align__(16) double lsm[];
  const int Nz = prm.Nz, T = blockDim.x;
  const int NzPad = (Nz + R - 1) / R * R;                      // source loop runs in blocks of R
  const int ext_len = NzPad + T * R;                           // e in [-NzPad, T R)
  double* tM = lsm;                                            // t_ext[e] at tM[e + NzPad]
  double* tBz = FIELD ? tM + ext_len : nullptr;
  double* tBr = FIELD ? tBz + ext_len : nullptr;
  double* xs = (FIELD ? tBr : tM) + ext_len;                   // [NzPad]
  double* cs = FIELD ? xs + NzPad : nullptr;
  if (prm.done != nullptr && *prm.done != 0) return;           // a converged CG batch: nothing left to do
  const int ir = blockIdx.y;
  const int j0 = blockIdx.x * prm.jr_chunk, j1 = min(j0 + prm.jr_chunk, prm.Nr);
  const int z0 = blockIdx.z * T * R;                           // first output of this tile
  const int iz0 = z0 + threadIdx.x * R;
  double yM[R], yBz[FIELD ? R : 1], yBr[FIELD ? R : 1];
#pragma unroll
  for (int k = 0; k < R; ++k) {
    yM[k] = 0.0;
    if (FIELD) yBz[k] = 0.0, yBr[k] = 0.0;
  }
  for (int jr = j0; jr < j1; ++jr) {
    __syncthreads();
    const long long trow = (static_cast<long long>(ir) * prm.Nr + jr) * Nz;
    const long long xrow = static_cast<long long>(jr) * Nz;
    for (int s = threadIdx.x; s < ext_len; s += T) {           // mirrored table row; zero outside |e| < Nz
      const int e = s - NzPad + z0;                            // e = iz - jz of window slot s for this tile
      const int d = abs(e);
      const bool in = d < Nz;
      tM[s] = in ? prm.TM[trow + d] : 0.0;
      if (FIELD) {
        tBz[s] = in ? prm.TBz[trow + d] : 0.0;
        const double br = in ? prm.TBr[trow + d] : 0.0;
        tBr[s] = e < 0 ? -br : br;
      }
    }
    for (int s = threadIdx.x; s < NzPad; s += T) {
      xs[s] = s < Nz ? prm.x[xrow + s] : 0.0;
      if (FIELD) cs[s] = s < Nz ? prm.cur[xrow + s] : 0.0;
    }
    __syncthreads();
    // Element of (output k, source jz): t_ext[iz0 + k - jz] = wM[k - jz].  As jz grows the window slides: the new
    // element enters at output 0 and every older one moves up one output, so an element keeps its REGISTER if
    // output k reads register (k - jz) mod R: with the jz loop unrolled R times all indices are compile-time.
    const double* wM = tM + (iz0 - z0) + NzPad;
    const double* wBz = FIELD ? tBz + (iz0 - z0) + NzPad : nullptr;
    const double* wBr = FIELD ? tBr + (iz0 - z0) + NzPad : nullptr;
    double WM[R], WBz[FIELD ? R : 1], WBr[FIELD ? R : 1];
#pragma unroll
    for (int k = 1; k < R; ++k) {                              // jz = 0: outputs k >= 1 (output 0 is loaded in the loop)
      WM[k] = wM[k];
      if (FIELD) WBz[k] = wBz[k], WBr[k] = wBr[k];
    }
    for (int jb = 0; jb < NzPad; jb += R) {
#pragma unroll
      for (int u = 0; u < R; ++u) {
        const int jz = jb + u;
        constexpr int kR = R;
        const int reg0 = (kR - u) % kR;                        // register of output 0 at this source
        WM[reg0] = wM[-jz];
        if (FIELD) WBz[reg0] = wBz[-jz], WBr[reg0] = wBr[-jz];
        const double x = xs[jz];
        const double c = FIELD ? cs[jz] : 0.0;
#pragma unroll
        for (int k = 0; k < R; ++k) {
          const int reg = (reg0 + k) % kR;
          yM[k] = fma(WM[reg], x, yM[k]);
          if (FIELD) {
            yBz[k] = fma(WBz[reg], c, yBz[k]);
            yBr[k] = fma(WBr[reg], c, yBr[k]);
          }
        }
      }
    }
  }
  const long long orow = static_cast<long long>(ir) * Nz;
#pragma unroll
  for (int k = 0; k < R; ++k) {
    const int iz = iz0 + k;
    if (iz < Nz) {
      asm volatile("red.global.add.f64 [%0], %1;" ::"l"(prm.yacc + orow + iz), "d"(yM[k]) : "memory");
      if (FIELD) {
        asm volatile("red.global.add.f64 [%0], %1;" ::"l"(prm.bzacc + orow + iz), "d"(yBz[k]) : "memory");
        asm volatile("red.global.add.f64 [%0], %1;" ::"l"(prm.bracc + orow + iz), "d"(yBr[k]) : "memory");
      }
    }
  }
}

// ---- block-Toeplitz sweep on the FP64 tensor cores (mma.sync m8n8k4, SASS DMMA) ---------------------------------------
// The product is a dense contraction, so it belongs on the tensor pipe: one DMMA does 256 multiply-adds for one issue
// slot (measured 37.1 TFLOP/s = the full FP64 rate, 16 cycles per mma per sub-partition), where the multiply-add kernel
// above is capped at 2/3 of the rate by its three-register-operand DFMAs.  With iz = 8p + q, jz = 8a + b and d = p - a:
//     Y[p][q] += sum_b X[p - d][b] * t[8d + q - b]
// is, for 8 consecutive p and a fixed block offset d, an (8 x 8) += (8 x 8)(8 x 8) product = two m8n8k4 steps whose
// A operand is a block of 8 x 8 source values (rows = source blocks p - d) and whose B operand is the Toeplitz block
// T_d[b][q] = t[8d + q - b].  A warp owns NT tiles of 64 outputs which share every B fragment; the fused sweep shares
// the A fragment of the ring currents between the Bz and Br tables.  Fragments are read from shared memory:
//   * the source row in 8-blocks padded to a stride of 12 slots (conflict-free for the row-strided A pattern); in the
//     fused sweep a slot is the pair {x, ring current}, so one LDS.128 fetches both A fragments;
//   * the mirrored table row t_ext[e]; in the fused sweep the three tables are interleaved per offset, so the three
//     B fragments are one pointer with immediate offsets (stride 3 is odd: conflict-free).
// The offset loop is split into segments with a compile-time tile mask (the first 8 offsets reach only tile 0, the last
// 8 only tile 1), its pointers advance by constants, and the fragments of the next k-step are loaded before the DMMAs
// of the current one are issued (two register sets alternate, no copies).
constexpr int kMmaNT = 2;
constexpr int kMmaBlk = 12;                                        // slots per source 8-block in shared memory

__device__ __forceinline__ void dmma(double (&c)[2], double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
               : "+d"(c[0]), "+d"(c[1])
               : "d"(a), "d"(b));
}

template <bool FIELD>
struct MmaFrag {
  double b[FIELD ? 3 : 1];                                         // B fragments: k = lk (+4 kk), n = li, per table
  double ax[kMmaNT], ac[FIELD ? kMmaNT : 1];                       // A fragments: row li = output block, k = lk (+4 kk)
};

template <bool FIELD, int MASK>
__device__ __forceinline__ void mma_load(MmaFrag<FIELD>& f, const double* pa, const double* pb) {
  f.b[0] = pb[0];
  if constexpr (FIELD) f.b[1] = pb[1], f.b[2] = pb[2];
#pragma unroll
  for (int j = 0; j < kMmaNT; ++j) {
    if (!((MASK >> j) & 1)) continue;
    if constexpr (FIELD) {
      const double2 v = *reinterpret_cast<const double2*>(pa + j * 8 * kMmaBlk * 2);
      f.ax[j] = v.x, f.ac[j] = v.y;
    } else {
      f.ax[j] = pa[j * 8 * kMmaBlk];
    }
  }
}

template <bool FIELD, int MASK>
__device__ __forceinline__ void mma_issue(double (&acc)[kMmaNT][FIELD ? 3 : 1][2], const MmaFrag<FIELD>& f) {
#pragma unroll
  for (int j = 0; j < kMmaNT; ++j) {
    if (!((MASK >> j) & 1)) continue;
    dmma(acc[j][0], f.ax[j], f.b[0]);
    if constexpr (FIELD) {
      dmma(acc[j][1], f.ac[j], f.b[1]);
      dmma(acc[j][2], f.ac[j], f.b[2]);
    }
  }
}

// Offsets d0..d1 for the tiles in MASK.  pa / pb: this lane's A / B fragment of k-step 0 at offset d0.  The last trip
// loads the fragments of offset d1 + 1, which are not used: the shared arrays carry one guard block for that.
template <bool FIELD, int MASK>
__device__ __forceinline__ void mma_segment(double (&acc)[kMmaNT][FIELD ? 3 : 1][2], const double* pa, const double* pb,
                                            int d0, int d1) {
  constexpr int W = FIELD ? 2 : 1, TW = FIELD ? 3 : 1;
  if (d0 > d1) return;
  MmaFrag<FIELD> f0, f1;
  mma_load<FIELD, MASK>(f0, pa, pb);
  for (int d = d0; d <= d1; ++d) {
    mma_load<FIELD, MASK>(f1, pa + 4 * W, pb - 4 * TW);            // k-step 1 of offset d
    mma_issue<FIELD, MASK>(acc, f0);
    pa -= kMmaBlk * W;
    pb += 8 * TW;
    mma_load<FIELD, MASK>(f0, pa, pb);                             // k-step 0 of offset d + 1
    mma_issue<FIELD, MASK>(acc, f1);
  }
}

// <= 8 warps per CTA; the register budget of three 8-warp CTAs (<= 80 per thread, 78 used by the fused sweep) keeps the
// warp count shared-memory bound (102 registers unbounded: config 2 8.07 ms, this budget 7.87 ms; 64 registers: 8.18 ms)
template <bool FIELD>
__global__ void __launch_bounds__(256, 3) table_sweep_mma_kernel(LatticeSweepParams prm, int P, int n_asplit, int A_c) {
  // The CTA owns the outputs of its warps (8 NT p-blocks each) and the SOURCE blocks a in [a_lo, a_hi): splitting the
  // sources as well as the outputs keeps the shared-memory windows near 50 KB (four CTAs per SM) on long rows.
  extern __shared__ __align__(16) double lsm[];
  constexpr int NT = kMmaNT, NTAB = FIELD ? 3 : 1, W = FIELD ? 2 : 1, TW = FIELD ? 3 : 1;
  static_assert(NT == 2, "the segment split below is written for two tiles per warp");
  const int Nz = prm.Nz, T = blockDim.x;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarps = T >> 5;
  const int zt = blockIdx.z / n_asplit, as = blockIdx.z - zt * n_asplit;
  const int a_lo = as * A_c, a_hi = min(a_lo + A_c, P);
  const int p_lo = zt * nwarps * 8 * NT;                          // first p-block of the CTA's outputs
  const int np_cta = nwarps * 8 * NT;
  const int xblocks = A_c + 15;                                   // source blocks a_lo - 8 .. a_lo + A_c + 6
  const int e0 = 8 * (p_lo - (a_lo + A_c) + 1) - 8;               // first offset iz - jz of the table window
  const int tlen = 8 * (np_cta + A_c + 8) + 32;                   // incl. the guard of the look-ahead load
  double* xc = lsm;                                               // slot (blk, b) at [(blk * 12 + b) * W (+ 1: current)]
  double* tt = xc + xblocks * kMmaBlk * W;                        // t_ext[e] of table k at [(e - e0) * TW + k]
  if (prm.done != nullptr && *prm.done != 0) return;
  const int ir = blockIdx.y;
  const int j0 = blockIdx.x * prm.jr_chunk, j1 = min(j0 + prm.jr_chunk, prm.Nr);
  const int pw = p_lo + warp * 8 * NT;                            // first 8-block of this warp's outputs
  const int li = lane >> 2, lk = lane & 3;
  double acc[NT][NTAB][2];
#pragma unroll
  for (int j = 0; j < NT; ++j)
#pragma unroll
    for (int t = 0; t < NTAB; ++t) acc[j][t][0] = acc[j][t][1] = 0.0;
  // offset ranges of the two tiles (tile 1 = tile 0 shifted by 8 blocks) and the three segments of the union
  const int lo0 = pw - (a_hi - 1), hi0 = pw + 7 - a_lo, lo1 = lo0 + 8, hi1 = hi0 + 8;
  const bool two = pw + 8 < P;                                    // tile 1 inside the row
  for (int jr = j0; jr < j1; ++jr) {
    __syncthreads();
    const long long trow = (static_cast<long long>(ir) * prm.Nr + jr) * Nz;
    const long long xrow = static_cast<long long>(jr) * Nz;
    for (int s = threadIdx.x; s < xblocks * 8; s += T) {          // source blocks of this CTA, zero outside its range
      const int blk = s >> 3, b = s & 7;
      const int a = a_lo - 8 + blk, j = 8 * a + b;
      const bool in = a >= a_lo && a < a_hi && j < Nz;
      const double xv = in ? prm.x[xrow + j] : 0.0;
      if constexpr (FIELD) {
        const double cv = in ? prm.cur[xrow + j] : 0.0;
        reinterpret_cast<double2*>(xc)[blk * kMmaBlk + b] = make_double2(xv, cv);
      } else {
        xc[blk * kMmaBlk + b] = xv;
      }
    }
    for (int s = threadIdx.x; s < tlen; s += T) {                 // mirrored table row, zero outside |e| < Nz
      const int e = s + e0, d = abs(e);
      const bool in = d < Nz;
      tt[s * TW] = in ? prm.TM[trow + d] : 0.0;
      if constexpr (FIELD) {
        tt[s * TW + 1] = in ? prm.TBz[trow + d] : 0.0;
        const double br = in ? prm.TBr[trow + d] : 0.0;
        tt[s * TW + 2] = e < 0 ? -br : br;
      }
    }
    __syncthreads();
    if (pw >= P) continue;                                        // warp beyond the row: only helps with the fills
    // fragment addresses at offset d: A (tile 0) slot ((pw + li - d - a_lo + 8) * 12 + lk), B element 8 d + li - lk - e0
    auto pa_at = [&](int d) { return xc + ((pw + li - d - a_lo + 8) * kMmaBlk + lk) * W; };
    auto pb_at = [&](int d) { return tt + (8 * d + li - lk - e0) * TW; };
    if (!two) {
      mma_segment<FIELD, 1>(acc, pa_at(lo0), pb_at(lo0), lo0, hi0);
    } else {
      const int a1 = min(hi0, lo1 - 1), c0 = max(hi0 + 1, lo1);
      mma_segment<FIELD, 1>(acc, pa_at(lo0), pb_at(lo0), lo0, a1);
      mma_segment<FIELD, 3>(acc, pa_at(lo1), pb_at(lo1), lo1, hi0);
      mma_segment<FIELD, 2>(acc, pa_at(c0), pb_at(c0), c0, hi1);
    }
  }
  const long long orow = static_cast<long long>(ir) * Nz;
#pragma unroll
  for (int j = 0; j < NT; ++j) {
    const int iz = 8 * (pw + 8 * j + li) + 2 * lk;                // C fragment: row li, columns 2 lk, 2 lk + 1
#pragma unroll
    for (int h = 0; h < 2; ++h) {
      if (iz + h < Nz) {
        asm volatile("red.global.add.f64 [%0], %1;" ::"l"(prm.yacc + orow + iz + h), "d"(acc[j][0][h]) : "memory");
        if (FIELD) {
          asm volatile("red.global.add.f64 [%0], %1;" ::"l"(prm.bzacc + orow + iz + h), "d"(acc[j][1][h]) : "memory");
          asm volatile("red.global.add.f64 [%0], %1;" ::"l"(prm.bracc + orow + iz + h), "d"(acc[j][2][h]) : "memory");
        }
      }
    }
  }
}

}  // namespace

cudaError_t launch_table_build(int Nr, int Nz, double r_inner, double h, double soft_self2, double* TM, double* TBz,
                               double* TBr, int sm_count, cudaStream_t stream) {
  table_build_kernel<<<sm_count * 8, 256, 0, stream>>>(Nr, Nz, r_inner, h, soft_self2, TM, TBz, TBr);
  return cudaGetLastError();
}

// T threads x R outputs per thread covering Nz with the least padding (R odd, T a multiple of 32)
void lattice_sweep_shape(int Nz, int* T_out, int* R_out, int* tiles_out) {
  int bestT = 32, bestR = 1, bestTiles = (Nz + 31) / 32;
  long long bestCost = -1;
  const int Rs[5] = {1, 3, 5, 7, 9};
  for (int T = 32; T <= 256; T += 32)
    for (int ri = 0; ri < 5; ++ri) {
      const int R = Rs[ri];
      const int tiles = (Nz + T * R - 1) / (T * R);
      // cost ~ issue slots per source element: T threads x (3 cycles per multiply-add x R + 2 shared-memory reads)
      const long long cost = static_cast<long long>(tiles) * T * (3 * R + 2) * 8 - T / 32;
      if (bestCost < 0 || cost < bestCost) bestCost = cost, bestT = T, bestR = R, bestTiles = tiles;
    }
  *T_out = bestT;
  *R_out = bestR;
  *tiles_out = bestTiles;
}

size_t lattice_sweep_smem(int Nz, int T, int R, bool field) {
  const int NzPad = (Nz + R - 1) / R * R;
  const int ext_len = NzPad + T * R;
  return sizeof(double) * (static_cast<size_t>(field ? 3 : 1) * ext_len + static_cast<size_t>(field ? 2 : 1) * NzPad);
}

template <int R>
static cudaError_t launch_R(const LatticeSweepParams& prm, bool field, dim3 grid, int T, size_t smem, cudaStream_t stream) {
  if (field) {
    cudaFuncSetAttribute(table_sweep_kernel<R, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, static_cast<int>(smem));
    table_sweep_kernel<R, true><<<grid, T, smem, stream>>>(prm);
  } else {
    cudaFuncSetAttribute(table_sweep_kernel<R, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, static_cast<int>(smem));
    table_sweep_kernel<R, false><<<grid, T, smem, stream>>>(prm);
  }
  return cudaGetLastError();
}

// tensor-core variant
static size_t mma_sweep_smem(bool field, int nwarps, int A_c) {
  const int np_cta = nwarps * 8 * kMmaNT;
  return sizeof(double) * (static_cast<size_t>(field ? 2 : 1) * (A_c + 15) * kMmaBlk +
                           static_cast<size_t>(field ? 3 : 1) * (8 * (np_cta + A_c + 8) + 32));
}

// Launch shape of the tensor-core sweep: warps per CTA (each owns 8 NT output blocks), CTAs per row, and the number of
// source-block ranges a row is split into.  Measured on B200 (config 2: 80 blocks = 5 warp tiles, config 3: 150 blocks
// = 10 warp tiles; fused / M-only sweep in ms):
//   config 2: one 5-warp CTA per row 7.87 / 2.65 (four / six CTAs resident per SM); 3 + 2 warps 9.18 / 2.67; 2 + 2 + 1
//             warps 9.85 / 3.19; sources split in two 9.18 / 2.94
//   config 3: 4 + 4 + 2 warps 143.6 / 46.2 (three 74 KB CTAs = 12 warps per SM); 5 + 5 warps 185.4 / 49.8 (two 77 KB
//             CTAs = 10 warps: 3, 3, 2, 2 per sub-partition); 3 + 3 + 3 + 1 190.8 / 48.8; 5 + 5 on half the sources each
//             149.3 / 52.8 (four CTAs = 20 warps, but a tile of 8 output blocks sweeps A_c + 7 block offsets for A_c
//             source blocks: 9 % padding instead of 4.5 %)
// The DMMA pipe is per sub-partition, so a launch is as fast as its most loaded sub-partition; beyond ~12 resident warps
// the count itself matters little; CTAs of 1-2 warps pay for their window fills.  So: among >= 3 warps per CTA (fewer
// only if the row has fewer tiles) with the sources unsplit (split only when the windows do not fit otherwise), estimate
// the resident warps R per SM from shared memory and registers and take the smallest ceil(R / 4) / (R / 4); on a tie
// fewer CTAs per row, then more resident warps.
static void mma_sweep_shape(bool field, int P, int regs_per_thread, int* nwarps_out, int* ztiles_out, int* nas_out) {
  const int wn = (P + 8 * kMmaNT - 1) / (8 * kMmaNT);
  const int regs_per_warp = ((regs_per_thread * 32 + 511) / 512) * 512;
  *nwarps_out = std::min(wn, 8), *ztiles_out = (wn + 7) / 8, *nas_out = 1;
  for (int nas = 1; nas <= 16; ++nas) {
    const int A_c = (P + nas - 1) / nas;
    double best = 1e300;
    int bestR = 0, bestZ = 0;
    for (int nw = std::min(wn, 3); nw <= 8; ++nw) {
      const int ztiles = (wn + nw - 1) / nw, nwarps = (wn + ztiles - 1) / ztiles;
      if (nwarps != nw) continue;                                  // the equalised shape is enumerated under its own nw
      const size_t smem = mma_sweep_smem(field, nwarps, A_c);
      if (smem > 227u * 1024u) continue;
      const int by_smem = static_cast<int>((228u * 1024u) / (smem + 1024u));
      const int by_regs = 65536 / (regs_per_warp * nwarps);
      const int ctas = std::min(std::min(by_smem, by_regs), std::min(32, 64 / nwarps));
      if (ctas < 1) continue;
      const int R = ctas * nwarps;
      const double cost = static_cast<double>((R + 3) / 4) / (R / 4.0) * (R < 8 ? 8.0 / R : 1.0);
      const bool better = cost < best - 1e-9 ||
                          (cost < best + 1e-9 && (ztiles < bestZ || (ztiles == bestZ && R > bestR)));
      if (better) best = cost, bestR = R, bestZ = ztiles, *nwarps_out = nwarps, *ztiles_out = ztiles, *nas_out = nas;
    }
    if (bestR > 0) return;                                         // a shape fits with this split
  }
}

template <bool FIELD>
static cudaError_t launch_mma_T(LatticeSweepParams prm, int sm_count, cudaStream_t stream) {
  static int regs = 0;                                               // of this instantiation (the same on every device)
  if (regs == 0) {
    cudaFuncAttributes at;
    const cudaError_t e = cudaFuncGetAttributes(&at, table_sweep_mma_kernel<FIELD>);
    if (e != cudaSuccess) return e;
    regs = at.numRegs;
  }
  const int P = (prm.Nz + 7) / 8;
  int nwarps, ztiles, n_asplit;
  mma_sweep_shape(FIELD, P, regs, &nwarps, &ztiles, &n_asplit);
  const int A_c = (P + n_asplit - 1) / n_asplit;
  // many small CTAs (a few source rows each): the fill of one CTA overlaps the DMMA phase of its neighbours on the SM
  // and the tail of the launch stays short (measured: 10.7 ms at 12 CTAs per SM, 9.3 ms at one source row per CTA)
  const long long want = 1000ll * sm_count;
  const int per_split = prm.Nr * ztiles * n_asplit;
  int splits = static_cast<int>(std::max<long long>(1, std::min<long long>(prm.Nr, want / std::max(1, per_split))));
  prm.jr_chunk = (prm.Nr + splits - 1) / splits;
  splits = (prm.Nr + prm.jr_chunk - 1) / prm.jr_chunk;
  const dim3 grid(splits, prm.Nr, ztiles * n_asplit);
  const size_t smem = mma_sweep_smem(FIELD, nwarps, A_c);
  cudaFuncSetAttribute(table_sweep_mma_kernel<FIELD>, cudaFuncAttributeMaxDynamicSharedMemorySize, static_cast<int>(smem));
  table_sweep_mma_kernel<FIELD><<<grid, nwarps * 32, smem, stream>>>(prm, P, n_asplit, A_c);
  return cudaGetLastError();
}

// tensor-core variant
static cudaError_t launch_table_sweep_mma(const LatticeSweepParams& prm, bool field, int sm_count, cudaStream_t stream) {
  return field ? launch_mma_T<true>(prm, sm_count, stream) : launch_mma_T<false>(prm, sm_count, stream);
}

cudaError_t launch_table_sweep(const LatticeSweepParams& prm_in, bool field, int sm_count, cudaStream_t stream) {
  LatticeSweepParams prm = prm_in;
  if (prm.Nz >= 128) return launch_table_sweep_mma(prm, field, sm_count, stream);   // shorter rows: FMA kernel
  int T, R, tiles;
  lattice_sweep_shape(prm.Nz, &T, &R, &tiles);
  // split the source rows so that the grid fills the GPU several times over
  const long long want = 16ll * sm_count;
  int splits = static_cast<int>(std::max<long long>(1, std::min<long long>(prm.Nr, want / std::max(1, prm.Nr * tiles))));
  prm.jr_chunk = (prm.Nr + splits - 1) / splits;
  splits = (prm.Nr + prm.jr_chunk - 1) / prm.jr_chunk;
  const dim3 grid(splits, prm.Nr, tiles);
  const size_t smem = lattice_sweep_smem(prm.Nz, T, R, field);
  switch (R) {
    case 1: return launch_R<1>(prm, field, grid, T, smem, stream);
    case 3: return launch_R<3>(prm, field, grid, T, smem, stream);
    case 5: return launch_R<5>(prm, field, grid, T, smem, stream);
    case 7: return launch_R<7>(prm, field, grid, T, smem, stream);
    default: return launch_R<9>(prm, field, grid, T, smem, stream);
  }
}

}  // namespace qs
