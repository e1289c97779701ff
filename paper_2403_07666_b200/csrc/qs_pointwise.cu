// qs_pointwise.cu — K5 material law, K6 explicit heat sub-step, K7 event detector, step statistics.
//
// All three are streaming passes over per-cell FP64 arrays (HBM/L2 bound):
//   K5 reads J, H, bracc, bzacc, jc0_scale, r, area, selfcoef, diagM and writes Br, Bz, E, dE/dJ, Q, b, shift, Hd,
//      Jc, rho (C5, C4, C7).
//   K6 one explicit finite-volume sub-step in enthalpy form (C9; PAPER.md:75 heat equation with Robin borders):
//      a CTA stages T^2 of its tile plus a one-cell halo in shared memory (one sqrt per staged cell), so the
//      algorithmic traffic is read H, Q + write H = 24 B per cell per sub-step.  Lattices of <= 4096 cells run all
//      sub-steps of a step in one launch: one CTA, or a thread-block cluster of 8 CTAs with DSMEM halo rows.
//   K7 one warp per turn over the CSR cell list: Tmax, mean|E|, max|J|/Jc, min rho/rho_n -> flags (C10).
#include <algorithm>
#include <cooperative_groups.h>

#include "qs_internal.h"
#include "qs_pair.cuh"
#include "qs_tma.cuh"

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
__device__ __forceinline__ double warp_min(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v = fmin(v, __shfl_xor_sync(0xffffffffu, v, o));
  return v;
}
__device__ __forceinline__ void atomic_max_pos(double* addr, double v) {   // v >= 0: IEEE order == integer order
  atomicMax(reinterpret_cast<unsigned long long*>(addr), static_cast<unsigned long long>(__double_as_longlong(v)));
}

// T^2 from the enthalpy H = C3/4 T^4 + C1/2 T^2
__device__ __forceinline__ double tsq_of_H(double H, double C3, double C1) {
  return (-0.5 * C1 + sqrt(0.25 * C1 * C1 + C3 * H)) / (0.5 * C3);
}

// T^2 from H with the fast reciprocal square root (MUFU seed + one Halley step): argument > 0 always (H >= 0)
__device__ __forceinline__ double tsq_fast(double H, double C3, double qC1sq, double hC1, double inv_hC3) {
  const double a = fma(C3, H, qC1sq);                 // C1^2/4 + C3 H
  const double y0 = rsqrt_seed(a);
  const double g = a * y0;
  const double e = fma(-g, y0, 1.0);
  const double s = fma(g * e, fma(0.375, e, 0.5), g); // sqrt(a)
  return (s - hC1) * inv_hC3;
}

// 1/x for a positive normal x: MUFU seed + two Newton steps (relative error ~ 1 ulp)
__device__ __forceinline__ double rcp_fast(double x) {
  double y;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
  double e = fma(-x, y, 1.0);
  y = fma(y, e, y);
  e = fma(-x, y, 1.0);
  return fma(y, e, y);
}
// sqrt(a), a >= 0: MUFU seed + one Halley step; exact zero for a == 0
__device__ __forceinline__ double sqrt_pos(double a) {
  const double y0 = rsqrt_seed(a + 1e-300);           // a == 0: g = 0 * 1e150 = 0, e = 1, result 0
  const double g = a * y0;
  const double e = fma(-g, y0, 1.0);
  return fma(g * e, fma(0.375, e, 0.5), g);
}
// x^e for 0 < x < ~1 (the strain term |eps|^1.7): exp(e log x) with both series written out against coefficient
// tables in constant memory (the FMA takes them as constant-bank operands: no register or move traffic, which is
// what makes the library log/exp expensive here).  log m = 2 atanh((m-1)/(m+1)) to z^15 on m in [1/sqrt2, sqrt2),
// exp r to r^11 on |r| <= ln2/2: absolute error of the exponent < 2e-14, relative error of the power likewise.
__device__ __constant__ double kLogC[7] = {2.0 / 3.0, 2.0 / 5.0, 2.0 / 7.0, 2.0 / 9.0, 2.0 / 11.0, 2.0 / 13.0, 2.0 / 15.0};
__device__ __constant__ double kExpC[10] = {1.0 / 2.0,       1.0 / 6.0,        1.0 / 24.0,        1.0 / 120.0,        1.0 / 720.0,
                                            1.0 / 5040.0,    1.0 / 40320.0,    1.0 / 362880.0,    1.0 / 3628800.0,    1.0 / 39916800.0};
__device__ __forceinline__ double pow_small(double x, double e) {
  int hi = __double2hiint(x);
  const int lo = __double2loint(x);
  int k = (hi >> 20) - 1023;
  hi = (hi & 0x000fffff) | 0x3ff00000;                 // mantissa in [1, 2)
  if (hi >= 0x3ff6a09f) hi -= 0x00100000, k += 1;      // > sqrt(2): halve
  const double m = __hiloint2double(hi, lo);
  const double z = (m - 1.0) * rcp_fast(m + 1.0);
  const double z2 = z * z;
  double p = kLogC[6];
#pragma unroll
  for (int j = 5; j >= 0; --j) p = fma(p, z2, kLogC[j]);
  const double logm = fma(z * z2, p, z + z);           // 2 z + 2 z^3/3 + ...
  const double t = e * fma(static_cast<double>(k), 0.69314718055994530942, logm);
  if (t < -700.0) return 0.0;
  const double shifter = 6755399441055744.0;           // 1.5 * 2^52: rounds to nearest integer in the low word
  const double nf = fma(t, 1.4426950408889634074, shifter);
  const int n = __double2loint(nf);
  const double nr = nf - shifter;
  double r = fma(-nr, 0.693147180369123816490, t);     // ln2 high part (33 bits)
  r = fma(-nr, 1.90821492927058770002e-10, r);         // ln2 low part
  double q = kExpC[9];
#pragma unroll
  for (int j = 8; j >= 0; --j) q = fma(q, r, kExpC[j]);
  q = fma(q * r, r, r) + 1.0;                          // 1 + r + r^2 (1/2 + r/6 + ...)
  return __hiloint2double(__double2hiint(q) + (n << 20), __double2loint(q));
}

// x^k, k >= 0 integer, by binary powering
__device__ __forceinline__ double ipow_bin(double x, int k) {
  double r = 1.0;
  while (k) {
    if (k & 1) r *= x;
    x *= x;
    k >>= 1;
  }
  return r;
}

struct MaterialConsts {   // host-side reciprocals of the constant divisors (qs_material)
  double inv_Tc, inv_B0, inv_Y, inv_rho_n, hC1, qC1sq, inv_hC3;
};

// Lattice: blockIdx.y strides over radial rows (per-row geometry from rowtab), threads over iz.  Free rings: flat.
#ifndef QS_MAT_MINB
#define QS_MAT_MINB 6   // resident CTAs per SM the register budget is sized for (40 registers per thread)
#endif
#ifndef QS_MAT_WAVES
#define QS_MAT_WAVES 8   // CTAs launched per resident slot on lattices (each walks rows with that stride); 16.8 M cells:
                        // 1: 0.224 ms, 2: 0.219, 4: 0.214, 8: 0.212, 32: 0.215
#endif
template <bool FROM_ACC, bool AUX, bool EVENTS>
__global__ void __launch_bounds__(256, QS_MAT_MINB) material_kernel(MaterialParams mp, MaterialConsts k, MaterialArgs a) {
  const double two_pi = 2.0 * kPi;
  // one flat cell index for both launch shapes.  Lattice: grid.x covers the columns, blockIdx.y strides over the
  // radial rows (step = gridDim.y rows; the row index is kept for the per-row table).  Free rings: grid-stride.
  const bool lat = a.Nz > 0;
  const int ncol = lat ? a.Nz : a.N;
  const int col0 = blockIdx.x * blockDim.x + threadIdx.x;
  const unsigned wmask = __ballot_sync(0xffffffffu, col0 < ncol);   // lanes of this warp that own a column
  if (col0 >= ncol) return;
  constexpr bool ev_on = EVENTS;                        // lattice launches: uniform trips
  const int tcol = ev_on ? col0 / a.cells_per_side : 0;
  const long long N = a.N;
  const long long step = lat ? static_cast<long long>(gridDim.y) * ncol : static_cast<long long>(gridDim.x) * blockDim.x;
  const int rstep = lat ? gridDim.y : 0;
  struct In { double J, H, b0, b1, s; };
  auto load = [&](long long i) {
    In v;
    v.J = a.J[i];
    v.H = a.H[i];
    v.b0 = FROM_ACC ? a.bracc[i] : a.Br[i];
    v.b1 = FROM_ACC ? a.bzacc[i] : a.Bz[i];
    v.s = a.jc0_scale ? a.jc0_scale[i] : 1.0;
    return v;
  };
  auto cell = [&](const long long i, const int row_i, const In& cur) {
    double r, area, selfc, dM, inv_area;
    if (lat) {
      const double4 t = a.rowtab[row_i];
      r = t.x, selfc = t.y, dM = t.z, area = t.w;
      inv_area = a.inv_area;
    } else {
      r = a.r[i], area = a.area[i], selfc = a.selfcoef[i], dM = a.diagM[i];
      inv_area = rcp_fast(area);
    }
    const double J = cur.J;
    const double U = tsq_fast(cur.H, mp.C3, k.qC1sq, k.hC1, k.inv_hC3);
    const double T = sqrt_pos(U);
    double Br, Bz;
    if (FROM_ACC) {
      Br = (0.25 * kMu0) * cur.b0 * rcp_fast(r);
      Bz = (0.25 * kMu0) * cur.b1 + selfc * (area * J) + a.Bext;
      a.Br[i] = Br;
      a.Bz[i] = Bz;
    } else {
      Br = cur.b0;
      Bz = cur.b1;
    }
    const double eps = J * Bz * r * k.inv_Y;
    const double Bmag = sqrt_pos(fma(Br, Br, Bz * Bz));
    const double fT0 = fma(-T, k.inv_Tc, 1.0), fT = fT0 > 0.0 ? fT0 : 0.0;
    const double ae = fabs(eps);
    const double pw = ae > 1e-290 ? pow_small(ae, mp.eps_exp) : 0.0;    // |eps|^eps_exp
    const double fe0 = fma(-mp.eps_coef, pw, 1.0), fe = fe0 > 0.0 ? fe0 : 0.0;
    const double s = cur.s;
    // Jc = num/den and 1/Jc = den/num from one reciprocal of num den
    const double num = mp.Jc0 * s * fT * fT * fe, den = fma(Bmag, k.inv_B0, 1.0);
    double Jc = 0.0, rho, dEdJ;
    double xr = 0.0;                               // |J| / Jc of this cell (C10)
    if (num <= 0.0) {
      rho = mp.rho_n;
      dEdJ = mp.rho_n;
      if (J != 0.0) xr = __longlong_as_double(0x7ff0000000000000LL);
    } else {
      const double R = rcp_fast(num * den);
      Jc = num * num * R;
      if (J == 0.0) {
        rho = 0.0;
        dEdJ = 0.0;
      } else {
      const double invJc = den * den * R;
      const double x = fabs(J) * invJc;
      xr = x;
      double xp;
      if (mp.n_int == 20) {                       // the configs' n = 20: x^19 = x^16 x^2 x
        const double x2 = x * x, x4 = x2 * x2, x8 = x4 * x4;
        xp = (x8 * x8) * (x2 * x);
      } else {
        xp = mp.n_int > 0 ? ipow_bin(x, mp.n_int - 1) : exp((mp.n_exp - 1.0) * log(x));
      }
      // rho = rho_sc rho_n / (rho_sc + rho_n), w = rho_n / (rho_sc + rho_n); rho_sc may have overflowed: clamp
      const double rho_sc = fmin((mp.Ec * invJc) * xp, 1e290);
      const double w = mp.rho_n * rcp_fast(rho_sc + mp.rho_n);
      rho = rho_sc * w;
      dEdJ = rho * fma(mp.n_exp - 1.0, w, 1.0);
      }
    }
    const double E = rho * J;
    a.E[i] = E;
    a.Q[i] = E * J;
    if (AUX) {
      a.dEdJ[i] = dEdJ;
      a.Jc[i] = Jc;
      a.rho[i] = rho;
    }
    if (ev_on) {   // per-turn max |J|/Jc and min rho: group the lanes of a turn, two 32-bit reductions per 64-bit key
      const int turn = a.rowturn ? a.rowturn[row_i] + tcol : a.turn_id[i];
      // common case: the whole warp lies in one turn (n >= 32 or aligned); else group the lanes by turn
      const int t0 = __shfl_sync(wmask, turn, __ffs(wmask) - 1);
      const unsigned grp = __all_sync(wmask, turn == t0) ? wmask : __match_any_sync(wmask, turn);
      const unsigned long long xb = static_cast<unsigned long long>(__double_as_longlong(xr));
      const unsigned long long rb = ~static_cast<unsigned long long>(__double_as_longlong(rho));   // min -> max of the complement
      const unsigned xh = __reduce_max_sync(grp, static_cast<unsigned>(xb >> 32));
      const unsigned xl = __reduce_max_sync(grp, static_cast<unsigned>(xb >> 32) == xh ? static_cast<unsigned>(xb) : 0u);
      const unsigned rh = __reduce_max_sync(grp, static_cast<unsigned>(rb >> 32));
      const unsigned rl = __reduce_max_sync(grp, static_cast<unsigned>(rb >> 32) == rh ? static_cast<unsigned>(rb) : 0u);
      if ((threadIdx.x & 31) == __ffs(grp) - 1) {
        atomicMax(a.xmax_bits + turn, (static_cast<unsigned long long>(xh) << 32) | xl);
        atomicMin(a.rmin_bits + turn, ~((static_cast<unsigned long long>(rh) << 32) | rl));
      }
    }
    const double shift = mp.theta * a.dt * (two_pi * r * dEdJ * inv_area);
    a.shift[i] = shift;
    a.Hd[i] = dM + shift;
  };
  // No software pipeline: one cell per trip, memory latency is covered by occupancy (40 registers, 6 CTAs = 48 warps per
  // SM).  Measured on 16.8 M cells (B200, material_kernel<0,0,1>): this loop at 6 / 7 / 8 CTAs per SM 0.219 ms, at 5
  // (44 registers) 0.229 ms; inputs prefetched one cell ahead at 64 registers 0.248 ms; two cells ahead (64 registers,
  // 68 B of spills) 0.260 ms, at 80 registers 0.287 ms.
  long long i = (lat ? static_cast<long long>(blockIdx.y) * ncol : 0) + col0;
  int row = lat ? blockIdx.y : 0;
  for (; i < N; i += step, row += rstep) cell(i, row, load(i));
}

__global__ void rowtab_kernel(int Nr, int Nz, const double* __restrict__ r, const double* __restrict__ selfcoef,
                              const double* __restrict__ diagM, const double* __restrict__ area,
                              double4* __restrict__ rowtab) {
  const int ir = blockIdx.x * blockDim.x + threadIdx.x;
  if (ir >= Nr) return;
  const long long c = static_cast<long long>(ir) * Nz;
  rowtab[ir] = make_double4(r[c], selfcoef[c], diagM[c], area[c]);
}

__global__ void enthalpy_kernel(int n, double C3, double C1, const double* __restrict__ T, double* __restrict__ H) {
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
    const double t = T[i], t2 = t * t;
    H[i] = 0.25 * C3 * t2 * t2 + 0.5 * C1 * t2;
  }
}
__global__ void temperature_kernel(int n, double C3, double C1, const double* __restrict__ H, double* __restrict__ T) {
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x)
    T[i] = sqrt(tsq_of_H(H[i], C3, C1));
}

// ---- K6: one explicit sub-step (C9) -----------------------------------------------------------------------------
// Marching stencil without shared-memory tiles: a warp owns 30 consecutive columns (iz) plus one halo lane on each
// side and marches along r over a strip of rows, keeping T^2 of the previous, current and next row in registers
// (one square root per cell and row; the Kirchhoff flux needs only T^2); the z-neighbours come from the adjacent
// lanes by shuffles.  Conductivities, face areas and the cell volume are folded into per-row / per-column
// coefficient tables (LatticeParams), so a cell update is 4 differences, 4 multiply-adds, the source and the
// update: read H, Q and write H = 24 B per cell.
constexpr int kHeatLanes = 30;           // owner lanes per warp (lanes 0 and 31 carry the halo columns)
constexpr int kHeatCols = 2 * kHeatLanes; // useful columns per warp: every lane holds two adjacent columns
constexpr int kHeatWarps = 8;
constexpr int kHeatMaxRows = 32;          // rows per strip (64: same time on a 4096 x 4096 lattice; 128 and 256, one wave: 12 % slower)

// T from T^2 (border cells only), same fast root
__device__ __forceinline__ double sqrt_fast(double a) {
  const double y0 = rsqrt_seed(a);
  const double g = a * y0;
  const double e = fma(-g, y0, 1.0);
  return fma(g * e, fma(0.375, e, 0.5), g);
}

template <bool VEC>   // VEC: Nz even, so that the column pair of a lane is 16-byte aligned in every row
__global__ void __launch_bounds__(kHeatWarps * 32, 3) heat_kernel(MaterialParams mp, LatticeParams lp, int rows_per_cta,
                                                               const double* __restrict__ Hin,
                                                               const double* __restrict__ Q, double* __restrict__ Hout,
                                                               double dtsub) {
  __shared__ double4 srow[kHeatMaxRows];               // (hr_p, hr_m, rb_r, -) of the rows of this strip
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int iz0 = 2 * ((blockIdx.x * kHeatWarps + warp) * kHeatLanes + lane - 1);
  const int r0 = blockIdx.y * rows_per_cta, r1 = min(r0 + rows_per_cta, lp.Nr);
  if (threadIdx.x < r1 - r0)
    srow[threadIdx.x] = make_double4(lp.hr_p[r0 + threadIdx.x], lp.hr_m[r0 + threadIdx.x], lp.rb_r[r0 + threadIdx.x], 0.0);
  __syncthreads();
  const bool in0 = iz0 >= 0 && iz0 < lp.Nz, in1 = iz0 + 1 >= 0 && iz0 + 1 < lp.Nz;
  const bool own = lane >= 1 && lane <= kHeatLanes;
  const bool own0 = own && in0, own1 = own && in1;
  const double C3 = mp.C3, qC1sq = 0.25 * mp.C1 * mp.C1, hC1 = 0.5 * mp.C1, inv_hC3 = 2.0 / mp.C3;
  const double zp0 = in0 ? lp.hz_p[iz0] : 0.0, zm0 = in0 ? lp.hz_m[iz0] : 0.0, zb0 = in0 ? lp.rb_z[iz0] : 0.0;
  const double zp1 = in1 ? lp.hz_p[iz0 + 1] : 0.0, zm1 = in1 ? lp.hz_m[iz0 + 1] : 0.0, zb1 = in1 ? lp.rb_z[iz0 + 1] : 0.0;
  // lanes (partly) outside the pack read a clamped column pair and are ignored
  const int izc = max(0, min(iz0, lp.Nz - 2 + (lp.Nz & 1)));
  const bool pair_ok = in0 && in1;
  const long long Nz = lp.Nz;
  const double* hn = Hin + static_cast<long long>(r0) * Nz + izc;     // walks one row ahead of the update
  const double* q = Q + static_cast<long long>(r0) * Nz + izc;
  double* o = Hout + static_cast<long long>(r0) * Nz + izc;
  auto load2 = [&](const double* ptr) -> double2 {
    if (VEC) return *reinterpret_cast<const double2*>(ptr);
    double2 v;
    v.x = ptr[0];
    v.y = pair_ok ? ptr[1] : ptr[0];
    return v;
  };
  double2 Up = make_double2(0.0, 0.0);
  if (r0 > 0) {
    const double2 h = load2(hn - Nz);
    Up = make_double2(tsq_fast(h.x, C3, qC1sq, hC1, inv_hC3), tsq_fast(h.y, C3, qC1sq, hC1, inv_hC3));
  }
  double2 Hc = load2(hn);
  double2 Uc = make_double2(tsq_fast(Hc.x, C3, qC1sq, hC1, inv_hC3), tsq_fast(Hc.y, C3, qC1sq, hC1, inv_hC3));
  const int last = lp.Nr - 1;
  // software pipeline: the enthalpy row two ahead and the source row one ahead are in flight while a row is updated
  // (past the last row of the pack the pointer stays on the last row: its coefficient is 0)
  if (r0 < last) hn += Nz;
  double2 Hn = load2(hn);
  if (r0 + 1 < last) hn += Nz;
  double2 Hn2 = load2(hn);
  double2 qc = load2(q);
  if (r0 + 1 < r1) q += Nz;
  double2 qn = load2(q);
  const bool zborder = (zb0 != 0.0) || (zb1 != 0.0);
  for (int ir = r0; ir < r1; ++ir) {
    if (ir + 2 < last) hn += Nz;
    const double2 Hn3 = load2(hn);                     // enthalpy row ir + 3 (clamped to the last row)
    if (ir + 2 < r1) q += Nz;
    const double2 qn2 = load2(q);                      // source row ir + 2 (clamped to the strip)
    const double2 Un = make_double2(tsq_fast(Hn.x, C3, qC1sq, hC1, inv_hC3), tsq_fast(Hn.y, C3, qC1sq, hC1, inv_hC3));
    const double Ul = __shfl_up_sync(0xffffffffu, Uc.y, 1), Ur = __shfl_down_sync(0xffffffffu, Uc.x, 1);
    if (own0) {
      const double4 rc = srow[ir - r0];
      double a0 = fma(rc.x, Un.x - Uc.x, qc.x), a1 = fma(rc.x, Un.y - Uc.y, qc.y);
      a0 = fma(rc.y, Up.x - Uc.x, a0);
      a1 = fma(rc.y, Up.y - Uc.y, a1);
      const double dzc = Uc.y - Uc.x;
      a0 = fma(zp0, dzc, a0);
      a1 = fma(-zm1, dzc, a1);
      a0 = fma(zm0, Ul - Uc.x, a0);
      a1 = fma(zp1, Ur - Uc.y, a1);
      if (rc.z != 0.0 || zborder) {                    // Robin borders of the winding pack (rare: rb = 0 inside)
        a0 = fma(-(rc.z + zb0), sqrt_fast(Uc.x) - lp.T_bath, a0);
        a1 = fma(-(rc.z + zb1), sqrt_fast(Uc.y) - lp.T_bath, a1);
      }
      const double2 out = make_double2(fma(dtsub, a0, Hc.x), fma(dtsub, a1, Hc.y));
      if (VEC) {
        *reinterpret_cast<double2*>(o) = out;
      } else {
        o[0] = out.x;
        if (own1) o[1] = out.y;
      }
    }
    Up = Uc;
    Uc = Un;
    Hc = Hn;
    Hn = Hn2;
    Hn2 = Hn3;
    qc = qn;
    qn = qn2;
    o += Nz;
  }
}

// ---- K6, TMA-pipelined variant (Nz even): same marching scheme, but every warp streams its 512-byte row segments
// of H and Q through a ring of kHeatStages shared-memory stages with TMA bulk copies (cp.async.bulk + mbarrier,
// issued by lane 0), so that kHeatStages rows per warp are in flight whatever the register budget.
#ifndef QS_HEAT_STAGES
#define QS_HEAT_STAGES 8
#endif
#ifndef QS_HEAT_MINB
#define QS_HEAT_MINB 3
#endif
constexpr int kHeatStages = QS_HEAT_STAGES;
constexpr int kHeatMinB = QS_HEAT_MINB;   // resident CTAs per SM the registers and the shared-memory ring are sized for
struct HeatStage {
  double h[64];
  double q[64];
};
struct HeatSmem {
  HeatStage st[kHeatWarps][kHeatStages];
  double4 srow[kHeatMaxRows];
  uint64_t bar[kHeatWarps][kHeatStages];
};

__global__ void __launch_bounds__(kHeatWarps * 32, kHeatMinB) heat_tma_kernel(MaterialParams mp, LatticeParams lp,
                                                                      int rows_per_cta, const double* __restrict__ Hin,
                                                                      const double* __restrict__ Q,
                                                                      double* __restrict__ Hout, double dtsub) {
  extern __shared__ __align__(128) unsigned char heat_smem_raw[];
  HeatSmem& sm = *reinterpret_cast<HeatSmem*>(heat_smem_raw);
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int r0 = blockIdx.y * rows_per_cta, r1 = min(r0 + rows_per_cta, lp.Nr), nrows = r1 - r0;
  if (threadIdx.x < nrows)
    sm.srow[threadIdx.x] = make_double4(lp.hr_p[r0 + threadIdx.x], lp.hr_m[r0 + threadIdx.x], lp.rb_r[r0 + threadIdx.x], 0.0);
  if (threadIdx.x < kHeatWarps * kHeatStages) mbar_init(&sm.bar[threadIdx.x / kHeatStages][threadIdx.x % kHeatStages], 1);
  asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  __syncthreads();
  const int col_lo = (blockIdx.x * kHeatWarps + warp) * kHeatCols - 2;      // first column of the warp's 64-wide window
  const int cs = max(col_lo, 0), ce = min(col_lo + 64, lp.Nz);             // clipped to the pack
  if (col_lo + 2 >= lp.Nz) return;                                          // no owned column in this warp
  const uint32_t seg_bytes = static_cast<uint32_t>(ce - cs) * 8u;
  const int soff = cs - col_lo;
  const int iz0 = col_lo + 2 * lane;
  const bool in0 = iz0 >= 0 && iz0 < lp.Nz, in1 = iz0 + 1 >= 0 && iz0 + 1 < lp.Nz;
  const bool own0 = lane >= 1 && lane <= kHeatLanes && in0;
  const double C3 = mp.C3, qC1sq = 0.25 * mp.C1 * mp.C1, hC1 = 0.5 * mp.C1, inv_hC3 = 2.0 / mp.C3;
  const double zp0 = in0 ? lp.hz_p[iz0] : 0.0, zm0 = in0 ? lp.hz_m[iz0] : 0.0, zb0 = in0 ? lp.rb_z[iz0] : 0.0;
  const double zp1 = in1 ? lp.hz_p[iz0 + 1] : 0.0, zm1 = in1 ? lp.hz_m[iz0 + 1] : 0.0, zb1 = in1 ? lp.rb_z[iz0 + 1] : 0.0;
  const bool zborder = (zb0 != 0.0) || (zb1 != 0.0);
  const long long Nz = lp.Nz;
  // stage t holds row g = r0 - 1 + t of H (0 <= t <= nrows + 1) and, for 1 <= t <= nrows, of Q
  const int T_last = nrows + 1;
  auto row_ok = [&](int t) { const int g = r0 - 1 + t; return g >= 0 && g < lp.Nr; };
  // fill(t) is called for t = 0, 1, 2, ... in this order: the element offset of row t is carried, not recomputed
  long long fill_off = static_cast<long long>(r0 - 1) * Nz + cs;
  auto fill = [&](int t) {
    const long long off = fill_off;
    fill_off += Nz;
    if (lane != 0 || t > T_last) return;
    HeatStage& s = sm.st[warp][t % kHeatStages];
    uint64_t* b = &sm.bar[warp][t % kHeatStages];
    if (!row_ok(t)) {          // a row outside the pack: complete the phase empty, the parity sequence stays regular
      mbar_arrive(b);
      return;
    }
    const bool needq = t >= 1 && t <= nrows;
    mbar_expect_tx(b, needq ? 2u * seg_bytes : seg_bytes);
    bulk_g2s(&s.h[soff], Hin + off, seg_bytes, b);
    if (needq) bulk_g2s(&s.q[soff], Q + off, seg_bytes, b);
  };
  // the column slots of this warp's window that no bulk copy ever writes (outside the winding pack) hold zeros for the
  // whole kernel, so the per-row reads need no masks
#pragma unroll
  for (int t = 0; t < kHeatStages; ++t) {
    HeatStage& s = sm.st[warp][t];
    if (!in0) s.h[2 * lane] = 0.0, s.q[2 * lane] = 0.0;
    if (!in1) s.h[2 * lane + 1] = 0.0, s.q[2 * lane + 1] = 0.0;
  }
  __syncwarp();
#pragma unroll
  for (int t = 0; t < kHeatStages; ++t) fill(t);
  // A row's stage is refilled only after the row has been the CENTRE row of an update, so H and Q of the centre row are
  // read from shared memory where they are used (two LDS.128) instead of riding through two register rotations.
  auto wait_h = [&](int t) {                            // waits for stage t, returns this lane's column pair of H
    mbar_wait(&sm.bar[warp][t % kHeatStages], (t / kHeatStages) & 1);
    if (!row_ok(t)) return make_double2(0.0, 0.0);
    return *reinterpret_cast<const double2*>(&sm.st[warp][t % kHeatStages].h[2 * lane]);
  };
  {
    double2 h = wait_h(0);
    double2 Up = make_double2(0.0, 0.0);
    if (r0 > 0) Up = make_double2(tsq_fast(h.x, C3, qC1sq, hC1, inv_hC3), tsq_fast(h.y, C3, qC1sq, hC1, inv_hC3));
    __syncwarp();
    fill(kHeatStages);                                  // row -1 is never a centre row: its stage is free again
    h = wait_h(1);
    double2 Uc = make_double2(tsq_fast(h.x, C3, qC1sq, hC1, inv_hC3), tsq_fast(h.y, C3, qC1sq, hC1, inv_hC3));
    double* o = Hout + static_cast<long long>(r0) * Nz + max(iz0, 0);
    for (int k = 0; k < nrows; ++k) {
      const double2 Hn = wait_h(k + 2);
      const double2 Un = make_double2(tsq_fast(Hn.x, C3, qC1sq, hC1, inv_hC3), tsq_fast(Hn.y, C3, qC1sq, hC1, inv_hC3));
      const double Ul = __shfl_up_sync(0xffffffffu, Uc.y, 1), Ur = __shfl_down_sync(0xffffffffu, Uc.x, 1);
      if (own0) {
        const HeatStage& sc = sm.st[warp][(k + 1) % kHeatStages];
        const double2 Hc = *reinterpret_cast<const double2*>(&sc.h[2 * lane]);
        const double2 qc = *reinterpret_cast<const double2*>(&sc.q[2 * lane]);
        const double4 rc = sm.srow[k];
        double a0 = fma(rc.x, Un.x - Uc.x, qc.x), a1 = fma(rc.x, Un.y - Uc.y, qc.y);
        a0 = fma(rc.y, Up.x - Uc.x, a0);
        a1 = fma(rc.y, Up.y - Uc.y, a1);
        const double dzc = Uc.y - Uc.x;
        a0 = fma(zp0, dzc, a0);
        a1 = fma(-zm1, dzc, a1);
        a0 = fma(zm0, Ul - Uc.x, a0);
        a1 = fma(zp1, Ur - Uc.y, a1);
        if (rc.z != 0.0 || zborder) {                    // Robin borders of the winding pack (rare: rb = 0 inside)
          a0 = fma(-(rc.z + zb0), sqrt_fast(Uc.x) - lp.T_bath, a0);
          a1 = fma(-(rc.z + zb1), sqrt_fast(Uc.y) - lp.T_bath, a1);
        }
        *reinterpret_cast<double2*>(o) = make_double2(fma(dtsub, a0, Hc.x), fma(dtsub, a1, Hc.y));
      }
      Up = Uc;
      Uc = Un;
      o += Nz;
      __syncwarp();                                     // every lane is done with the centre row's stage
      fill(k + 1 + kHeatStages);
    }
  }
}

// ---- K6, in-SM variant for small lattices (N <= kHeatSmallMax cells): ALL m sub-steps of a step in one launch.
// One CTA of 1024 threads keeps the enthalpy of its cells in registers and T^2 of the whole lattice in shared
// memory; a sub-step is "publish T^2, barrier, update H, barrier".  Replaces m launches (144 per step at config 1)
// by one; the arithmetic per cell and sub-step is the one of the marching kernel.
constexpr int kHeatSmallThreads = 1024;
constexpr int kHeatSmallPer = 4;
constexpr int kHeatSmallMax = kHeatSmallThreads * kHeatSmallPer;   // 4096 cells = 32 KB of T^2 (config 1: 64 x 64)

__global__ void __launch_bounds__(kHeatSmallThreads, 1) heat_small_kernel(MaterialParams mp, LatticeParams lp, int m,
                                                                          const double* __restrict__ Hin,
                                                                          const double* __restrict__ Q,
                                                                          double* __restrict__ Hout, double dtsub) {
  extern __shared__ __align__(16) double hs_smem[];
  const int N = lp.Nr * lp.Nz, Nz = lp.Nz, Nr = lp.Nr;
  double* Us = hs_smem;                                   // [N] T^2
  double* crp = Us + N;                                   // per-row coefficients [Nr] x 3, per-column [Nz] x 3
  double* crm = crp + Nr;
  double* crb = crm + Nr;
  double* czp = crb + Nr;
  double* czm = czp + Nz;
  double* czb = czm + Nz;
  for (int i = threadIdx.x; i < Nr; i += blockDim.x) crp[i] = lp.hr_p[i], crm[i] = lp.hr_m[i], crb[i] = lp.rb_r[i];
  for (int i = threadIdx.x; i < Nz; i += blockDim.x) czp[i] = lp.hz_p[i], czm[i] = lp.hz_m[i], czb[i] = lp.rb_z[i];
  const double C3 = mp.C3, qC1sq = 0.25 * mp.C1 * mp.C1, hC1 = 0.5 * mp.C1, inv_hC3 = 2.0 / mp.C3;
  double H[kHeatSmallPer], q[kHeatSmallPer];
  int ir[kHeatSmallPer], iz[kHeatSmallPer];
#pragma unroll
  for (int k = 0; k < kHeatSmallPer; ++k) {
    const int i = threadIdx.x + k * kHeatSmallThreads;
    H[k] = q[k] = 0.0;
    ir[k] = iz[k] = 0;
    if (i < N) {
      ir[k] = i / Nz, iz[k] = i - ir[k] * Nz;
      H[k] = Hin[i];
      q[k] = Q[i];
    }
  }
  for (int s = 0; s < m; ++s) {
#pragma unroll
    for (int k = 0; k < kHeatSmallPer; ++k) {
      const int i = threadIdx.x + k * kHeatSmallThreads;
      if (i < N) Us[i] = tsq_fast(H[k], C3, qC1sq, hC1, inv_hC3);
    }
    __syncthreads();
#pragma unroll
    for (int k = 0; k < kHeatSmallPer; ++k) {
      const int i = threadIdx.x + k * kHeatSmallThreads;
      if (i < N) {
        const double u = Us[i];
        // neighbours outside the pack have coefficient 0: read the cell itself instead
        const double un = ir[k] + 1 < Nr ? Us[i + Nz] : u, up = ir[k] > 0 ? Us[i - Nz] : u;
        const double ur = iz[k] + 1 < Nz ? Us[i + 1] : u, ul = iz[k] > 0 ? Us[i - 1] : u;
        double a = fma(crp[ir[k]], un - u, q[k]);
        a = fma(crm[ir[k]], up - u, a);
        a = fma(czp[iz[k]], ur - u, a);
        a = fma(czm[iz[k]], ul - u, a);
        const double rb = crb[ir[k]] + czb[iz[k]];
        if (rb != 0.0) a = fma(-rb, sqrt_fast(u) - lp.T_bath, a);
        H[k] = fma(dtsub, a, H[k]);
      }
    }
    __syncthreads();
  }
#pragma unroll
  for (int k = 0; k < kHeatSmallPer; ++k) {
    const int i = threadIdx.x + k * kHeatSmallThreads;
    if (i < N) Hout[i] = H[k];
  }
}

// ---- K6, cluster variant of the in-SM kernel: the same "all m sub-steps in one launch", spread over a thread-block
// CLUSTER of 8 CTAs (8 SMs instead of one: the single-CTA kernel is FP64-bound on its SM, 2 us per sub-step at config 1).
// CTA c owns a band of rows_per rows; T^2 of its band lives in its shared memory in two buffers (sub-step parity), the
// rows just above and below the band are read from the neighbour CTAs' shared memory (DSMEM), and ONE cluster barrier
// per sub-step separates "publish" from "read": a CTA overwrites buffer b again only two sub-steps later, after a
// barrier that every reader of b has passed.  Same arithmetic per cell, in the same order, as heat_small_kernel.
constexpr int kHeatClusterCtas = 8;
constexpr int kHeatClusterThreads = 512;
constexpr int kHeatClusterPer = 2;                                  // cells per thread: bands of <= 1024 cells

__global__ void __launch_bounds__(kHeatClusterThreads, 1) heat_cluster_kernel(MaterialParams mp, LatticeParams lp, int m,
                                                                              int rows_per, const double* __restrict__ Hin,
                                                                              const double* __restrict__ Q,
                                                                              double* __restrict__ Hout, double dtsub) {
  extern __shared__ __align__(16) double hc_smem[];
  namespace cg = cooperative_groups;
  cg::cluster_group cluster = cg::this_cluster();
  const int rank = static_cast<int>(cluster.block_rank());
  const int Nz = lp.Nz, Nr = lp.Nr;
  const int band = rows_per * Nz;                                   // cells of a full band (buffer stride)
  const int r0 = rank * rows_per, r1 = min(r0 + rows_per, Nr);      // this CTA's rows [r0, r1): may be empty
  const int cells = max(r1 - r0, 0) * Nz;
  double* U[2] = {hc_smem, hc_smem + band};                         // T^2 of the band, by sub-step parity
  double* crp = hc_smem + 2 * band;                                 // per-row coefficients of the band x 3, per-column x 3
  double* crm = crp + rows_per;
  double* crb = crm + rows_per;
  double* czp = crb + rows_per;
  double* czm = czp + Nz;
  double* czb = czm + Nz;
  for (int i = threadIdx.x; i < r1 - r0; i += blockDim.x)
    crp[i] = lp.hr_p[r0 + i], crm[i] = lp.hr_m[r0 + i], crb[i] = lp.rb_r[r0 + i];
  for (int i = threadIdx.x; i < Nz; i += blockDim.x) czp[i] = lp.hz_p[i], czm[i] = lp.hz_m[i], czb[i] = lp.rb_z[i];
  // the neighbours' buffers: the band above ends with row r0 - 1 (its last row), the band below starts with row r1
  const bool has_up = r0 > 0 && cells > 0, has_dn = r1 < Nr && cells > 0;
  const double* Uup[2] = {nullptr, nullptr};
  const double* Udn[2] = {nullptr, nullptr};
  if (has_up) {
    double* base = cluster.map_shared_rank(hc_smem, rank - 1);
    Uup[0] = base + (rows_per - 1) * Nz, Uup[1] = base + band + (rows_per - 1) * Nz;
  }
  if (has_dn) {
    double* base = cluster.map_shared_rank(hc_smem, rank + 1);
    Udn[0] = base, Udn[1] = base + band;
  }
  const double C3 = mp.C3, qC1sq = 0.25 * mp.C1 * mp.C1, hC1 = 0.5 * mp.C1, inv_hC3 = 2.0 / mp.C3;
  double H[kHeatClusterPer], q[kHeatClusterPer];
  int lr[kHeatClusterPer], iz[kHeatClusterPer];
#pragma unroll
  for (int k = 0; k < kHeatClusterPer; ++k) {
    const int i = threadIdx.x + k * kHeatClusterThreads;
    H[k] = q[k] = 0.0;
    lr[k] = iz[k] = 0;
    if (i < cells) {
      lr[k] = i / Nz, iz[k] = i - lr[k] * Nz;
      H[k] = Hin[r0 * Nz + i];
      q[k] = Q[r0 * Nz + i];
    }
  }
  for (int s = 0; s < m; ++s) {
    double* Us = U[s & 1];
#pragma unroll
    for (int k = 0; k < kHeatClusterPer; ++k) {
      const int i = threadIdx.x + k * kHeatClusterThreads;
      if (i < cells) Us[i] = tsq_fast(H[k], C3, qC1sq, hC1, inv_hC3);
    }
    cluster.sync();
#pragma unroll
    for (int k = 0; k < kHeatClusterPer; ++k) {
      const int i = threadIdx.x + k * kHeatClusterThreads;
      if (i < cells) {
        const double u = Us[i];
        const int gr = r0 + lr[k];
        // neighbours outside the pack have coefficient 0: read the cell itself instead
        double un = u, up = u;
        if (gr + 1 < Nr) un = gr + 1 < r1 ? Us[i + Nz] : Udn[s & 1][iz[k]];
        if (gr > 0) up = lr[k] > 0 ? Us[i - Nz] : Uup[s & 1][iz[k]];
        const double ur = iz[k] + 1 < Nz ? Us[i + 1] : u, ul = iz[k] > 0 ? Us[i - 1] : u;
        double a = fma(crp[lr[k]], un - u, q[k]);
        a = fma(crm[lr[k]], up - u, a);
        a = fma(czp[iz[k]], ur - u, a);
        a = fma(czm[iz[k]], ul - u, a);
        const double rb = crb[lr[k]] + czb[iz[k]];
        if (rb != 0.0) a = fma(-rb, sqrt_fast(u) - lp.T_bath, a);
        H[k] = fma(dtsub, a, H[k]);
      }
    }
  }
  cluster.sync();                                                  // nobody leaves while a neighbour may still read its band
#pragma unroll
  for (int k = 0; k < kHeatClusterPer; ++k) {
    const int i = threadIdx.x + k * kHeatClusterThreads;
    if (i < cells) Hout[r0 * Nz + i] = H[k];
  }
}

// ---- K6, temporally blocked variant: up to kHbHalo sub-steps per launch.  A CTA owns a TILE x TILE block of cells,
// loads it with a halo of kHbHalo cells on every side (H, Q once from HBM / L2), keeps H and Q of its cells in
// registers and T^2 of the region in shared memory (two buffers, one barrier per sub-step), advances the WHOLE region
// msub <= kHbHalo sub-steps - the error of the missing outer neighbours moves inward one cell per sub-step and never
// reaches the tile - and writes the tile.  Per step of m sub-steps the enthalpy and the source cross HBM m/4 times
// instead of m times (the algorithmic minimum becomes 24 B per cell per launch group).
constexpr int kHbHalo = 4;
template <int TILE, int THREADS>
__global__ void __launch_bounds__(THREADS) heat_block_kernel(MaterialParams mp, LatticeParams lp, int msub,
                                                             const double* __restrict__ Hin, const double* __restrict__ Q,
                                                             double* __restrict__ Hout, double dtsub) {
  constexpr int W = TILE + 2 * kHbHalo, NC = W * W, PER = (NC + THREADS - 1) / THREADS;
  extern __shared__ __align__(16) double hb_smem[];
  double* U0 = hb_smem;                 // [NC] T^2, ping
  double* U1 = U0 + NC;                 // [NC] pong
  double* crp = U1 + NC;                // [W] x 3 row coefficients, [W] x 3 column coefficients (0 outside the pack)
  double* crm = crp + W;
  double* crb = crm + W;
  double* czp = crb + W;
  double* czm = czp + W;
  double* czb = czm + W;
  const int Nr = lp.Nr, Nz = lp.Nz;
  const int r0 = blockIdx.y * TILE - kHbHalo, c0 = blockIdx.x * TILE - kHbHalo;
  for (int i = threadIdx.x; i < W; i += THREADS) {
    const int gr = r0 + i, gc = c0 + i;
    const bool rin = gr >= 0 && gr < Nr, cin = gc >= 0 && gc < Nz;
    crp[i] = rin ? lp.hr_p[gr] : 0.0, crm[i] = rin ? lp.hr_m[gr] : 0.0, crb[i] = rin ? lp.rb_r[gr] : 0.0;
    czp[i] = cin ? lp.hz_p[gc] : 0.0, czm[i] = cin ? lp.hz_m[gc] : 0.0, czb[i] = cin ? lp.rb_z[gc] : 0.0;
  }
  const double C3 = mp.C3, qC1sq = 0.25 * mp.C1 * mp.C1, hC1 = 0.5 * mp.C1, inv_hC3 = 2.0 / mp.C3;
  double H[PER], q[PER];
#pragma unroll
  for (int k = 0; k < PER; ++k) {
    const int idx = threadIdx.x + k * THREADS;
    H[k] = q[k] = 0.0;
    if (idx < NC) {
      const int row = idx / W, col = idx - row * W;
      const int gr = r0 + row, gc = c0 + col;
      if (gr >= 0 && gr < Nr && gc >= 0 && gc < Nz) {
        const long long g = static_cast<long long>(gr) * Nz + gc;
        H[k] = Hin[g];
        q[k] = Q[g];
      }
      U0[idx] = tsq_fast(H[k], C3, qC1sq, hC1, inv_hC3);
    }
  }
  __syncthreads();
  for (int s = 0; s < msub; ++s) {
    const double* Uc = (s & 1) ? U1 : U0;
    double* Un = (s & 1) ? U0 : U1;
#pragma unroll
    for (int k = 0; k < PER; ++k) {
      const int idx = threadIdx.x + k * THREADS;
      if (idx < NC) {
        const int row = idx / W, col = idx - row * W;
        const double u = Uc[idx];
        // neighbours outside the region: the cell itself (pack borders have coefficient 0; region borders are halo)
        const double un = row + 1 < W ? Uc[idx + W] : u, up = row > 0 ? Uc[idx - W] : u;
        const double ur = col + 1 < W ? Uc[idx + 1] : u, ul = col > 0 ? Uc[idx - 1] : u;
        double a = fma(crp[row], un - u, q[k]);
        a = fma(crm[row], up - u, a);
        a = fma(czp[col], ur - u, a);
        a = fma(czm[col], ul - u, a);
        const double rb = crb[row] + czb[col];
        // (u > 0: region cells outside the pack hold T^2 = 0 up to rounding and must stay finite - a NaN there would
        // reach the pack through 0 * NaN)
        if (rb != 0.0 && u > 0.0) a = fma(-rb, sqrt_fast(u) - lp.T_bath, a);
        H[k] = fma(dtsub, a, H[k]);
        if (s + 1 < msub) Un[idx] = tsq_fast(H[k], C3, qC1sq, hC1, inv_hC3);
      }
    }
    __syncthreads();
  }
#pragma unroll
  for (int k = 0; k < PER; ++k) {
    const int idx = threadIdx.x + k * THREADS;
    if (idx < NC) {
      const int row = idx / W, col = idx - row * W;
      const int gr = r0 + row, gc = c0 + col;
      if (row >= kHbHalo && row < kHbHalo + TILE && col >= kHbHalo && col < kHbHalo + TILE && gr < Nr && gc < Nz)
        Hout[static_cast<long long>(gr) * Nz + gc] = H[k];
    }
  }
}
constexpr size_t heat_block_smem(int tile) {
  return sizeof(double) * (2 * static_cast<size_t>(tile + 2 * kHbHalo) * (tile + 2 * kHbHalo) + 6 * (tile + 2 * kHbHalo));
}

// ---- K7 ---------------------------------------------------------------------------------------------------
// One CTA per constraint group (32 .. 256 threads: the power of two next to the group's cell count).
constexpr int kEventBlockMax = 256;
__global__ void __launch_bounds__(kEventBlockMax) events_kernel(int n_turns, const int* __restrict__ ptr,
                                                                const int* __restrict__ idx, MaterialParams mp,
                                                                EventArgs e, Scalars* sc) {
  __shared__ double red[5][kEventBlockMax / 32];
  __shared__ int redbad[kEventBlockMax / 32];
  const int w = blockIdx.x, lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nw = blockDim.x >> 5;
  double tsq = 0.0, esum = 0.0, qv = 0.0, pmax = 0.0, dj = 0.0;
  int bad = 0;
  for (int k = ptr[w] + threadIdx.x; k < ptr[w + 1]; k += blockDim.x) {
    const int i = idx[k];
    const double t2 = tsq_of_H(e.H[i], mp.C3, mp.C1);
    tsq = fmax(tsq, t2);
    esum += fabs(e.E[i]);
    const double q = e.Q[i];
    qv = fma(q, 2.0 * kPi * e.r[i] * e.area[i], qv);       // Joule power of the wire [W]
    pmax = fmax(pmax, q);
    if (e.J) {   // step statistics folded into this pass (every cell belongs to one group)
      const double Ji = e.J[i];
      dj = fmax(dj, fabs(Ji - e.Jold[i]));
      if (!isfinite(Ji) || !isfinite(t2) || !(t2 > 0.0)) bad = 1;
    }
  }
  tsq = warp_max(tsq);
  esum = warp_sum(esum);
  qv = warp_sum(qv);
  pmax = warp_max(pmax);
  dj = warp_max(dj);
  bad = __any_sync(0xffffffffu, bad);
  if (nw > 1) {   // combine the warps of the CTA
    if (lane == 0) red[0][wid] = tsq, red[1][wid] = esum, red[2][wid] = qv, red[3][wid] = pmax, red[4][wid] = dj, redbad[wid] = bad;
    __syncthreads();
    if (threadIdx.x != 0) return;
    for (int k = 1; k < nw; ++k) {
      tsq = fmax(tsq, red[0][k]);
      esum += red[1][k];
      qv += red[2][k];
      pmax = fmax(pmax, red[3][k]);
      dj = fmax(dj, red[4][k]);
      bad |= redbad[k];
    }
  }
  if (e.J) {
    if (threadIdx.x == 0) {
      if (dj > 0.0 && isfinite(dj)) atomic_max_pos(&sc->djmax, dj);
      if (tsq > 0.0 && isfinite(tsq)) atomic_max_pos(&sc->tmax, sqrt(tsq));
      atomicAdd(&sc->joule, qv);
      if (bad) atomicOr(&sc->nonfinite, 1);
    }
  }
  const double xmax = __longlong_as_double(static_cast<long long>(e.xmax_bits[w]));
  const double rmin = __longlong_as_double(static_cast<long long>(e.rmin_bits[w])) / mp.rho_n;
  if (threadIdx.x != 0) return;
  const double Tmax = sqrt(tsq);
  const double ebar = esum / static_cast<double>(ptr[w + 1] - ptr[w]);
  int fl = 0;
  if (Tmax > mp.T_fluxjump) fl |= 1;
  if (e.have_prev && (ebar - e.ebar_prev[w]) / e.dt > mp.dEdt_spike) fl |= 2;
  if (xmax > 1.0) fl |= 4;
  if (Tmax > mp.Tc) fl |= 8;
  if (rmin > 0.95) fl |= 16;
  const int old = e.flags[w];
  if ((fl & 3) && !(old & 3)) e.count[w] += 1;
  const bool first = fl && e.t_first[w] < 0.0;
  if (first) e.t_first[w] = e.t_new;
  {  // per-wire statistics (f3; PAPER.md:107 T_max, P_max, Q_FJ; PAPER.md:119-121 Q_q, P_q, T_q at the quench time)
    double* W = e.wire;
    const int nt = n_turns;
    const double dE = e.dt * qv;
    double Ej = W[w];
    if (first) W[8 * nt + w] = Ej;                         // energy before the step of the first event
    Ej += dE;
    W[w] = Ej;
    if (fl & 7) W[nt + w] += dE;                           // Q_FJ: while a flux-jump flag is set
    W[2 * nt + w] = fmax(W[2 * nt + w], pmax);
    W[3 * nt + w] = fmax(W[3 * nt + w], Tmax);
    if ((fl & 24) && W[4 * nt + w] < 0.0) {                // first step with a quench flag
      W[4 * nt + w] = e.t_new;
      W[5 * nt + w] = Tmax;
      W[6 * nt + w] = pmax;
      W[7 * nt + w] = Ej - W[8 * nt + w];
    }
  }
  int ret = 0;
  if ((fl & 7) && !(old & 7)) ret |= 1;
  if (fl & 24) ret |= 2;
  if (ret) atomicOr(&sc->event_or, ret);
  e.flags[w] = fl;
  e.ebar_prev[w] = ebar;
}

__global__ void stats_kernel(int n, double C3, double C1, const double* __restrict__ J,
                             const double* __restrict__ Jold, const double* __restrict__ H,
                             const double* __restrict__ Q, const double* __restrict__ r,
                             const double* __restrict__ area, Scalars* sc) {
  double tsq = 0.0, joule = 0.0, dj = 0.0;
  int bad = 0;
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
    const double t2 = tsq_of_H(H[i], C3, C1);
    dj = fmax(dj, fabs(J[i] - Jold[i]));
    if (!isfinite(J[i]) || !isfinite(t2) || !(t2 > 0.0)) bad = 1;
    tsq = fmax(tsq, t2);
    joule = fma(Q[i], 2.0 * kPi * r[i] * area[i], joule);
  }
  tsq = warp_max(tsq);
  joule = warp_sum(joule);
  dj = warp_max(dj);
  bad = __any_sync(0xffffffffu, bad);
  if ((threadIdx.x & 31) == 0) {
    if (dj > 0.0 && isfinite(dj)) atomic_max_pos(&sc->djmax, dj);
    if (tsq > 0.0 && isfinite(tsq)) atomic_max_pos(&sc->tmax, sqrt(tsq));
    atomicAdd(&sc->joule, joule);
    if (bad) atomicOr(&sc->nonfinite, 1);
  }
}
}  // namespace

#define QS_LAUNCH(v) (g_sm_count = (v).sm_count, ++*(v).launches)

void k_material(const VecCtx& v, const MaterialParams& mp, const MaterialArgs& a) {
  QS_LAUNCH(v);
  MaterialConsts k;
  k.inv_Tc = 1.0 / mp.Tc;
  k.inv_B0 = 1.0 / mp.B0;
  k.inv_Y = 1.0 / mp.Y;
  k.inv_rho_n = 1.0 / mp.rho_n;
  k.hC1 = 0.5 * mp.C1;
  k.qC1sq = 0.25 * mp.C1 * mp.C1;
  k.inv_hC3 = 2.0 / mp.C3;
  dim3 grid(grid_for(a.N), 1);
  if (a.Nz > 0) {   // 2-D: no integer division per cell
    const int nrow = a.N / a.Nz;
    grid.x = (a.Nz + kBlock - 1) / kBlock;
    grid.y = std::min(nrow, std::max(1, QS_MAT_WAVES * QS_MAT_MINB * g_sm_count / static_cast<int>(grid.x)));
  }
  const bool ev = a.xmax_bits != nullptr, aux = a.dEdJ != nullptr;
#define QS_MAT(F_, A_, E_) material_kernel<F_, A_, E_><<<grid, kBlock, 0, v.stream>>>(mp, k, a)
  if (a.from_acc) {
    if (ev) QS_MAT(true, false, true); else QS_MAT(true, false, false);
  } else if (aux) {
    if (ev) QS_MAT(false, true, true); else QS_MAT(false, true, false);
  } else {
    if (ev) QS_MAT(false, false, true); else QS_MAT(false, false, false);
  }
#undef QS_MAT
}
void k_build_rowtab(const VecCtx& v, int Nr, int Nz, const double* r, const double* selfcoef, const double* diagM,
                    const double* area, double4* rowtab) {
  QS_LAUNCH(v);
  rowtab_kernel<<<(Nr + 127) / 128, 128, 0, v.stream>>>(Nr, Nz, r, selfcoef, diagM, area, rowtab);
}
void k_enthalpy_from_T(const VecCtx& v, const MaterialParams& mp, const double* T, double* H, int n) {
  QS_LAUNCH(v);
  enthalpy_kernel<<<grid_for(n), kBlock, 0, v.stream>>>(n, mp.C3, mp.C1, T, H);
}
void k_T_from_enthalpy(const VecCtx& v, const MaterialParams& mp, const double* H, double* T, int n) {
  QS_LAUNCH(v);
  temperature_kernel<<<grid_for(n), kBlock, 0, v.stream>>>(n, mp.C3, mp.C1, H, T);
}
void k_heat_substep(const VecCtx& v, const MaterialParams& mp, const LatticeParams& lp, const double* Hin,
                    const double* Q, double* Hout, double dtsub) {
  QS_LAUNCH(v);
  const int gx = (lp.Nz + kHeatWarps * kHeatCols - 1) / (kHeatWarps * kHeatCols);
  // strips of rows: long enough to amortise the two halo rows, and chosen so that the CTAs fill whole waves of
  // the resident CTAs per SM (a 2.6-wave launch idles 14 % of the GPU in its last wave)
  if (g_sm_count == 0) grid_for(1);
  const bool tma = lp.Nz % 2 == 0;   // 16-byte aligned row segments: TMA pipeline
  const long long resident = static_cast<long long>(tma ? kHeatMinB : 3) * g_sm_count;
  int rows = 4;
  double best = -1.0;
  for (int cand = kHeatMaxRows; cand >= 4; --cand) {
    const long long ctas = static_cast<long long>(gx) * ((lp.Nr + cand - 1) / cand);
    const long long waves = (ctas + resident - 1) / resident;
    // useful fraction: wave fill x halo-row overhead
    const double eff = static_cast<double>(ctas) / static_cast<double>(waves * resident) * cand / (cand + 2.0);
    if (eff > best + 1e-9) best = eff, rows = cand;
  }
  dim3 grid(gx, (lp.Nr + rows - 1) / rows);
  if (tma) {
    heat_tma_kernel<<<grid, kHeatWarps * 32, sizeof(HeatSmem), v.stream>>>(mp, lp, rows, Hin, Q, Hout, dtsub);
  } else
    heat_kernel<false><<<grid, kHeatWarps * 32, 0, v.stream>>>(mp, lp, rows, Hin, Q, Hout, dtsub);
}
bool k_heat_all_substeps(const VecCtx& v, const MaterialParams& mp, const LatticeParams& lp, int m, const double* Hin,
                         const double* Q, double* Hout, double dtsub) {
  const long long N = static_cast<long long>(lp.Nr) * lp.Nz;
  if (N > kHeatSmallMax || m < 2) return false;
  QS_LAUNCH(v);
  const int rows_per = (lp.Nr + kHeatClusterCtas - 1) / kHeatClusterCtas;
  if (lp.Nr >= 2 * kHeatClusterCtas && rows_per * lp.Nz <= kHeatClusterThreads * kHeatClusterPer) {   // 8 SMs instead of one
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(kHeatClusterCtas);
    cfg.blockDim = dim3(kHeatClusterThreads);
    cfg.dynamicSmemBytes = sizeof(double) * (2 * static_cast<size_t>(rows_per) * lp.Nz + 3 * (rows_per + lp.Nz));
    cfg.stream = v.stream;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = kHeatClusterCtas;
    at[0].val.clusterDim.y = 1;
    at[0].val.clusterDim.z = 1;
    cfg.attrs = at;
    cfg.numAttrs = 1;
    if (cudaLaunchKernelEx(&cfg, heat_cluster_kernel, mp, lp, m, rows_per, Hin, Q, Hout, dtsub) == cudaSuccess) return true;
    cudaGetLastError();                                            // cluster launch refused: the single-CTA kernel below
  }
  heat_small_kernel<<<1, kHeatSmallThreads, sizeof(double) * (N + 3 * (lp.Nr + lp.Nz)), v.stream>>>(mp, lp, m, Hin, Q, Hout,
                                                                                                 dtsub);
  return true;
}
int k_heat_block_max() { return kHbHalo; }
// msub <= kHbHalo sub-steps in one launch (lattices too large for the in-SM kernel)
void k_heat_block(const VecCtx& v, const MaterialParams& mp, const LatticeParams& lp, int msub, const double* Hin,
                  const double* Q, double* Hout, double dtsub) {
  QS_LAUNCH(v);
  const long long tiles64 = static_cast<long long>((lp.Nr + 63) / 64) * ((lp.Nz + 63) / 64);
  if (tiles64 >= 4ll * g_sm_count) {   // big lattices: 64 x 64 tiles (halo overhead 27 %), two CTAs per SM
    dim3 grid((lp.Nz + 63) / 64, (lp.Nr + 63) / 64);
    heat_block_kernel<64, 1024><<<grid, 1024, heat_block_smem(64), v.stream>>>(mp, lp, msub, Hin, Q, Hout, dtsub);
  } else {                             // the coil configs: 32 x 32 tiles so that every SM has work
    dim3 grid((lp.Nz + 31) / 32, (lp.Nr + 31) / 32);
    heat_block_kernel<32, 256><<<grid, 256, heat_block_smem(32), v.stream>>>(mp, lp, msub, Hin, Q, Hout, dtsub);
  }
}
void pointwise_prepare_device() {
  cudaFuncSetAttribute(heat_block_kernel<64, 1024>, cudaFuncAttributeMaxDynamicSharedMemorySize, static_cast<int>(heat_block_smem(64)));
  cudaFuncSetAttribute(heat_block_kernel<32, 256>, cudaFuncAttributeMaxDynamicSharedMemorySize, static_cast<int>(heat_block_smem(32)));
  cudaFuncSetAttribute(heat_tma_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, static_cast<int>(sizeof(HeatSmem)));
  cudaFuncSetAttribute(heat_small_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 160 * 1024);   // N + 3 (Nr + Nz) doubles <= 131 KB
}
void k_events(const VecCtx& v, const MaterialParams& mp, const EventArgs& e) {
  if (!v.n_turns) return;
  QS_LAUNCH(v);
  int bt = 32;
  while (bt < (v.N + v.n_turns - 1) / v.n_turns && bt < kEventBlockMax) bt <<= 1;
  events_kernel<<<v.n_turns, bt, 0, v.stream>>>(v.n_turns, v.turn_ptr, v.turn_idx, mp,
                                                                                e, v.sc);
}
void k_step_stats(const VecCtx& v, const MaterialParams& mp, const double* J, const double* Jold, const double* H,
                  const double* Q, const double* r, const double* area) {
  QS_LAUNCH(v);
  stats_kernel<<<grid_for(v.N), kBlock, 0, v.stream>>>(v.N, mp.C3, mp.C1, J, Jold, H, Q, r, area, v.sc);
}

}  // namespace qs
