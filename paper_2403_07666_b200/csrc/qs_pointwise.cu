// qs_pointwise.cu — K5 material law, K6 explicit heat sub-step, K7 event detector, step statistics.
//
// All three are streaming passes over per-cell FP64 arrays (HBM/L2 bound):
//   K5 reads J, H, bracc, bzacc, jc0_scale, r, area, selfcoef, diagM and writes Br, Bz, E, dE/dJ, Q, b, shift, Hd,
//      Jc, rho (C5, C4, C7).
//   K6 one explicit finite-volume sub-step in enthalpy form (C9; PAPER.md:75 heat equation with Robin borders):
//      a CTA stages T^2 of its tile plus a one-cell halo in shared memory (one sqrt per staged cell), so the
//      algorithmic traffic is read H, Q + write H = 24 B per cell per sub-step.
//   K7 one warp per turn over the CSR cell list: Tmax, mean|E|, max|J|/Jc, min rho/rho_n -> flags (C10).
#include "qs_internal.h"

namespace qs {

namespace {
constexpr int kBlock = 256;
int g_sm_count = 0;
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

__global__ void material_kernel(MaterialParams mp, MaterialArgs a) {
  const double two_pi = 2.0 * kPi;
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < a.N; i += gridDim.x * blockDim.x) {
    const double J = a.J[i], r = a.r[i], area = a.area[i];
    const double T = sqrt(tsq_of_H(a.H[i], mp.C3, mp.C1));
    double Br, Bz;
    if (a.from_acc) {
      Br = (0.25 * kMu0) * a.bracc[i] / r;
      Bz = (0.25 * kMu0) * a.bzacc[i] + a.selfcoef[i] * (area * J) + a.Bext;
    } else {
      Br = a.Br[i];
      Bz = a.Bz[i];
    }
    const double eps = J * Bz * r / mp.Y;
    const double Bmag = sqrt(Br * Br + Bz * Bz);
    const double fT = fmax(1.0 - T / mp.Tc, 0.0);
    const double fe = fmax(1.0 - mp.eps_coef * pow(fabs(eps), mp.eps_exp), 0.0);
    const double s = a.jc0_scale ? a.jc0_scale[i] : 1.0;
    const double Jc = mp.Jc0 * s * fT * fT / (1.0 + Bmag / mp.B0) * fe;
    double rho, dEdJ;
    if (Jc <= 0.0) {
      rho = mp.rho_n;
      dEdJ = mp.rho_n;
    } else if (J == 0.0) {
      rho = 0.0;
      dEdJ = 0.0;
    } else {
      const double x = fabs(J) / Jc;
      double xp = 1.0;
      if (mp.n_int > 0) {
        for (int k = 1; k < mp.n_int; ++k) xp *= x;          // x^(n-1), same multiplication chain as the oracle
      } else {
        xp = pow(x, mp.n_exp - 1.0);
      }
      const double rho_sc = (mp.Ec / Jc) * xp;
      const bool big = rho_sc >= mp.rho_n;
      const double u = big ? mp.rho_n / rho_sc : rho_sc / mp.rho_n;     // in [0, 1], no inf/inf
      rho = (big ? mp.rho_n : rho_sc) / (1.0 + u);
      const double w = (big ? u : 1.0) / (1.0 + u);
      dEdJ = rho * (1.0 + (mp.n_exp - 1.0) * w);
    }
    const double E = rho * J;
    a.Br[i] = Br;
    a.Bz[i] = Bz;
    a.E[i] = E;
    a.dEdJ[i] = dEdJ;
    a.Q[i] = E * J;
    a.Jc[i] = Jc;
    a.rho[i] = rho;
    a.b[i] = -two_pi * r * (E + 0.5 * r * a.Bdot);
    const double shift = mp.theta * a.dt * (two_pi * r * dEdJ / area);
    a.shift[i] = shift;
    a.Hd[i] = a.diagM[i] + shift;
  }
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

// ---- K6: one explicit sub-step.  Tile = kTz cells along z (contiguous) x kTr cells along r. ------------------
constexpr int kTz = 64, kTr = 8;   // 512 cells per CTA, 256 threads -> 2 cells per thread along r
__global__ void __launch_bounds__(256) heat_kernel(MaterialParams mp, LatticeParams lp, const double* __restrict__ Hin,
                                                   const double* __restrict__ Q, double* __restrict__ Hout,
                                                   double dtsub) {
  __shared__ double U[kTr + 2][kTz + 2];          // T^2 of the tile and its halo
  const int tz0 = blockIdx.x * kTz, tr0 = blockIdx.y * kTr;
  // stage: (kTr+2) x (kTz+2) entries, out-of-pack entries are never read
  for (int e = threadIdx.x; e < (kTr + 2) * (kTz + 2); e += blockDim.x) {
    const int lr = e / (kTz + 2), lz = e - lr * (kTz + 2);
    const int ir = tr0 + lr - 1, iz = tz0 + lz - 1;
    double u = 0.0;
    if (ir >= 0 && ir < lp.Nr && iz >= 0 && iz < lp.Nz) u = tsq_of_H(Hin[(long long)ir * lp.Nz + iz], mp.C3, mp.C1);
    U[lr][lz] = u;
  }
  __syncthreads();
  const int lz = threadIdx.x & (kTz - 1);
  const int iz = tz0 + lz;
  const double two_pi = 2.0 * kPi, h = lp.h;
#pragma unroll
  for (int sub = 0; sub < kTr * kTz / 256; ++sub) {
    const int lr = (threadIdx.x >> 6) + sub * (256 / kTz);
    const int ir = tr0 + lr;
    if (ir >= lp.Nr || iz >= lp.Nz) continue;
    const long long c = (long long)ir * lp.Nz + iz;
    const double rc = lp.r_inner + (ir + 0.5) * h;
    const double u = U[lr + 1][lz + 1];
    double F = 0.0;
    if (ir + 1 < lp.Nr) {   // radial face ir | ir+1, area 2 pi (r_c + h/2) h
      const double kap = (ir / lp.n == (ir + 1) / lp.n) ? mp.k_in : mp.k_between;
      F += kap * (U[lr + 2][lz + 1] - u) / (2.0 * h) * (two_pi * (rc + 0.5 * h) * h);
    }
    if (ir > 0) {           // radial face ir-1 | ir, area 2 pi (r_{c-1} + h/2) h
      const double kap = ((ir - 1) / lp.n == ir / lp.n) ? mp.k_in : mp.k_between;
      const double rm = lp.r_inner + (ir - 0.5) * h;
      F -= kap * (u - U[lr][lz + 1]) / (2.0 * h) * (two_pi * (rm + 0.5 * h) * h);
    }
    if (iz + 1 < lp.Nz) {   // axial faces, area 2 pi r_c h
      const double kap = (iz / lp.n == (iz + 1) / lp.n) ? mp.k_in : mp.k_between;
      F += kap * (U[lr + 1][lz + 2] - u) / (2.0 * h) * (two_pi * rc * h);
    }
    if (iz > 0) {
      const double kap = ((iz - 1) / lp.n == iz / lp.n) ? mp.k_in : mp.k_between;
      F -= kap * (u - U[lr + 1][lz]) / (2.0 * h) * (two_pi * rc * h);
    }
    if (ir == 0 || ir == lp.Nr - 1 || iz == 0 || iz == lp.Nz - 1) {   // Robin borders of the winding pack
      const double dT = sqrt(u) - lp.T_bath;
      double loss = 0.0;
      if (ir == 0) loss += lp.h_conv[0] * dT * two_pi * (rc - 0.5 * h) * h;
      if (ir == lp.Nr - 1) loss += lp.h_conv[1] * dT * two_pi * (rc + 0.5 * h) * h;
      if (iz == 0) loss += lp.h_conv[2] * dT * two_pi * rc * h;
      if (iz == lp.Nz - 1) loss += lp.h_conv[3] * dT * two_pi * rc * h;
      F -= loss;
    }
    const double vol = two_pi * rc * h * h;
    Hout[c] = Hin[c] + dtsub * (F / vol + Q[c]);
  }
}

// ---- K7 ---------------------------------------------------------------------------------------------------
__global__ void events_kernel(int n_turns, const int* __restrict__ ptr, const int* __restrict__ idx,
                              MaterialParams mp, EventArgs e, Scalars* sc) {
  const int w = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
  if (w >= n_turns) return;
  double tsq = 0.0, esum = 0.0, xmax = 0.0, rmin = 1e300;
  for (int k = ptr[w] + lane; k < ptr[w + 1]; k += 32) {
    const int i = idx[k];
    tsq = fmax(tsq, tsq_of_H(e.H[i], mp.C3, mp.C1));
    esum += fabs(e.E[i]);
    const double J = e.J[i], Jc = e.Jc[i];
    const double ratio = Jc > 0.0 ? fabs(J) / Jc : (J != 0.0 ? __longlong_as_double(0x7ff0000000000000LL) : 0.0);
    xmax = fmax(xmax, ratio);
    rmin = fmin(rmin, e.rho[i] / mp.rho_n);
  }
  tsq = warp_max(tsq);
  esum = warp_sum(esum);
  xmax = warp_max(xmax);
  rmin = warp_min(rmin);
  if (lane != 0) return;
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
  if (fl && e.t_first[w] < 0.0) e.t_first[w] = e.t_new;
  int ret = 0;
  if ((fl & 7) && !(old & 7)) ret |= 1;
  if (fl & 24) ret |= 2;
  if (ret) atomicOr(&sc->event_or, ret);
  e.flags[w] = fl;
  e.ebar_prev[w] = ebar;
}

__global__ void stats_kernel(int n, double C3, double C1, const double* __restrict__ J, const double* __restrict__ H,
                             const double* __restrict__ Q, const double* __restrict__ r,
                             const double* __restrict__ area, Scalars* sc) {
  double tsq = 0.0, joule = 0.0;
  int bad = 0;
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
    const double t2 = tsq_of_H(H[i], C3, C1);
    if (!isfinite(J[i]) || !isfinite(t2) || !(t2 > 0.0)) bad = 1;
    tsq = fmax(tsq, t2);
    joule = fma(Q[i], 2.0 * kPi * r[i] * area[i], joule);
  }
  tsq = warp_max(tsq);
  joule = warp_sum(joule);
  bad = __any_sync(0xffffffffu, bad);
  if ((threadIdx.x & 31) == 0) {
    if (tsq > 0.0 && isfinite(tsq)) atomic_max_pos(&sc->tmax, sqrt(tsq));
    atomicAdd(&sc->joule, joule);
    if (bad) atomicOr(&sc->nonfinite, 1);
  }
}
}  // namespace

#define QS_LAUNCH(v) (++*(v).launches)

void k_material(const VecCtx& v, const MaterialParams& mp, const MaterialArgs& a) {
  QS_LAUNCH(v);
  material_kernel<<<grid_for(a.N), kBlock, 0, v.stream>>>(mp, a);
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
  dim3 grid((lp.Nz + kTz - 1) / kTz, (lp.Nr + kTr - 1) / kTr);
  heat_kernel<<<grid, 256, 0, v.stream>>>(mp, lp, Hin, Q, Hout, dtsub);
}
void k_events(const VecCtx& v, const MaterialParams& mp, const EventArgs& e) {
  if (!v.n_turns) return;
  QS_LAUNCH(v);
  events_kernel<<<(v.n_turns * 32 + kBlock - 1) / kBlock, kBlock, 0, v.stream>>>(v.n_turns, v.turn_ptr, v.turn_idx, mp,
                                                                                e, v.sc);
}
void k_step_stats(const VecCtx& v, const MaterialParams& mp, const double* J, const double* H, const double* Q,
                  const double* r, const double* area) {
  QS_LAUNCH(v);
  stats_kernel<<<grid_for(v.N), kBlock, 0, v.stream>>>(v.N, mp.C3, mp.C1, J, H, Q, r, area, v.sc);
}

}  // namespace qs
