// qs_adi.cu — ADI heat step (the paper's thermal method, "solved by ADI"; reading C15).
//
// Peaceman-Rachford on U = T^2 with the capacity H' = dH/dU = C3/2 U + C1/2 lagged at the start of the sub-step and the
// Robin loss linearised about U^k (beta = rb/(2 T^k), c = rb (T^k/2 - T_b)):
//   (2H'/delta - L_r + beta_r) U*  = 2H'/delta U^k + L_z U^k - rb_z (T^k - T_b) + Q - c_r          implicit in r
//   (2H'/delta - L_z + beta_z) U'  = 2H'/delta U*  + L_r U* - beta_r U* - c_r + Q - c_z            implicit in z
//   H <- H + H' (U' - U^k)                       (the two half-steps are an exact energy balance for H' dU)
// L_r, L_z use the per-row / per-column coefficient tables of the explicit kernel (LatticeParams).
//
// Five passes per sub-step: prep1 (U, H', right-hand side and diagonal of the r-systems), Thomas along r (one thread
// per column, coalesced across iz), prep2 (r-part of the operator on U*, right-hand side and diagonal of the
// z-systems, written TRANSPOSED through a shared-memory tile), Thomas along z on the transposed arrays (one thread per
// row, coalesced across ir), finish (transpose back, enthalpy update).
#include "qs_internal.h"
#include "qs_pair.cuh"

namespace qs {

namespace {

__device__ __forceinline__ double sqrt_seeded(double a) {   // a > 0
  const double y0 = rsqrt_seed(a);
  const double g = a * y0;
  const double e = fma(-g, y0, 1.0);
  return fma(g * e, fma(0.375, e, 0.5), g);
}
__device__ __forceinline__ double tsq_from_H(double H, double C3, double C1) {
  return (sqrt_seeded(fma(C3, H, 0.25 * C1 * C1)) - 0.5 * C1) * (2.0 / C3);
}

// pass 1: canonical layout c = ir Nz + iz
__global__ void adi_prep1_kernel(MaterialParams mp, LatticeParams lp, double two_over_delta, const double* __restrict__ H,
                                 const double* __restrict__ Q, double* __restrict__ U, double* __restrict__ Hp,
                                 double* __restrict__ rhs, double* __restrict__ diag) {
  const int iz = blockIdx.x * blockDim.x + threadIdx.x, ir = blockIdx.y;
  if (iz >= lp.Nz) return;
  const long long c = static_cast<long long>(ir) * lp.Nz + iz;
  const double u = tsq_from_H(H[c], mp.C3, mp.C1);
  const double T = sqrt_seeded(u);
  const double hp = 0.5 * mp.C3 * u + 0.5 * mp.C1;
  const double zp = lp.hz_p[iz], zm = lp.hz_m[iz];
  const double un = zp != 0.0 ? tsq_from_H(H[c + 1], mp.C3, mp.C1) : u;
  const double ul = zm != 0.0 ? tsq_from_H(H[c - 1], mp.C3, mp.C1) : u;
  const double rbr = lp.rb_r[ir], rbz = lp.rb_z[iz];
  const double w = two_over_delta * hp;
  double r = fma(w, u, Q[c]);
  r = fma(zp, un - u, r);
  r = fma(zm, ul - u, r);
  r -= rbz * (T - lp.T_bath);
  r -= rbr * (0.5 * T - lp.T_bath);
  U[c] = u;
  Hp[c] = hp;
  rhs[c] = r;
  diag[c] = w + lp.hr_p[ir] + lp.hr_m[ir] + rbr / (2.0 * T);
}

// Thomas algorithm along the SLOW axis of an [n_slow][n_fast] array: one thread per fast index.
// System i: -lo[i] x_{i-1} + diag_i x_i - hi[i] x_{i+1} = rhs_i  (lo[0] = hi[n_slow-1] = 0 by construction of the tables)
__global__ void adi_thomas_kernel(int n_slow, int n_fast, const double* __restrict__ lo, const double* __restrict__ hi,
                                  const double* __restrict__ diag, const double* __restrict__ rhs,
                                  double* __restrict__ cp, double* __restrict__ x) {
  const int f = blockIdx.x * blockDim.x + threadIdx.x;
  if (f >= n_fast) return;
  double cprev = 0.0, rprev = 0.0;
  for (int i = 0; i < n_slow; ++i) {
    const long long k = static_cast<long long>(i) * n_fast + f;
    const double a = -lo[i], cc = -hi[i];
    const double den = 1.0 / fma(-a, cprev, diag[k]);
    cprev = cc * den;
    rprev = fma(-a, rprev, rhs[k]) * den;
    cp[k] = cprev;
    x[k] = rprev;                                   // r' for now
  }
  double xn = 0.0;
  for (int i = n_slow - 1; i >= 0; --i) {
    const long long k = static_cast<long long>(i) * n_fast + f;
    xn = fma(-cp[k], xn, x[k]);
    x[k] = xn;
  }
}

// pass 3: reads canonical, writes rhs2 / diag2 transposed ([iz][ir]) through a 32 x 33 tile
__global__ void adi_prep2_kernel(MaterialParams mp, LatticeParams lp, double two_over_delta, const double* __restrict__ U,
                                 const double* __restrict__ Hp, const double* __restrict__ Us,
                                 const double* __restrict__ Q, double* __restrict__ rhsT, double* __restrict__ diagT) {
  __shared__ double tr[32][33], td[32][33];
  const int iz0 = blockIdx.x * 32, ir0 = blockIdx.y * 32;
  for (int dy = threadIdx.y; dy < 32; dy += blockDim.y) {
    const int ir = ir0 + dy, iz = iz0 + threadIdx.x;
    double r = 0.0, d = 1.0;
    if (ir < lp.Nr && iz < lp.Nz) {
      const long long c = static_cast<long long>(ir) * lp.Nz + iz;
      const double us = Us[c], hp = Hp[c];
      const double T = sqrt_seeded(U[c]);
      const double rp = lp.hr_p[ir], rm = lp.hr_m[ir];
      const double un = rp != 0.0 ? Us[c + lp.Nz] : us, up = rm != 0.0 ? Us[c - lp.Nz] : us;
      const double rbr = lp.rb_r[ir], rbz = lp.rb_z[iz];
      const double w = two_over_delta * hp;
      r = fma(w, us, Q[c]);
      r = fma(rp, un - us, r);
      r = fma(rm, up - us, r);
      r -= rbr / (2.0 * T) * us;
      r -= rbr * (0.5 * T - lp.T_bath);
      r -= rbz * (0.5 * T - lp.T_bath);
      d = w + lp.hz_p[iz] + lp.hz_m[iz] + rbz / (2.0 * T);
    }
    tr[dy][threadIdx.x] = r;
    td[dy][threadIdx.x] = d;
  }
  __syncthreads();
  for (int dy = threadIdx.y; dy < 32; dy += blockDim.y) {
    const int iz = iz0 + dy, ir = ir0 + threadIdx.x;      // transposed: fast index is ir
    if (ir < lp.Nr && iz < lp.Nz) {
      const long long k = static_cast<long long>(iz) * lp.Nr + ir;
      rhsT[k] = tr[threadIdx.x][dy];
      diagT[k] = td[threadIdx.x][dy];
    }
  }
}

// pass 5: U' arrives transposed; H <- H + H' (U' - U^k) in canonical layout
__global__ void adi_finish_kernel(LatticeParams lp, const double* __restrict__ UnT, const double* __restrict__ U,
                                  const double* __restrict__ Hp, const double* __restrict__ Hin, double* __restrict__ Hout) {
  __shared__ double t[32][33];
  const int iz0 = blockIdx.x * 32, ir0 = blockIdx.y * 32;
  for (int dy = threadIdx.y; dy < 32; dy += blockDim.y) {
    const int iz = iz0 + dy, ir = ir0 + threadIdx.x;
    t[dy][threadIdx.x] = (ir < lp.Nr && iz < lp.Nz) ? UnT[static_cast<long long>(iz) * lp.Nr + ir] : 0.0;
  }
  __syncthreads();
  for (int dy = threadIdx.y; dy < 32; dy += blockDim.y) {
    const int ir = ir0 + dy, iz = iz0 + threadIdx.x;
    if (ir < lp.Nr && iz < lp.Nz) {
      const long long c = static_cast<long long>(ir) * lp.Nz + iz;
      Hout[c] = fma(Hp[c], t[threadIdx.x][dy] - U[c], Hin[c]);
    }
  }
}

}  // namespace

// One ADI sub-step of length delta.  scratch: six arrays of N doubles.  Five launches.
int k_heat_adi_substep(const VecCtx& v, const MaterialParams& mp, const LatticeParams& lp, const double* Hin,
                       const double* Q, double* Hout, double delta, double* const scratch[6]) {
  double *U = scratch[0], *Hp = scratch[1], *rhs = scratch[2], *diag = scratch[3], *cp = scratch[4], *x = scratch[5];
  const double w = 2.0 / delta;
  const dim3 g1((lp.Nz + 127) / 128, lp.Nr);
  adi_prep1_kernel<<<g1, 128, 0, v.stream>>>(mp, lp, w, Hin, Q, U, Hp, rhs, diag);
  adi_thomas_kernel<<<(lp.Nz + 63) / 64, 64, 0, v.stream>>>(lp.Nr, lp.Nz, lp.hr_m, lp.hr_p, diag, rhs, cp, x);   // x = U*
  const dim3 gt((lp.Nz + 31) / 32, (lp.Nr + 31) / 32), bt(32, 8);
  adi_prep2_kernel<<<gt, bt, 0, v.stream>>>(mp, lp, w, U, Hp, x, Q, rhs, diag);                                   // transposed
  adi_thomas_kernel<<<(lp.Nr + 63) / 64, 64, 0, v.stream>>>(lp.Nz, lp.Nr, lp.hz_m, lp.hz_p, diag, rhs, cp, x);   // x = U'^T
  adi_finish_kernel<<<gt, bt, 0, v.stream>>>(lp, x, U, Hp, Hin, Hout);
  *v.launches += 5;
  return 5;
}

}  // namespace qs
