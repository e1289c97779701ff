// qs_pair.cuh — per-pair arithmetic of the ring-to-ring operator (device only).
//
// What is computed (north_star "K(k) and E(k) evaluated on the fly by AGM in FP64"):
//   A2 = (ri+rj)^2 + dz^2,  B2 = (ri-rj)^2 + dz^2                       (k'^2 = B2/A2)
//   AGM on (a0, b0) = (sqrt A2, sqrt B2):  a_{n+1} = (a_n+b_n)/2, b_{n+1} = sqrt(a_n b_n), c_{n+1} = (a_n-b_n)/2
//   M_ij          = (mu0 pi/2) * S / a_inf ,        S = sum_{n>=1} 2^{n-1} c_n^2
//   K/sqrt(A2)    = (pi/2) / a_inf
//   E/sqrt(A2)    = (pi/2) / a_inf * ((A2+B2)/2 - S) / A2
//
// How (differs from the textbook recurrence, same numbers): the recurrence is run on the SQUARES
// u_n = a_n^2, v_n = b_n^2, so that one iteration needs exactly one reciprocal square root and the two
// start-up roots sqrt(A2), sqrt(B2) are never taken:
//   p = sqrt(u v) (= a_n b_n);  4 c_{n+1}^2 = u + v - 2p;  u' = (u + v + 2p)/4;  v' = p
// After NIT such iterations one more AGM step is applied in closed form to first order in
// delta = (u - v)/u (no root):  1/a_inf ~= (1 + delta/4)/sqrt(u),  S += 2^NIT (u-v)^2/(16 u).
// Truncation error < 1e-16 relative when k'^2 >= kKp2Min[NIT] (table in qs_operator.cu, derived with
// 60-digit arithmetic).  The reciprocal square root is the MUFU seed plus one cubic correction.
#pragma once
#include <cuda_runtime.h>

namespace qs {

__device__ __forceinline__ double rsqrt_seed(double x) {
  double y;
  asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
  return y;
}

// 1/sqrt(x), x positive and normal.  Seed error e0 (<= 2^-20) -> 2.5 e0^3 after one Halley step.
__device__ __forceinline__ double rsqrt_fast(double x) {
  const double y = rsqrt_seed(x);
  const double t = x * y;
  const double e = fma(-t, y, 1.0);
  const double q = fma(0.375, e, 0.5);
  const double ye = y * e;
  return fma(ye, q, y);
}

struct PairAGM {
  double S;      // sum_{n>=1} 2^{n-1} c_n^2                     [m^2]
  double yinf;   // 1 / a_inf                                    [1/m]
  double y0sq;   // 1 / (A2 B2)   (field kernels only)           [1/m^4]
  double mid;    // (A2 + B2)/2 = ri^2 + rj^2 + dz^2             [m^2]
};

template <int NIT, bool FIELD>
__device__ __forceinline__ PairAGM agm_pair(double A2, double B2) {
  PairAGM o;
  double u = A2, v = B2, S = 0.0;
  o.y0sq = 0.0;
  o.mid = 0.0;
  double coef = 0.25;                         // 2^{n-1} / 4
#pragma unroll
  for (int n = 0; n < NIT; ++n) {
    const double w = u * v;
    const double y = rsqrt_fast(w);
    const double p = w * y;
    const double s = u + v;
    if (FIELD && n == 0) {
      o.y0sq = y * y;
      o.mid = 0.5 * s;
    }
    S = fma(coef, fma(-2.0, p, s), S);
    u = fma(0.5, p, 0.25 * s);
    v = p;
    coef *= 2.0;
  }
  const double y = rsqrt_fast(u);
  const double d = u - v;
  const double delta = d * (y * y);
  o.S = fma(coef * 0.25 * d, delta, S);       // + 2^NIT (u-v)^2 / (16 u)
  o.yinf = fma(0.25 * delta, y, y);
  return o;
}

}  // namespace qs
