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
// u_n = a_n^2, v_n = b_n^2, so that one iteration needs exactly one square root (MUFU seed + one cubic
// correction, 5 FP64 operations) and the two start-up roots sqrt(A2), sqrt(B2) are never taken:
//   p = sqrt(u v) (= a_n b_n);  4 c_{n+1}^2 = u + v - 2p;  u' = (u + v + 2p)/4;  v' = p
// (10 FP64 operations per iteration: u' is formed as p + c_{n+1}^2, which needs no separate division by 4).
// After NIT iterations the rest of the AGM is summed in closed form as a power series in
// delta = 1 - v/u = k_NIT^2 (the modulus at level NIT), from the identities
//   1/agm(a, b)                       = (1/a) F(delta),  F = (2/pi) K = sum_j ((2j-1)!!/(2j)!!)^2 delta^j
//   sum_{m>NIT} 2^{m-1} c_m^2         = 2^NIT u G(delta), G = 1 - E/K - delta/2 = delta^2/16 + delta^3/32 + ...
// truncated after delta^DF in F and delta^DG in G, (DF, DG) = (3, 4) or (5, 6).  Truncation error
// < 1e-16 relative in M, K and E when k'^2 >= the class threshold (table in qs_operator.cu, derived with
// 60-digit arithmetic).
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
  return y * fma(q, e, 1.0);                  // y (1 + e/2 + 3 e^2/8); no multiply-add has three register operands
}

struct PairAGM {
  double S;      // sum_{n>=1} 2^{n-1} c_n^2                     [m^2]
  double yinf;   // 1 / a_inf                                    [1/m]
  double y0sq;   // 1 / (A2 B2)   (field kernels only)           [1/m^4]
  double mid;    // (A2 + B2)/2 = ri^2 + rj^2 + dz^2             [m^2]
};

// HI = false: series to (delta^3, delta^4); HI = true: (delta^5, delta^6)
template <int NIT, bool HI, bool FIELD>
__device__ __forceinline__ PairAGM agm_pair(double A2, double B2) {
  PairAGM o;
  double u = A2, v = B2, S = 0.0;
  o.y0sq = 0.0;
  o.mid = 0.0;
  double coef = 0.25;                         // 2^{n-1} / 4
#pragma unroll
  for (int n = 0; n < NIT; ++n) {
    const double w = u * v;
    const double y0 = rsqrt_seed(w);
    const double g = w * y0;                  // ~ sqrt(w)
    const double e = fma(-g, y0, 1.0);        // 1 - w y0^2
    const double q = fma(0.375, e, 0.5);
    const double zc = fma(q, e, 1.0);         // 1 + e/2 + 3 e^2/8
    const double p = g * zc;                  // sqrt(w)
    const double s = u + v;
    if (FIELD && n == 0) {
      const double y = y0 * zc;               // 1/sqrt(w)
      o.y0sq = y * y;
      o.mid = 0.5 * s;
    }
    const double t = fma(-2.0, p, s);         // 4 c_{n+1}^2 = u + v - 2p
    S = fma(coef, t, S);
    u = fma(0.25, t, p);                      // (u + v + 2p)/4 = p + c_{n+1}^2
    v = p;
    coef *= 2.0;
  }
  // closed-form rest: delta = (u - v)/u
  const double y = rsqrt_fast(u);
  const double d = u - v;
  const double delta = d * (y * y);
  const double c2N = 4.0 * coef;              // 2^NIT
  double F, G;
  if (HI) {
    F = fma(fma(fma(fma(3969.0 / 65536.0, delta, 1225.0 / 16384.0), delta, 25.0 / 256.0), delta, 9.0 / 64.0), delta, 0.25);
    G = fma(fma(fma(fma(c2N * (727.0 / 65536.0), delta, c2N * (59.0 / 4096.0)), delta, c2N * (41.0 / 2048.0)), delta,
                c2N / 32.0), delta, c2N / 16.0);
  } else {
    F = fma(fma(25.0 / 256.0, delta, 9.0 / 64.0), delta, 0.25);
    G = fma(fma(c2N * (41.0 / 2048.0), delta, c2N / 32.0), delta, c2N / 16.0);
  }
  o.yinf = y * fma(delta, F, 1.0);            // y (1 + delta/4 + 9 delta^2/64 + ...)
  o.S = fma(d * delta, G, S);                 // + 2^NIT u (delta^2/16 + delta^3/32 + ...)
  return o;
}

}  // namespace qs
