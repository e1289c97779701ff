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
//   p = sqrt(u v) (= a_n b_n);  t = 4 c_{n+1}^2 = u + v - 2p;  u' = (u + v + 2p)/4 = p + t/4;  v' = p
// (10 FP64 operations per iteration).
// After NIT iterations the rest of the AGM is summed in closed form as a power series in
// delta = 1 - v/u = k_NIT^2 (the modulus at level NIT), from the identities
//   1/agm(a, b)                       = (1/a) F(delta),  F = (2/pi) K = sum_j ((2j-1)!!/(2j)!!)^2 delta^j
//   sum_{m>NIT} 2^{m-1} c_m^2         = 2^NIT u G(delta), G = 1 - E/K - delta/2 = delta^2/16 + delta^3/32 + ...
// truncated after delta^(ORD+1) in F and delta^(ORD+2) in G, ORD = 2..6.  Truncation error < 1e-16 relative in M, K
// and E when k'^2 >= the class threshold (table in qs_operator.cu, derived with 60-digit arithmetic).
// The series variable actually used is x = 4 delta = t_NIT / u (u - v = t_NIT / 4 after the last iteration, so no
// subtraction is needed); the powers of 4 are folded into the coefficients (all exact binary fractions).
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
  double emS;    // (A2 + B2)/2 - S   (field kernels only; E/sqrt(A2) = (pi/2) yinf emS / A2)   [m^2]
};

// F(delta) = 1 + delta (kF[0] + kF[1] delta + ...),  G(delta) = delta^2 (kG[0] + kG[1] delta + ...)
__device__ constexpr double kSeriesF[8] = {1.0 / 4.0,           9.0 / 64.0,           25.0 / 256.0,
                                           1225.0 / 16384.0,    3969.0 / 65536.0,     53361.0 / 1048576.0,
                                           184041.0 / 4194304.0, 41409225.0 / 1073741824.0};
__device__ constexpr double kSeriesG[8] = {1.0 / 16.0,          1.0 / 32.0,           41.0 / 2048.0,
                                           59.0 / 4096.0,       727.0 / 65536.0,      1171.0 / 131072.0,
                                           498409.0 / 67108864.0, 848479.0 / 134217728.0};
__host__ __device__ constexpr double pow4(int j) { return j <= 0 ? 1.0 : 4.0 * pow4(j - 1); }

// Horner evaluation of sum_{j=0..ORD} c_j x^j with compile-time coefficients c_j = scale * tab[j] / 4^j
template <int ORD, int J = ORD>
struct Horner {
  static __device__ __forceinline__ double run(const double (&tab)[8], double scale, double x) {
    if constexpr (J == ORD) {
      return Horner<ORD, J - 1>::run_acc(tab, scale, x, scale * tab[ORD] / pow4(ORD));
    } else {
      return 0.0;
    }
  }
  static __device__ __forceinline__ double run_acc(const double (&tab)[8], double scale, double x, double acc) {
    const double next = fma(acc, x, scale * tab[J] / pow4(J));
    if constexpr (J == 0) return next;
    else return Horner<ORD, J - 1>::run_acc(tab, scale, x, next);
  }
};

// ORD = order of the series tail (2: "lo", 4: "hi" of round 1; 3, 5, 6 fill the ladder in between)
template <int NIT, int ORD, bool FIELD>
__device__ __forceinline__ PairAGM agm_pair(double A2, double B2) {
  static_assert(ORD >= 1 && ORD <= 7, "series order");
  PairAGM o;
  double u = A2, v = B2, S = 0.0, t = 0.0, s1 = 0.0;
  o.y0sq = 0.0;
  o.emS = 0.0;
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
      s1 = s;
    }
    t = fma(-2.0, p, s);                      // 4 c_{n+1}^2 = u + v - 2p
    S = fma(coef, t, S);
    u = fma(0.25, t, p);                      // (u + v + 2p)/4 = p + c_{n+1}^2
    v = p;
    coef *= 2.0;
  }
  // closed-form rest in x = 4 delta = t / u  (u - v = t/4)
  const double y = rsqrt_fast(u);
  const double x = t * (y * y);
  const double c2N = 4.0 * coef;              // 2^NIT
  const double F = Horner<ORD>::run(kSeriesF, 0.25, x);          // (1/4) sum kF[j] delta^j
  const double G = Horner<ORD>::run(kSeriesG, c2N / 16.0, x);    // 2^NIT / 16 sum kG[j] delta^j
  o.yinf = y * fma(x, F, 1.0);                // y (1 + delta/4 + 9 delta^2/64 + ...)
  o.S = fma(t * x, G, S);                     // + 2^NIT (u - v) delta (1/16 + delta/32 + ...)
  if (FIELD) o.emS = fma(0.5, s1, -o.S);
  return o;
}

}  // namespace qs
