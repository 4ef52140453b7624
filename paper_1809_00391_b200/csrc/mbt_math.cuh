// mbt_math.cuh -- device arithmetic of the tracker: Philox4x32-10, uniforms, Box-Muller, sine.
//
// Compiled with --fmad=false: every fused multiply-add in this library is written out as fma(),
// everything else rounds operation by operation (BASELINE north_star (i): "FMA contraction controlled").
//
// Nothing here is shared with oracle/ (the CPU oracle has its own generator and uses libm).
#pragma once
#include <stdint.h>

namespace mbt {

// ------------------------------------------------------------------ Philox4x32-10
// Salmon, Moraes, Dror, Shaw, SC'11.  Round: (hi0:lo0) = M0*c0, (hi1:lo1) = M1*c2,
// c <- (hi1^c1^k0, lo1, hi0^c3^k1, lo0); the key is bumped by the Weyl constants after each round.
// The ten round keys depend only on the seed, so the host expands them once (PhiloxKeys) and the
// device round is 2 wide multiplies + 2 three-input XORs.
struct PhiloxKeys {
  uint32_t k0[10];
  uint32_t k1[10];
};

#define MBT_PHILOX_M0 0xD2511F53u
#define MBT_PHILOX_M1 0xCD9E8D57u
#define MBT_PHILOX_W0 0x9E3779B9u
#define MBT_PHILOX_W1 0xBB67AE85u

__host__ __device__ inline PhiloxKeys philox_expand_key(uint32_t k0, uint32_t k1) {
  PhiloxKeys K;
  for (int r = 0; r < 10; ++r) {
    K.k0[r] = k0;
    K.k1[r] = k1;
    k0 += MBT_PHILOX_W0;
    k1 += MBT_PHILOX_W1;
  }
  return K;
}

__device__ __forceinline__ void philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, const PhiloxKeys &K,
                                              uint32_t &x0, uint32_t &x1, uint32_t &x2, uint32_t &x3) {
#pragma unroll
  for (int r = 0; r < 10; ++r) {
    const uint64_t p0 = (uint64_t)MBT_PHILOX_M0 * (uint64_t)c0;
    const uint64_t p1 = (uint64_t)MBT_PHILOX_M1 * (uint64_t)c2;
    const uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
    const uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
    c0 = hi1 ^ c1 ^ K.k0[r];
    c1 = lo1;
    c2 = hi0 ^ c3 ^ K.k1[r];
    c3 = lo0;
  }
  x0 = c0; x1 = c1; x2 = c2; x3 = c3;
}

// u = (k + 1/2) 2^-52 with k the top 52 bits of the 64-bit word hi:lo (reading D8): exactly
// representable and strictly inside (0,1).  Built without an int->double conversion:
// bits(0x3FF<<52 | k) = 1 + k 2^-52, then one exact addition of (2^-53 - 1).
__device__ __forceinline__ double uniform52(uint32_t lo, uint32_t hi) {
  const uint32_t khi = hi >> 12;
  const uint32_t klo = __funnelshift_r(lo, hi, 12);
  const double d = __hiloint2double((int)(0x3FF00000u | khi), (int)klo);
  return d + (0x1p-53 - 1.0);
}

// ------------------------------------------------------------------ Box-Muller
// r = sqrt(-2 log u1), theta = 2 pi u2, (z_c, z_s) = (r cos theta, r sin theta)   (reading D8).
// ACCURATE variant (library log / sqrt / sincospi): initial distribution and self-tests.
__device__ __forceinline__ void box_muller_accurate(double u1, double u2, double &zc, double &zs) {
  const double r = sqrt(-2.0 * log(u1));
  double s, c;
  sincospi(2.0 * u2, &s, &c);
  zc = r * c;
  zs = r * s;
}

// sin and cos on [-pi/4, pi/4] as Taylor polynomials with coefficients (-1)^n / (2n+1)!, (-1)^n / (2n)!.
// NS / NC = number of terms after the leading x / 1.  Truncation error at |x| = pi/4:
//   sin: NS = 6 -> x^15/15! = 2.0e-14, NS = 7 -> x^17/17! = 4.6e-17;
//   cos: NC = 7 -> x^16/16! = 1.0e-15, NC = 8 -> x^18/18! = 2.0e-18.
template <int NS>
__device__ __forceinline__ double sin_poly(double x) {
  constexpr double c[8] = {-1.0 / 6.0, 1.0 / 120.0, -1.0 / 5040.0, 1.0 / 362880.0, -1.0 / 39916800.0,
                           1.0 / 6227020800.0, -1.0 / 1307674368000.0, 1.0 / 355687428096000.0};
  const double z = x * x;
  double p = c[NS - 1];
#pragma unroll
  for (int i = NS - 2; i >= 0; --i) p = fma(p, z, c[i]);
  return fma(x * z, p, x);
}
template <int NC>
__device__ __forceinline__ double cos_poly(double x) {
  constexpr double c[8] = {-1.0 / 2.0, 1.0 / 24.0, -1.0 / 720.0, 1.0 / 40320.0, -1.0 / 3628800.0,
                           1.0 / 479001600.0, -1.0 / 87178291200.0, 1.0 / 20922789888000.0};
  const double z = x * x;
  double p = c[NC - 1];
#pragma unroll
  for (int i = NC - 2; i >= 0; --i) p = fma(p, z, c[i]);
  return fma(z, p, 1.0);
}

// FAST variant used by the per-turn excitation (S2): absolute error of z below 1e-13,
// i.e. A_q * err << 1e-12 * sigma_delta.
//   log(u): u = 2^e m, m in [sqrt(1/2), sqrt(2)); log m = 2 atanh(s), s = (m-1)/(m+1), |s| <= 0.1716,
//           odd series through s^15 (next term 3e-14 relative);
//   sqrt:   hardware reciprocal-sqrt seed + two Newton steps;
//   sin/cos(2 pi u2): exact quadrant split q = rint(4 u2), f = u2 - q/4 in [-1/8, 1/8] (exact), then
//           the two polynomials on 2 pi f and a quadrant rotation.
__device__ __forceinline__ void box_muller_fast(double u1, double u2, double &zc, double &zs) {
  // ---- log(u1)
  int hi = __double2hiint(u1);
  const int lo = __double2loint(u1);
  int e = (hi >> 20) - 1023;             // u1 is a positive normal number (>= 2^-53)
  hi = (hi & 0x000FFFFF) | 0x3FF00000;   // m in [1,2)
  if (hi >= 0x3FF6A09F) {                // m >= sqrt(2) (to within the table of high words): halve
    hi -= 0x00100000;
    e += 1;
  }
  const double m = __hiloint2double(hi, lo);
  const double num = m - 1.0;            // exact
  const double den = m + 1.0;
  // reciprocal of den in [1.707, 2.414]: fp32 seed, two Newton steps in fp64
  double rcp = (double)__frcp_rn((float)den);
  rcp = fma(fma(-den, rcp, 1.0), rcp, rcp);
  rcp = fma(fma(-den, rcp, 1.0), rcp, rcp);
  double s = num * rcp;
  s = fma(fma(-den, s, num), rcp, s);    // one correction of the quotient
  const double s2 = s * s;
  double p = 1.0 / 15.0;
  p = fma(p, s2, 1.0 / 13.0);
  p = fma(p, s2, 1.0 / 11.0);
  p = fma(p, s2, 1.0 / 9.0);
  p = fma(p, s2, 1.0 / 7.0);
  p = fma(p, s2, 1.0 / 5.0);
  p = fma(p, s2, 1.0 / 3.0);
  const double ls = fma(s * s2, p, s);   // atanh(s)
  // -2 log u = -(2 e ln2 + 4 atanh s)
  const double ed = (double)e;
  double x = fma(ed, -1.38629436111989057245e+00, -4.0 * ls);      // -2 ln2 * e, high part
  x = fma(ed, -4.638093627692599e-17, x);                           // low part of 2 ln2
  // ---- r = sqrt(x), x in (0, 74]
  double y = (double)rsqrtf((float)x);
  y = fma(fma(-x * y, y, 1.0) * 0.5, y, y);
  y = fma(fma(-x * y, y, 1.0) * 0.5, y, y);
  double r = x * y;
  r = fma(fma(-r, r, x) * 0.5, y, r);
  // ---- sin, cos of 2 pi u2
  const double q = rint(4.0 * u2);       // 0..4
  const double f = fma(q, -0.25, u2);    // exact, |f| <= 1/8
  const double th = 6.28318530717958647692 * f;
  const double sn = sin_poly<6>(th), cs = cos_poly<7>(th);
  const int qi = (int)q;
  double c = (qi & 1) ? -sn : cs;
  double sv = (qi & 1) ? cs : sn;
  if (qi & 2) { c = -c; sv = -sv; }
  zc = r * c;
  zs = r * sv;
}

// ------------------------------------------------------------------ sine of the RF phase
// sin(y) for the RF kick (S1).  |y| < 2^16: Cody-Waite reduction by pi/2 split into three 33-bit pieces
// (k * piece is exact for |k| < 2^20, the remainder carries 99 bits of pi/2) and one polynomial chosen by the quadrant; larger or non-finite arguments
// (particles long lost from the bucket) take the library routine.
__device__ __forceinline__ double sin_rf(double y) {
  if (!(fabs(y) < 65536.0)) return sin(y);
  const double k = rint(y * 6.36619772367581382433e-01);
  double r = fma(k, -1.57079632673412561417e+00, y);
  r = fma(k, -6.07710050630396597660e-11, r);
  r = fma(k, -2.02226624871116645580e-21, r);
  const int ki = (int)k;
  const double v = (ki & 1) ? cos_poly<8>(r) : sin_poly<7>(r);
  return (ki & 2) ? -v : v;
}

}  // namespace mbt
