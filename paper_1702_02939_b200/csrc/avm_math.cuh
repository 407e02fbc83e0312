// avm_math.cuh — the three elementary functions of the director update (row a4; PAPER.md:50,
// :104; R8, R16), written for the FP64 pipe of sm_100a.
//
//   log_unit(u)        ln u            for u in (0,1), normal               (Box-Muller radius)
//   cos_2pi(u)         cos(2 pi u)     for u = (m + 1/2) 2^-52 in (0,1)     (Box-Muller angle)
//   sincos_any(t,s,c)  sin t, cos t    for any finite t                     (director n = (cos, sin))
//
// Why not the CUDA math library: its log / cospi / sincos spend a third of their issue slots on
// materialising polynomial coefficients (UMOV pairs) and on special cases that cannot occur
// here.  These versions keep every coefficient in constant memory, where DFMA reads it as an
// operand, and use plain Taylor / atanh series (the coefficients are 1/k! and 2/(2k+1), nothing
// fitted), long enough that the truncation error is below 2^-56 on the reduced range.  Each is
// accurate to about one ulp (tests/test_device_math.py checks them against mpmath on the host:
// the file also compiles as plain C++).
#pragma once
#include <math.h>
#include <stdint.h>
#include <string.h>

#if defined(__CUDACC__)
#define AVM_HD __host__ __device__ __forceinline__
#else
#define AVM_HD inline
#endif

namespace avm {

#if defined(__CUDA_ARCH__)
#define AVM_COEF static __constant__ double
#else
#define AVM_COEF static const double
#endif

// sin r = r + r z (S[0] + z (S[1] + ...)),  z = r^2,  S[k] = (-1)^(k+1) / (2k+3)!
AVM_COEF kSin[11] = {-1.0 / 6.0, 1.0 / 120.0, -1.0 / 5040.0, 1.0 / 362880.0, -1.0 / 39916800.0,
                     1.0 / 6227020800.0, -1.0 / 1307674368000.0, 1.0 / 355687428096000.0,
                     -1.0 / 121645100408832000.0, 1.0 / 51090942171709440000.0,
                     -1.0 / 25852016738884976640000.0};
// cos r = 1 - z/2 + z^2 (C[0] + z (C[1] + ...)),  C[k] = (-1)^k / (2k+4)!
AVM_COEF kCos[7] = {1.0 / 24.0, -1.0 / 720.0, 1.0 / 40320.0, -1.0 / 3628800.0, 1.0 / 479001600.0,
                    -1.0 / 87178291200.0, 1.0 / 20922789888000.0};
// ln((1+s)/(1-s)) = 2 s + s z (L[0] + z (L[1] + ...)),  z = s^2,  L[k] = 2 / (2k+3)
AVM_COEF kLog[10] = {2.0 / 3.0, 2.0 / 5.0, 2.0 / 7.0, 2.0 / 9.0, 2.0 / 11.0, 2.0 / 13.0, 2.0 / 15.0,
                     2.0 / 17.0, 2.0 / 19.0, 2.0 / 21.0};

AVM_HD double bits_to_double(uint32_t hi, uint32_t lo) {
#if defined(__CUDA_ARCH__)
  return __hiloint2double((int)hi, (int)lo);
#else
  const uint64_t b = ((uint64_t)hi << 32) | lo;
  double x;
  memcpy(&x, &b, 8);
  return x;
#endif
}
AVM_HD uint32_t hi_bits(double x) {
#if defined(__CUDA_ARCH__)
  return (uint32_t)__double2hiint(x);
#else
  uint64_t b;
  memcpy(&b, &x, 8);
  return (uint32_t)(b >> 32);
#endif
}
AVM_HD uint32_t lo_bits(double x) {
#if defined(__CUDA_ARCH__)
  return (uint32_t)__double2loint(x);
#else
  uint64_t b;
  memcpy(&b, &x, 8);
  return (uint32_t)b;
#endif
}
// 1/q to ~2^-22 (MUFU.RCP64H on the device)
AVM_HD double rcp_seed(double q) {
#if defined(__CUDA_ARCH__)
  double y;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(q));
  return y;
#else
  return (double)(1.0f / (float)q);
#endif
}

// round-to-nearest integer of |x| < 2^31 as (double, int) without a conversion instruction:
// adding 1.5 * 2^52 leaves the integer in the low mantissa bits.
AVM_HD double round_magic(double x, int& q) {
  const double t = x + 6755399441055744.0;
  q = (int)lo_bits(t);
  return t - 6755399441055744.0;
}

// ln u, u in (0,1) normal.  u = 2^e m with m in [sqrt(1/2), sqrt(2)); f = m - 1; s = f / (2 + f);
// ln m = 2 s + s R(z) = f - s (f - R)   (because 2 s = f - s f), which keeps the leading term exact.
AVM_HD double log_unit(double u) {
  // move the exponent boundary from 1 to sqrt(2): add (1 - sqrt(1/2)) in units of the high word
  const uint32_t i = hi_bits(u) + (0x3ff00000u - 0x3fe6a09eu);
  const int e = (int)(i >> 20) - 1023;
  const double m = bits_to_double((i & 0x000fffffu) + 0x3fe6a09eu, lo_bits(u));
  const double f = m - 1.0;
  const double q = 2.0 + f;
  double y = rcp_seed(q);
  double r = fma(-q, y, 1.0);
  y = fma(y, r, y);
  r = fma(-q, y, 1.0);
  y = fma(y, r, y);
  double s = f * y;
  s = fma(fma(-q, s, f), y, s);
  const double z = s * s;
  double p = kLog[9];
  p = fma(p, z, kLog[8]); p = fma(p, z, kLog[7]); p = fma(p, z, kLog[6]); p = fma(p, z, kLog[5]);
  p = fma(p, z, kLog[4]); p = fma(p, z, kLog[3]); p = fma(p, z, kLog[2]); p = fma(p, z, kLog[1]);
  p = fma(p, z, kLog[0]);
  const double R = p * z;
  const double ed = (double)e;
  // ln 2 = hi + lo with 21 trailing zero bits in hi, so ed * hi is exact for |e| < 2^20
  const double c = fma(ed, 1.9082149292705877e-10, -(s * (f - R)));
  return fma(ed, 6.93147180369123816490e-01, f) + c;
}

// sin a for |a| <= pi/2 (Taylor to a^23: truncation below 2^-59 relative)
AVM_HD double sin_half_pi(double a) {
  const double z = a * a;
  double p = kSin[10];
  p = fma(p, z, kSin[9]); p = fma(p, z, kSin[8]); p = fma(p, z, kSin[7]); p = fma(p, z, kSin[6]);
  p = fma(p, z, kSin[5]); p = fma(p, z, kSin[4]); p = fma(p, z, kSin[3]); p = fma(p, z, kSin[2]);
  p = fma(p, z, kSin[1]); p = fma(p, z, kSin[0]);
  return fma(a * z, p, a);
}

// cos(2 pi u) for u = (m + 1/2) 2^-52 in (0,1):  cos(pi x) = sin(pi (1/2 - x)), x = 2u.  y = 1/2 - x
// is exact (a multiple of 2^-52 below 1.5 in magnitude); y - rint(y) in [-1/2, 1/2] is exact too,
// and sin(pi y) = (-1)^rint(y) sin(pi (y - rint(y))).
AVM_HD double cos_2pi(double u) {
  const double y = 0.5 - (u + u);
  int k;
  const double yr = y - round_magic(y, k);
  const double a = yr * 3.14159265358979323846;
  const double s = sin_half_pi(a);
  return bits_to_double(hi_bits(s) ^ ((uint32_t)k << 31), lo_bits(s));
}

// sin t and cos t, any finite t.  k = rint(t 2/pi); r = t - k pi/2 by a three-term Cody-Waite
// reduction with FMAs (pi/2 = P1 + P2 + P3 to ~160 bits), |r| <= pi/4 (+ rounding slack); Taylor
// to r^15 / r^16; quadrant fix-up on the sign bits.  |t| >= 2^30 (never reached by a diffusing
// director) falls back to the library routine.
AVM_HD void sincos_any(double t, double* sn, double* cs) {
  if (!(fabs(t) < 1073741824.0)) {
#if defined(__CUDA_ARCH__)
    ::sincos(t, sn, cs);
#else
    *sn = sin(t); *cs = cos(t);
#endif
    return;
  }
  int k;
  const double kd = round_magic(t * 6.36619772367581382433e-01, k);
  double r = fma(-kd, 1.57079632679489655800e+00, t);
  r = fma(-kd, 6.12323399573676603587e-17, r);
  r = fma(-kd, -1.49738490485916983294e-33, r);
  const double z = r * r;
  double ps = kSin[6];
  ps = fma(ps, z, kSin[5]); ps = fma(ps, z, kSin[4]); ps = fma(ps, z, kSin[3]); ps = fma(ps, z, kSin[2]);
  ps = fma(ps, z, kSin[1]); ps = fma(ps, z, kSin[0]);
  const double s = fma(r * z, ps, r);
  double pc = kCos[6];
  pc = fma(pc, z, kCos[5]); pc = fma(pc, z, kCos[4]); pc = fma(pc, z, kCos[3]); pc = fma(pc, z, kCos[2]);
  pc = fma(pc, z, kCos[1]); pc = fma(pc, z, kCos[0]);
  const double c = fma(z * z, pc, fma(z, -0.5, 1.0));
  // k mod 4:  0: (s, c)   1: (c, -s)   2: (-s, -c)   3: (-c, s)
  const double a = (k & 1) ? c : s, b = (k & 1) ? s : c;
  *sn = bits_to_double(hi_bits(a) ^ (((uint32_t)k & 2u) << 30), lo_bits(a));
  *cs = bits_to_double(hi_bits(b) ^ ((((uint32_t)k + 1u) & 2u) << 30), lo_bits(b));
}

}  // namespace avm
