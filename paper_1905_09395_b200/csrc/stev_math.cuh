// stev_math.cuh -- the arithmetic contract's device routines.
//
// STEV trajectories on stiff mechanisms amplify one-ulp differences into different step counts
// (SURVEY.md H1), so every floating-point operation on the integration path is fixed by the
// contract: explicit fused multiply-adds where stated, IEEE round-to-nearest +,*,/,sqrt elsewhere
// (this library is compiled with --fmad=false), and exp/log built from those plus bit operations.
// This file is the CUDA side's own implementation of DESIGN.md 5.3; nothing here is shared with the
// CPU oracle.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace stev {

constexpr double kRu = 8.31446261815324e7;  // erg/(mol K)      (R21)
constexpr double kRcal = 1.98720425864083;  // cal/(mol K)      (R21)
constexpr double kPatm = 1.01325e6;         // dyn/cm^2         (R21)
constexpr int kWindow = 13;

__host__ __device__ __forceinline__ double fma_rn(double a, double b, double c) {
#ifdef __CUDA_ARCH__
  return __fma_rn(a, b, c);
#else
  return __builtin_fma(a, b, c);
#endif
}

__host__ __device__ __forceinline__ double bits_to_double(unsigned long long u) {
#ifdef __CUDA_ARCH__
  return __longlong_as_double((long long)u);
#else
  double d;
  __builtin_memcpy(&d, &u, 8);
  return d;
#endif
}

__host__ __device__ __forceinline__ unsigned long long double_to_bits(double d) {
#ifdef __CUDA_ARCH__
  return (unsigned long long)__double_as_longlong(d);
#else
  unsigned long long u;
  __builtin_memcpy(&u, &d, 8);
  return u;
#endif
}

// exp(x): k = rint(x log2 e) through the 1.5*2^52 shift, two-step Cody-Waite reduction with
// fdlibm's ln2 split, Taylor polynomial of degree 13 (Horner, fma), scaling by 2^k in the exponent field.
// x > 709 -> +inf, x < -708 -> 0 (never a subnormal result), NaN -> NaN.
__host__ __device__ __forceinline__ double cexp(double x) {
  const double kShift = 6755399441055744.0;
  double t = fma_rn(x, 1.4426950408889634, kShift);
  double k = t - kShift;
  double r = fma_rn(-k, 6.93147180369123816490e-01, x);
  r = fma_rn(-k, 1.90821492927058770002e-10, r);
  double p = 1.6059043836821613e-10;
  p = fma_rn(p, r, 2.08767569878681e-09);
  p = fma_rn(p, r, 2.505210838544172e-08);
  p = fma_rn(p, r, 2.755731922398589e-07);
  p = fma_rn(p, r, 2.7557319223985893e-06);
  p = fma_rn(p, r, 2.48015873015873e-05);
  p = fma_rn(p, r, 0.0001984126984126984);
  p = fma_rn(p, r, 0.001388888888888889);
  p = fma_rn(p, r, 0.008333333333333333);
  p = fma_rn(p, r, 0.041666666666666664);
  p = fma_rn(p, r, 0.16666666666666666);
  p = fma_rn(p, r, 0.5);
  p = fma_rn(p, r, 1.0);
  p = fma_rn(p, r, 1.0);
  // 2^k: the low word of t holds k in two's complement; k + 1023 lands in the exponent field
  int ki = (int)(unsigned)(double_to_bits(t) & 0xffffffffull);
  double two_k = bits_to_double((unsigned long long)(long long)(ki + 1023) << 52);
  double res = p * two_k;
  if (x > 709.0) res = bits_to_double(0x7ff0000000000000ull);
  if (x < -708.0) res = 0.0;
  if (x != x) res = x;
  return res;
}

// log(x) for positive finite x: x = m 2^e, m in (sqrt(1/2), sqrt 2], f = (m-1)/(m+1),
// log m = 2f (1 + s/3 + ... + s^11/23) with s = f^2, result = e ln2_hi + (e ln2_lo + log m).
__host__ __device__ __forceinline__ double clog(double x) {
  unsigned long long u = double_to_bits(x);
  int e = (int)(u >> 52) - 1023;
  double m = bits_to_double((u & 0x000fffffffffffffull) | 0x3ff0000000000000ull);
  if (m > 1.4142135623730951) {
    m = m * 0.5;
    e = e + 1;
  }
  double f = (m - 1.0) / (m + 1.0);
  double s = f * f;
  double P = 0.043478260869565216;
  P = fma_rn(P, s, 0.047619047619047616);
  P = fma_rn(P, s, 0.05263157894736842);
  P = fma_rn(P, s, 0.058823529411764705);
  P = fma_rn(P, s, 0.06666666666666667);
  P = fma_rn(P, s, 0.07692307692307693);
  P = fma_rn(P, s, 0.09090909090909091);
  P = fma_rn(P, s, 0.1111111111111111);
  P = fma_rn(P, s, 0.14285714285714285);
  P = fma_rn(P, s, 0.2);
  P = fma_rn(P, s, 0.3333333333333333);
  double two_f = f + f;
  double log_m = fma_rn(two_f, s * P, two_f);
  double ed = (double)e;
  double res = fma_rn(ed, 6.93147180369123816490e-01, fma_rn(ed, 1.90821492927058770002e-10, log_m));
  if (x == 0.0) res = -bits_to_double(0x7ff0000000000000ull);
  if (x < 0.0 || x != x) res = bits_to_double(0x7ff8000000000000ull);
  if (x == bits_to_double(0x7ff0000000000000ull)) res = x;
  return res;
}

// The binary32 contract (stev_params.state_precision = STEV_STATE_FP32).
// exp: k = rint(x log2 e) through the 1.5 * 2^23 shift, Cody-Waite reduction with ln2_hi = 0x1.62e4p-1 (11 trailing zero
// bits), Taylor polynomial of degree 7 (Horner, fmaf), 2^k through the exponent field; > 88 -> +inf, < -87 -> 0.
__host__ __device__ __forceinline__ float fmaf_rn(float a, float b, float c) {
#ifdef __CUDA_ARCH__
  return __fmaf_rn(a, b, c);
#else
  return __builtin_fmaf(a, b, c);
#endif
}
__host__ __device__ __forceinline__ unsigned float_to_bits(float f) {
  unsigned u;
  __builtin_memcpy(&u, &f, 4);
  return u;
}
__host__ __device__ __forceinline__ float bits_to_float(unsigned u) {
  float f;
  __builtin_memcpy(&f, &u, 4);
  return f;
}
__host__ __device__ __forceinline__ float cexpf32(float x) {
  const float kShift = 12582912.0f;
  float t = fmaf_rn(x, 0x1.715476p+0f, kShift);
  float k = t - kShift;
  int ki = (int)(float_to_bits(t) & 0x7fffffu) - 0x400000;
  float r = fmaf_rn(-k, 0x1.62e4p-1f, x);
  r = fmaf_rn(-k, 0x1.7f7d1cp-20f, r);
  float p = 0x1.a01a02p-13f;
  p = fmaf_rn(p, r, 0x1.6c16c2p-10f);
  p = fmaf_rn(p, r, 0x1.111112p-7f);
  p = fmaf_rn(p, r, 0x1.555556p-5f);
  p = fmaf_rn(p, r, 0x1.555556p-3f);
  p = fmaf_rn(p, r, 0.5f);
  p = fmaf_rn(p, r, 1.0f);
  p = fmaf_rn(p, r, 1.0f);
  float res = p * bits_to_float((unsigned)(ki + 127) << 23);
  if (x > 88.0f) res = bits_to_float(0x7f800000u);
  if (x < -87.0f) res = 0.0f;
  if (x != x) res = x;
  return res;
}
// log for positive normal x: x = m 2^e, m in (sqrt(1/2), sqrt 2], f = (m-1)/(m+1), log m = 2f (1 + s/3 + s^2/5 + s^3/7 + s^4/9)
__host__ __device__ __forceinline__ float clogf32(float x) {
  unsigned u = float_to_bits(x);
  int e = (int)(u >> 23) - 127;
  float m = bits_to_float((u & 0x007fffffu) | 0x3f800000u);
  if (m > 0x1.6a09e6p+0f) {
    m = m * 0.5f;
    e = e + 1;
  }
  float f = (m - 1.0f) / (m + 1.0f);
  float s = f * f;
  float P = 0x1.c71c72p-4f;
  P = fmaf_rn(P, s, 0x1.24924ap-3f);
  P = fmaf_rn(P, s, 0x1.99999ap-3f);
  P = fmaf_rn(P, s, 0x1.555556p-2f);
  float two_f = f + f;
  float log_m = fmaf_rn(two_f, s * P, two_f);
  float ed = (float)e;
  float res = fmaf_rn(ed, 0x1.62e4p-1f, fmaf_rn(ed, 0x1.7f7d1cp-20f, log_m));
  if (x == 0.0f) res = -bits_to_float(0x7f800000u);
  if (x < 0.0f || x != x) res = bits_to_float(0x7fc00000u);
  if (x == bits_to_float(0x7f800000u)) res = x;
  return res;
}

// cos, sin of 2 pi n / 13, n = 0..12: the literal table of DESIGN.md 5.6.
__device__ __constant__ const double kCos13[13] = {
    1.0, 0.8854560256532099, 0.5680647467311559, 0.120536680255323, -0.35460488704253545,
    -0.7485107481711012, -0.970941817426052, -0.9709418174260521, -0.7485107481711013,
    -0.3546048870425359, 0.1205366802553232, 0.5680647467311548, 0.88545602565321};
__device__ __constant__ const double kSin13[13] = {
    0.0, 0.4647231720437685, 0.8229838658936564, 0.992708874098054, 0.9350162426854148,
    0.6631226582407952, 0.23931566428755768, -0.23931566428755743, -0.663122658240795,
    -0.9350162426854147, -0.992708874098054, -0.822983865893657, -0.4647231720437684};

// Same literals as compile-time constants, for fully unrolled DFT code (immediates instead of loads).
__host__ __device__ constexpr double cos13(int n) {
  constexpr double t[13] = {1.0, 0.8854560256532099, 0.5680647467311559, 0.120536680255323, -0.35460488704253545,
                            -0.7485107481711012, -0.970941817426052, -0.9709418174260521, -0.7485107481711013,
                            -0.3546048870425359, 0.1205366802553232, 0.5680647467311548, 0.88545602565321};
  return t[n];
}
__host__ __device__ constexpr double sin13(int n) {
  constexpr double t[13] = {0.0, 0.4647231720437685, 0.8229838658936564, 0.992708874098054, 0.9350162426854148,
                            0.6631226582407952, 0.23931566428755768, -0.23931566428755743, -0.663122658240795,
                            -0.9350162426854147, -0.992708874098054, -0.822983865893657, -0.4647231720437684};
  return t[n];
}

}  // namespace stev
