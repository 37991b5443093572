// stev_fast.cuh -- device helpers shared by the large-mechanism integrator kernels: the contract's exp / log with their
// coefficients in the constant bank, DFT window statistics, the square-root-free ringing filter, tensor-memory and
// named-barrier wrappers.  Arithmetic is the contract's, operation for operation.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

#include "stev_device.cuh"
#include "stev_math.cuh"

namespace stev {

// Twiddles of DESIGN.md 5.6 and the contract's exp / log coefficients in constant memory.  The arrays
// are deliberately NOT const-qualified: a const array is folded into 64-bit immediates, which sm_100 has to build with
// two moves per DFMA; a plain __constant__ array stays a constant-bank operand of the DFMA itself (no extra
// instruction, no register).  Nothing ever writes them.
static __device__ __constant__ double kTwCos[13] = {
    1.0, 0.8854560256532099, 0.5680647467311559, 0.120536680255323, -0.35460488704253545,
    -0.7485107481711012, -0.970941817426052, -0.9709418174260521, -0.7485107481711013,
    -0.3546048870425359, 0.1205366802553232, 0.5680647467311548, 0.88545602565321};
static __device__ __constant__ double kTwNegSin[13] = {
    -0.0, -0.4647231720437685, -0.8229838658936564, -0.992708874098054, -0.9350162426854148,
    -0.6631226582407952, -0.23931566428755768, 0.23931566428755743, 0.663122658240795,
    0.9350162426854147, 0.992708874098054, 0.822983865893657, 0.4647231720437684};
// exp: [0] log2 e, [1] 1.5*2^52, [2] ln2_hi, [3] ln2_lo, [4..17] 1/13! .. 1/0!
static __device__ __constant__ double kExpC[18] = {
    1.4426950408889634, 6755399441055744.0, 6.93147180369123816490e-01, 1.90821492927058770002e-10,
    1.6059043836821613e-10, 2.08767569878681e-09, 2.505210838544172e-08, 2.755731922398589e-07,
    2.7557319223985893e-06, 2.48015873015873e-05, 0.0001984126984126984, 0.001388888888888889,
    0.008333333333333333, 0.041666666666666664, 0.16666666666666666, 0.5, 1.0, 1.0};
// log: [0] sqrt 2, [1] ln2_hi, [2] ln2_lo, [3..13] 1/23, 1/21, .. 1/3
static __device__ __constant__ double kLogC[14] = {
    1.4142135623730951, 6.93147180369123816490e-01, 1.90821492927058770002e-10,
    0.043478260869565216, 0.047619047619047616, 0.05263157894736842, 0.058823529411764705,
    0.06666666666666667, 0.07692307692307693, 0.09090909090909091, 0.1111111111111111,
    0.14285714285714285, 0.2, 0.3333333333333333};

// The contract's exp (same operations, same order as stev_math.cuh / DESIGN.md 5.3).  p * 2^k is formed by adding k
// to the exponent field of p, which is the same number whenever the product is a normal double: p lies in
// [0.70, 1.42] and |x| <= 708 gives |k| <= 1022 with e^x >= 2^-1021.4.  Everything else takes the generic routine.
__device__ __forceinline__ double ab_exp(double x) {
  if (__builtin_expect(!(fabs(x) <= 708.0), 0)) return cexp(x);
  const double t = fma_rn(x, kExpC[0], kExpC[1]);
  const double k = t - kExpC[1];
  double r = fma_rn(-k, kExpC[2], x);
  r = fma_rn(-k, kExpC[3], r);
  double p = kExpC[4];
#pragma unroll
  for (int n = 5; n < 18; ++n) p = fma_rn(p, r, kExpC[n]);
  const int ki = __double2loint(t);
  return __hiloint2double(__double2hiint(p) + ki * 1048576, __double2loint(p));
}

// The contract's log for positive finite normal x (T and p_atm/(R_u T) on this path); other inputs take the generic routine.
__device__ __forceinline__ double ab_log(double x) {
  const int hi = __double2hiint(x);
  if (__builtin_expect(hi < 0x00100000 || hi >= 0x7ff00000, 0)) return clog(x);
  int e = (hi >> 20) - 1023;
  double m = __hiloint2double((hi & 0x000fffff) | 0x3ff00000, __double2loint(x));
  if (m > kLogC[0]) {
    m = m * 0.5;
    e = e + 1;
  }
  const double f = (m - 1.0) / (m + 1.0);
  const double s = f * f;
  double P = kLogC[3];
#pragma unroll
  for (int n = 4; n < 14; ++n) P = fma_rn(P, s, kLogC[n]);
  const double two_f = f + f;
  const double log_m = fma_rn(two_f, s * P, two_f);
  const double ed = (double)e;
  return fma_rn(ed, kLogC[1], fma_rn(ed, kLogC[2], log_m));
}

__device__ __forceinline__ void named_bar_sync(int id) { asm volatile("bar.sync %0, 64;" ::"r"(id) : "memory"); }
__device__ __forceinline__ void named_bar_arrive(int id) { asm volatile("bar.arrive %0, 64;" ::"r"(id) : "memory"); }

__device__ __forceinline__ void tmem_st2(uint32_t taddr, double v) {
  asm volatile("tcgen05.st.sync.aligned.32x32b.x2.b32 [%0], {%1, %2};" ::"r"(taddr), "r"((uint32_t)__double2loint(v)),
               "r"((uint32_t)__double2hiint(v))
               : "memory");
}
__device__ __forceinline__ void tmem_wait_st() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ void tmem_wait_ld() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ double lds_f64(const unsigned char *base, unsigned off) { return *(const double *)(base + off); }

// exp without the range check (the caller checks |x| <= 708 for the whole batch and falls back to ab_exp)
__device__ __forceinline__ double ab_exp_core(double x) {
  const double t = fma_rn(x, kExpC[0], kExpC[1]);
  const double k = t - kExpC[1];
  double r = fma_rn(-k, kExpC[2], x);
  r = fma_rn(-k, kExpC[3], r);
  double p = kExpC[4];
#pragma unroll
  for (int n = 5; n < 18; ++n) p = fma_rn(p, r, kExpC[n]);
  return __hiloint2double(__double2hiint(p) + __double2loint(t) * 1048576, __double2loint(p));
}
__device__ __forceinline__ bool ab_exp_out_of_range(double x) { return !(fabs(x) <= 708.0); }

// 13 doubles = 26 consecutive columns of this lane, issued as x16 + x8 + x2 (no wait)
__device__ __forceinline__ void tmem_ld26(uint32_t taddr, uint32_t (&r)[26]) {
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
      : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]), "=r"(r[9]),
        "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
      : "r"(taddr)
      : "memory");
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
               : "=r"(r[16]), "=r"(r[17]), "=r"(r[18]), "=r"(r[19]), "=r"(r[20]), "=r"(r[21]), "=r"(r[22]), "=r"(r[23])
               : "r"(taddr + 16)
               : "memory");
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x2.b32 {%0,%1}, [%2];" : "=r"(r[24]), "=r"(r[25]) : "r"(taddr + 24) : "memory");
}
__device__ __forceinline__ void unpack_window(const uint32_t (&r)[26], double (&x)[kWindow]) {
#pragma unroll
  for (int s = 0; s < kWindow; ++s) x[s] = __hiloint2double((int)r[2 * s + 1], (int)r[2 * s]);
}

// |X_M|^2 of the window (Eq 9).  The k = 0 terms of the contract's sums are fma(x0, 1, 0) = x0 and
// fma(x0, -0, 0) = +0 for every finite x0, so the sums start from them (a non-finite sample only occurs in the step
// that retires the cell with status 2, whose DFT is not evaluated).
template <int M>
__device__ __forceinline__ double ab_bin_sq(const double (&x)[kWindow]) {
  double re = x[0], im = 0.0;
#pragma unroll
  for (int k = 1; k < kWindow; ++k) {
    re = fma_rn(x[k], kTwCos[(M * k) % kWindow], re);
    im = fma_rn(x[k], kTwNegSin[(M * k) % kWindow], im);
  }
  return fma_rn(re, re, im * im);
}

// D^0 = |sum x| and the largest |X_m|^2 over the high bins NHF..6 (Eqs 9-10).  max of sqrt = sqrt of max (IEEE sqrt
// is monotone), so one square root at most is needed per window.
template <int NHF>
__device__ __forceinline__ void ab_window_stats(const double (&x)[kWindow], double &d0, double &m2) {
  double s = x[0];
#pragma unroll
  for (int k = 1; k < kWindow; ++k) s = s + x[k];
  d0 = fabs(s);
  double m = 0.0, v;   // the contract's running maximum starts at 0 and ignores NaN
  if (NHF <= 1) { v = ab_bin_sq<1>(x); m = (v > m) ? v : m; }
  if (NHF <= 2) { v = ab_bin_sq<2>(x); m = (v > m) ? v : m; }
  if (NHF <= 3) { v = ab_bin_sq<3>(x); m = (v > m) ? v : m; }
  if (NHF <= 4) { v = ab_bin_sq<4>(x); m = (v > m) ? v : m; }
  if (NHF <= 5) { v = ab_bin_sq<5>(x); m = (v > m) ? v : m; }
  { v = ab_bin_sq<6>(x); m = (v > m) ? v : m; }
  m2 = m;
}

// Eq 10 + Eq 12 exactly as written: f_ring = D^0 / max(sqrt(m2), 1e-300) < Tol_ring and D^0 < Tol_freq.
__device__ __forceinline__ bool ab_ring_exact(double d0, double m2, const SolverConsts &sc) {
  const double d_hi = sqrt(m2);
  const double f_ring = d0 / ((d_hi > 1.0e-300) ? d_hi : 1.0e-300);
  return (d_hi > 1.0e-300) && (f_ring < sc.tol_ring) && (d0 < sc.tol_freq);   // no high-frequency content: not ringing
}
// The same decision without the square root and the division whenever it is not close: with u = 2^-53,
// fl(d0/fl(sqrt m2)) = (d0/sqrt m2)(1 + 2.1u) at worst, while d0^2 and Tol_ring^2 m2 are each formed with at most
// three roundings, so  d0^2 < Tol_ring^2 m2 (1 - 1e-14)  implies f_ring < Tol_ring (1 - 4e-15) < Tol_ring, and
// symmetrically for >.  `sure` is false inside that band, when m2 leaves [2^-900, 2^901) (read off its exponent field:
// with 1e-9 < Tol_ring < 1e9, checked on the host, neither m2 nor Tol_ring^2 m2 is then near underflow, overflow or the
// 1e-300 guard) and for NaN (exponent field 0x7ff); the caller then evaluates ab_ring_exact.
__device__ __forceinline__ bool ab_ring_filter(double d0, double m2, const SolverConsts &sc, bool &sure) {
  const double lhs = d0 * d0, rhs = sc.tol_ring2 * m2;
  const bool below = lhs < rhs * sc.ring_lo, above = lhs > rhs * sc.ring_hi;
  const bool in_range = (((unsigned)__double2hiint(m2) >> 20) - 123u) < 1801u;   // m2 is +0, positive or NaN: no sign bit
  const bool small = d0 < sc.tol_freq;
  sure = !small || (sc.ring_filter_ok && in_range && (below || above));
  return below && small;
}

}  // namespace stev
