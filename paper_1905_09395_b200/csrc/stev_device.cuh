// stev_device.cuh -- device-side data layout and the STEV integrator kernel (rows a1-a6 of DESIGN.md section 1).
//
// Mapping: G lanes cooperate on one cell (G = 1..32, a power of two, chosen from the
// mechanism size).  Lane l of a group owns species l, l+G, ... and reactions l, l+G, ...  The cell's whole
// working set -- mass fractions, thermo, concentrations, progress rates, the rOF factors and the 13-deep DFT
// history of every reversible reaction -- lives in shared memory for the cell's entire integration, so the hot
// loop has no HBM traffic at all.  The mechanism tables are staged once per block in shared memory by one
// bulk-async (TMA) copy.  Blocks are persistent: a group that retires its cell pulls the next active cell from
// a global queue (warp-ballot + popc prefix, one atomic per warp), which is the variable-load idea of
// PAPER.md:105 without re-launching per iteration.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

#include "stev_math.cuh"

namespace stev {

// ---------------------------------------------------------------------------------------------------------
// Table image: one contiguous device buffer per (mechanism, estimator) pair, copied verbatim to shared
// memory.  Offsets are in bytes from the start of the image.  Reactions are stored in *internal* order:
// the Rrev reversible ones first, then the irreversible ones (each group in the caller's order), so that
// lanes never diverge on reversibility; `orig` maps internal -> caller index.
// ---------------------------------------------------------------------------------------------------------
struct DevTables {
  int S, R, Rrev, n_gather;
  int has_est, H, n_in, n_out, act, input_map;
  float h_ref_T;
  int o_invW, o_W, o_tmid, o_nasa;        // double [S], [S], [S], [2][14][S]
  int o_lnA, o_b, o_Ta, o_dnu;            // double [R] each
  int o_part;                             // uint64 [R]: r0,n0,r1,n1,p0,m0,p1,m1 (one byte each; count 0 = absent)
  int o_orig;                             // uint16 [R]
  int o_gptr, o_gent;                     // uint16 [S+1]; uint32 [n_gather] = internal reaction | (int8 coef) << 16
  int o_eshift, o_escale, o_W1T, o_b1, o_W2T, o_b2;  // float [n_in],[n_in],[n_in][H],[H],[H][n_out],[n_out]
  // real stoichiometric coefficients / rate-law exponents (Eqs 26-29; only if has_real):
  int has_real;
  int o_rcoef, o_rord;                    // double [R][4] each: coefficient / exponent of reactant entries 0, 1 and product entries 0, 1
  int o_gcoef;                            // double [n_gather]: signed coefficient of each gather entry
  int bytes;                              // multiple of 16
};

// NASA table rows (per range): 0..4 a1..a5 | 5..8 a2/2,a3/3,a4/4,a5/5 | 9 a6 | 10..12 a3/2,a4/3,a5/4 | 13 a7
constexpr int kNasaRows = 14;

// Per-cell shared-memory region, offsets in doubles; stride padded so that groups of one warp hit disjoint banks.
struct CellLayout {
  int oY, oConc, oG, oCp, oH, oQ, oRof, oRing, oHid;
  int rrev_pad;   // row length of the ring [13][rrev_pad]
  int stride;     // doubles per cell
};

struct SolverConsts {
  double y_step_max, delta_max, alpha, tol_ring, tol_freq, r_fac, inv_r_fac, rof_min;
  double tol_ring2, ring_lo, ring_hi;   // Tol_ring^2 and the 1 -+ 1e-14 band of the square-root-free ringing test
  int nhf, dft_enable, max_steps, energy_mode;
  int ring_filter_ok;                   // Tol_ring^2 is a normal number far from overflow and underflow
};

struct IntegrateArgs {
  DevTables tb;
  const unsigned char *table;
  CellLayout cl;
  SolverConsts sc;
  double t_f;
  long long n_active;        // entries in the active list of this pass
  const int *list;           // active-cell list (cell indices) or nullptr = identity
  long long ld;
  double *T;
  const double *p;
  double *Y;
  int *steps;
  unsigned char *status;     // may be nullptr
  int *queue_head;           // global work queue position
  int *worst_status;
  int chunk_steps;           // 0 = run to completion
  int restore;               // 1: cells of this pass resume from their spill record
  unsigned char *flags;      // [n_active] by list position: 1 = still active after this pass (chunked only)
  double *spill;             // [n_cells][spill_stride] records: t, steps, slot, rOF[Rrev], ring[13][Rrev]
  long long spill_stride;
};

struct RatesArgs {
  DevTables tb;
  const unsigned char *table;
  CellLayout cl;
  SolverConsts sc;
  long long n, ld;
  const double *T, *p, *Y, *rOF;
  double *dYdt, *dTdt, *q;
};

// ---------------------------------------------------------------------------------------------------------
// Staging of the table image: one elected thread issues a bulk asynchronous global->shared copy (TMA,
// cp.async.bulk) and everyone waits on the mbarrier it signals.
// ---------------------------------------------------------------------------------------------------------
__device__ __forceinline__ void stage_tables(unsigned char *smem_dst, const unsigned char *gsrc, int bytes,
                                             unsigned long long *mbar) {
  unsigned mbar_s = (unsigned)__cvta_generic_to_shared(mbar);
  unsigned dst_s = (unsigned)__cvta_generic_to_shared(smem_dst);
  if (threadIdx.x == 0) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(mbar_s));
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  if (threadIdx.x == 0) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(mbar_s), "r"(bytes) : "memory");
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst_s),
                 "l"(gsrc), "r"(bytes), "r"(mbar_s)
                 : "memory");
  }
  unsigned done = 0;
  while (!done) {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], 0;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(done)
        : "r"(mbar_s)
        : "memory");
  }
}

template <int G>
__device__ __forceinline__ void group_sync() {
  if (G > 1) __syncwarp();
}

// ---------------------------------------------------------------------------------------------------------
// The arithmetic of one precision (DESIGN.md section 5 for binary64, section 5b for binary32: stev_params.state_precision).
// ---------------------------------------------------------------------------------------------------------
template <typename RT> struct MathT;
template <> struct MathT<double> {
  static __device__ __forceinline__ double fma(double a, double b, double c) { return fma_rn(a, b, c); }
  static __device__ __forceinline__ double exp(double x) { return cexp(x); }
  static __device__ __forceinline__ double log(double x) { return clog(x); }
  static __device__ __forceinline__ double sqrt(double x) { return ::sqrt(x); }
  static __device__ __forceinline__ double abs(double x) { return fabs(x); }
  static __device__ __forceinline__ double inf() { return bits_to_double(0x7ff0000000000000ull); }
  static __device__ __forceinline__ double ru() { return kRu; }
  static __device__ __forceinline__ double patm() { return kPatm; }
  static __device__ __forceinline__ double r_floor() { return 1.0e-30; }     // Eq 1
  static __device__ __forceinline__ double y_small() { return 1.0e-20; }     // Eq 2 (R2)
  static __device__ __forceinline__ double ninety() { return 0.9; }          // Eq 2
  static __device__ __forceinline__ double dft_guard() { return 1.0e-300; }  // Eq 10 (R10)
  static __device__ __forceinline__ double land_tol() { return 1.0e-12; }    // R5
  static __device__ __forceinline__ double inv_r_fac(const SolverConsts &sc) { return sc.inv_r_fac; }
};
template <> struct MathT<float> {
  static __device__ __forceinline__ float fma(float a, float b, float c) { return __fmaf_rn(a, b, c); }
  static __device__ __forceinline__ float exp(float x) { return cexpf32(x); }
  static __device__ __forceinline__ float log(float x) { return clogf32(x); }
  static __device__ __forceinline__ float sqrt(float x) { return __fsqrt_rn(x); }
  static __device__ __forceinline__ float abs(float x) { return fabsf(x); }
  static __device__ __forceinline__ float inf() { return __int_as_float(0x7f800000); }
  static __device__ __forceinline__ float ru() { return 0x1.3d2becp+26f; }   // (float) 8.31446261815324e7
  static __device__ __forceinline__ float patm() { return 0x1.eec04p+19f; }  // (float) 1.01325e6
  static __device__ __forceinline__ float r_floor() { return 1.0e-30f; }
  static __device__ __forceinline__ float y_small() { return 1.0e-20f; }
  static __device__ __forceinline__ float ninety() { return 0.9f; }
  static __device__ __forceinline__ float dft_guard() { return 1.0e-30f; }   // R26
  static __device__ __forceinline__ float land_tol() { return 1.0e-6f; }     // R26
  static __device__ __forceinline__ float inv_r_fac(const SolverConsts &sc) { return 1.0f / (float)sc.r_fac; }
};

// min / or across the G lanes of a group (exact: min and or are associative and commutative)
template <int G, typename RT>
__device__ __forceinline__ RT group_min(RT v) {
#pragma unroll
  for (int off = G / 2; off >= 1; off >>= 1) {
    RT o = __shfl_xor_sync(0xffffffffu, v, off);
    v = (o < v) ? o : v;
  }
  return v;
}
template <int G>
__device__ __forceinline__ int group_or(int v) {
#pragma unroll
  for (int off = G / 2; off >= 1; off >>= 1) v |= __shfl_xor_sync(0xffffffffu, v, off);
  return v;
}

// Views of the staged tables.
template <typename RT>
struct TableView {
  const RT *invW, *W, *tmid, *nasa, *lnA, *b, *Ta, *dnu;
  const unsigned long long *part;
  const unsigned short *orig, *gptr;
  const unsigned *gent;
  const float *eshift, *escale, *W1T, *b1, *W2T, *b2;
  const RT *rcoef, *rord, *gcoef;
  __device__ __forceinline__ TableView(const unsigned char *base, const DevTables &tb) {
    rcoef = (const RT *)(base + tb.o_rcoef);
    rord = (const RT *)(base + tb.o_rord);
    gcoef = (const RT *)(base + tb.o_gcoef);
    invW = (const RT *)(base + tb.o_invW);
    W = (const RT *)(base + tb.o_W);
    tmid = (const RT *)(base + tb.o_tmid);
    nasa = (const RT *)(base + tb.o_nasa);
    lnA = (const RT *)(base + tb.o_lnA);
    b = (const RT *)(base + tb.o_b);
    Ta = (const RT *)(base + tb.o_Ta);
    dnu = (const RT *)(base + tb.o_dnu);
    part = (const unsigned long long *)(base + tb.o_part);
    orig = (const unsigned short *)(base + tb.o_orig);
    gptr = (const unsigned short *)(base + tb.o_gptr);
    gent = (const unsigned *)(base + tb.o_gent);
    eshift = (const float *)(base + tb.o_eshift);
    escale = (const float *)(base + tb.o_escale);
    W1T = (const float *)(base + tb.o_W1T);
    b1 = (const float *)(base + tb.o_b1);
    W2T = (const float *)(base + tb.o_W2T);
    b2 = (const float *)(base + tb.o_b2);
  }
};

// f * C^x (Eq 28; R22): x = 1, 2, 3 by repeated multiplication (the mass-action case, contract 5.5), x = 0
// leaves f, any other exponent as exp(x log C) through the contract routines, and C^x = 0 for C <= 0.
template <typename RT>
__device__ __forceinline__ RT times_power(RT f, RT c, RT x) {
  if (x == RT(1)) return f * c;
  if (x == RT(2)) return (f * c) * c;
  if (x == RT(3)) return ((f * c) * c) * c;
  if (x == RT(0)) return f;
  return f * ((c > RT(0)) ? MathT<RT>::exp(x * MathT<RT>::log(c)) : RT(0));
}

// What one right-hand-side evaluation leaves in registers (identical in every lane of the group).
template <typename RT>
struct RhsOut {
  RT c_tot, rho, dTdt, t_star;
};

// ---------------------------------------------------------------------------------------------------------
// Steps 1-6a of DESIGN.md section 2 for one cell, executed by the G lanes of a group.
//   in : T, p (registers, all lanes), cell[oY] mass fractions, cell[oRof] (if use_rof)
//   out: cell[oQ][k] effective progress rates (internal order), cell[oConc][i] := r_i = dY_i/dt,
//        cell[oG][i] := omega_i, RhsOut.  Ends with the group converged and all writes visible.
// ---------------------------------------------------------------------------------------------------------
template <int G, typename RT>
__device__ __forceinline__ RhsOut<RT> rhs_eval(const DevTables &tb, const TableView<RT> &tv, const CellLayout &cl,
                                               const SolverConsts &sc, RT *cell, int gl, RT T, RT p, bool use_rof) {
  using M = MathT<RT>;
  const RT alpha = (RT)sc.alpha, y_step_max = (RT)sc.y_step_max;
  const int S = tb.S, R = tb.R, Rrev = tb.Rrev;
  RT *cY = cell + cl.oY, *cConc = cell + cl.oConc, *cG = cell + cl.oG, *cCp = cell + cl.oCp, *cH = cell + cl.oH;
  RT *cQ = cell + cl.oQ;
  const RT *cRof = cell + cl.oRof;

  // -- a1: thermo (Eqs 15-16, R17).  g/RT always from NASA-7.
  const RT lnT = M::log(T);
  const RT invT = RT(1) / T;
  for (int i = gl; i < S; i += G) {
    const RT *c = tv.nasa + ((T < tv.tmid[i]) ? 0 : kNasaRows * S) + i;
    const RT a1 = c[0], a2 = c[S];
    RT hp = M::fma(M::fma(M::fma(M::fma(c[8 * S], T, c[7 * S]), T, c[6 * S]), T, c[5 * S]), T, a1);
    RT hRT = M::fma(c[9 * S], invT, hp);
    RT sp = M::fma(M::fma(M::fma(c[12 * S], T, c[11 * S]), T, c[10 * S]), T, a2);
    RT sR = M::fma(a1, lnT, M::fma(sp, T, c[13 * S]));
    cG[i] = hRT - sR;
    if (!tb.has_est) {
      cCp[i] = M::fma(M::fma(M::fma(M::fma(c[4 * S], T, c[3 * S]), T, c[2 * S]), T, a2), T, a1);
      cH[i] = hRT;
    }
  }
  // -- a7 (in-integrator, fp32 CUDA cores, R18): cp_i/R and h_i/(R T_ref) from the shallow MLP.
  if (tb.has_est) {
    float *hid = (float *)(cell + cl.oHid);
    const int H = tb.H, n_in = tb.n_in, n_out = tb.n_out;
    for (int jh = gl; jh < H; jh += G) {
      float z = tv.b1[jh];
      for (int k = 0; k < n_in; ++k) {
        const RT raw = (k == 0) ? T : ((k == 1) ? p : cY[k - 2]);
        float x = ((float)raw - tv.eshift[k]) * tv.escale[k];
        z = __fmaf_rn(tv.W1T[k * H + jh], x, z);
      }
      const RT zd = (RT)z;
      float a;
      if (tb.act == 0) a = (float)(RT(1) - RT(2) / (RT(1) + M::exp(RT(2) * zd)));
      else a = (float)(RT(1) / (RT(1) + M::exp(-zd)));
      hid[jh] = a;
    }
    group_sync<G>();
    for (int o = gl; o < n_out; o += G) {
      float y = tv.b2[o];
      for (int jh = 0; jh < H; ++jh) y = __fmaf_rn(tv.W2T[jh * n_out + o], hid[jh], y);
      if (o < S) cCp[o] = (RT)y;
      else cH[o - S] = ((RT)y * (RT)tb.h_ref_T) * invT;
    }
  }
  group_sync<G>();

  // -- mixture sums, sequential in species order (contract 5.4); every lane computes them redundantly.
  RT inv_wbar = RT(0), sum_cp = RT(0);
  for (int i = 0; i < S; ++i) {
    RT y = cY[i], w = tv.invW[i];
    inv_wbar = M::fma(y, w, inv_wbar);
    sum_cp = M::fma(y * w, cCp[i], sum_cp);
  }
  RhsOut<RT> out;
  out.c_tot = p / (M::ru() * T);
  out.rho = out.c_tot / inv_wbar;
  // -- small-species stabilisation (Eqs 6-7, R7): C** = gamma(y) rho y / W
  for (int i = gl; i < S; i += G) {
    RT y = cY[i];
    RT yp = (y > RT(0)) ? y : RT(0);
    RT c = (out.rho * yp) * tv.invW[i];
    if (alpha > RT(0)) c = (yp / (alpha + yp)) * c;
    cConc[i] = c;
  }
  group_sync<G>();

  // -- a2: rate constants and progress rates (Eqs 28-30; Eq 14).  Internal order:
  //    k < Rrev reversible, k >= Rrev irreversible, so the branch below is uniform except at one boundary.
  const RT ln_c0 = M::log(M::patm() / (M::ru() * T));
  for (int k = gl; k < R; k += G) {
    const RT ln_kf = M::fma(-tv.Ta[k], invT, M::fma(tv.b[k], lnT, tv.lnA[k]));
    RT fwd = M::exp(ln_kf);
    const unsigned long long pt = tv.part[k];
    const int r0 = (int)(pt & 0xff), n0 = (int)((pt >> 8) & 0xff), r1 = (int)((pt >> 16) & 0xff), n1 = (int)((pt >> 24) & 0xff);
    const int p0 = (int)((pt >> 32) & 0xff), m0 = (int)((pt >> 40) & 0xff), p1 = (int)((pt >> 48) & 0xff), m1 = (int)((pt >> 56) & 0xff);
    RT qk;
    if (tb.has_real) {
      // real coefficients and exponents (Eqs 26-29): same order of operations as the integer case below
      const RT *co = tv.rcoef + 4 * k, *od = tv.rord + 4 * k;
      fwd = times_power<RT>(fwd, cConc[r0], od[0]);
      if (n1) fwd = times_power<RT>(fwd, cConc[r1], od[1]);
      qk = fwd;
      if (k < Rrev) {
        RT dg = RT(0) - co[0] * cG[r0];
        if (n1) dg = dg - co[1] * cG[r1];
        dg = dg + co[2] * cG[p0];
        if (m1) dg = dg + co[3] * cG[p1];
        const RT ln_kc = M::fma(tv.dnu[k], ln_c0, -dg);
        RT rev = M::exp(ln_kf - ln_kc);
        rev = times_power<RT>(rev, cConc[p0], od[2]);
        if (m1) rev = times_power<RT>(rev, cConc[p1], od[3]);
        qk = (fwd - rev) * (use_rof ? cRof[k] : RT(1));
      }
    } else {
      {
        const RT c0 = cConc[r0];
        for (int n = 0; n < n0; ++n) fwd = fwd * c0;
        if (n1) {
          const RT c1 = cConc[r1];
          for (int n = 0; n < n1; ++n) fwd = fwd * c1;
        }
      }
      qk = fwd;
      if (k < Rrev) {
        RT dg = RT(0) - (RT)n0 * cG[r0];
        if (n1) dg = dg - (RT)n1 * cG[r1];
        dg = dg + (RT)m0 * cG[p0];
        if (m1) dg = dg + (RT)m1 * cG[p1];
        const RT ln_kc = M::fma(tv.dnu[k], ln_c0, -dg);
        RT rev = M::exp(ln_kf - ln_kc);
        const RT d0 = cConc[p0];
        for (int n = 0; n < m0; ++n) rev = rev * d0;
        if (m1) {
          const RT d1 = cConc[p1];
          for (int n = 0; n < m1; ++n) rev = rev * d1;
        }
        qk = (fwd - rev) * (use_rof ? cRof[k] : RT(1));
      }
    }
    cQ[k] = qk;
  }
  group_sync<G>();

  // -- source terms and the step limiter (Eqs 1-3): omega_i gathered in the caller's reaction
  //    order, r_i = W_i omega_i / rho, t* = min_i min(Y_step^max, y_i*) / r_i*.
  const RT inv_rho = RT(1) / out.rho;
  RT t_star = M::inf();
  for (int i = gl; i < S; i += G) {
    RT om = RT(0);
    const int e1 = tv.gptr[i + 1];
    for (int e = tv.gptr[i]; e < e1; ++e) {
      const unsigned ent = tv.gent[e];
      const RT coef = tb.has_real ? tv.gcoef[e] : (RT)(int)(signed char)(ent >> 16);
      om = om + coef * cQ[ent & 0xffffu];
    }
    const RT r = (tv.W[i] * om) * inv_rho;
    const RT y = cY[i];
    const RT r_star = (-r > M::r_floor()) ? -r : M::r_floor();
    const RT y_star = (y < M::y_small()) ? RT(1) : M::ninety() * y;
    const RT lim = ((y_step_max < y_star) ? y_step_max : y_star) / r_star;
    if (lim < t_star) t_star = lim;
    cConc[i] = r;   // concentrations are dead: reuse for dY_i/dt
    cG[i] = om;     // g/RT is dead: reuse for omega_i
  }
  out.t_star = group_min<G, RT>(t_star);
  group_sync<G>();

  // -- temperature equation (R15), enthalpy sum sequential in species order.
  RT sum_h = RT(0);
  for (int i = 0; i < S; ++i) sum_h = M::fma(cH[i], cG[i], sum_h);
  out.dTdt = (sc.energy_mode == 0) ? -((sum_h * M::ru()) * T) / (out.rho * (M::ru() * sum_cp)) : RT(0);
  return out;
}

// ---------------------------------------------------------------------------------------------------------
// a5: DFT ringing detection for one reversible reaction (Eqs 8-13).  x[0..12] is the window in
// physical slot order.  Direct sums with the contract's twiddle literals; the largest high-bin magnitude is
// sqrt(max |.|^2), which equals max sqrt(|.|^2) bit for bit because IEEE sqrt is monotone.
// ---------------------------------------------------------------------------------------------------------
template <int M, typename RT>
__device__ __forceinline__ RT dft_bin_sq(const RT (&x)[kWindow]) {
  RT re = RT(0), im = RT(0);
#pragma unroll
  for (int k = 0; k < kWindow; ++k) {
    re = MathT<RT>::fma(x[k], (RT)cos13((M * k) % kWindow), re);
    im = MathT<RT>::fma(x[k], -(RT)sin13((M * k) % kWindow), im);
  }
  return MathT<RT>::fma(re, re, im * im);
}

template <typename RT>
__device__ __forceinline__ bool dft_is_ringing(const RT (&x)[kWindow], const SolverConsts &sc) {
  RT d0 = RT(0);
#pragma unroll
  for (int k = 0; k < kWindow; ++k) d0 = d0 + x[k];
  d0 = MathT<RT>::abs(d0);
  RT m2 = RT(0), v;
  const int nhf = sc.nhf;
  if (nhf <= 1) { v = dft_bin_sq<1, RT>(x); m2 = (v > m2) ? v : m2; }
  if (nhf <= 2) { v = dft_bin_sq<2, RT>(x); m2 = (v > m2) ? v : m2; }
  if (nhf <= 3) { v = dft_bin_sq<3, RT>(x); m2 = (v > m2) ? v : m2; }
  if (nhf <= 4) { v = dft_bin_sq<4, RT>(x); m2 = (v > m2) ? v : m2; }
  if (nhf <= 5) { v = dft_bin_sq<5, RT>(x); m2 = (v > m2) ? v : m2; }
  { v = dft_bin_sq<6, RT>(x); m2 = (v > m2) ? v : m2; }
  const RT d_hi = MathT<RT>::sqrt(m2);
  const RT guard = MathT<RT>::dft_guard();
  const RT f_ring = d0 / ((d_hi > guard) ? d_hi : guard);
  return (d_hi > guard) && (f_ring < (RT)sc.tol_ring) && (d0 < (RT)sc.tol_freq);   // no high-frequency content: not ringing
}

// ---------------------------------------------------------------------------------------------------------
// The integrator.  One launch = one pass over the active-cell list.
// ---------------------------------------------------------------------------------------------------------
template <int G, typename RT>
__global__ void __launch_bounds__(512) stev_integrate_kernel(const __grid_constant__ IntegrateArgs a) {
  using M = MathT<RT>;
  extern __shared__ __align__(128) unsigned char smem[];
  __shared__ unsigned long long mbar;
  stage_tables(smem, a.table, a.tb.bytes, &mbar);
  const DevTables &tb = a.tb;
  const CellLayout &cl = a.cl;
  const SolverConsts &sc = a.sc;
  const TableView<RT> tv(smem, tb);
  const int S = tb.S, Rrev = tb.Rrev;

  const int lane = threadIdx.x & 31;
  const int gl = lane % G;                    // lane within the group
  const int grp = lane / G;                   // group within the warp
  RT *cell = (RT *)(smem + tb.bytes) + (size_t)(threadIdx.x / G) * cl.stride;
  RT *cY = cell + cl.oY, *cConc = cell + cl.oConc, *cQ = cell + cl.oQ, *cRof = cell + cl.oRof, *cRing = cell + cl.oRing;
  const int rp = cl.rrev_pad;

  const RT t_f = (RT)a.t_f;
  const RT dt_max = t_f * (RT)sc.delta_max;     // Eq 4
  const RT t_tol = M::land_tol() * t_f;         // R5 (R26 in binary32)
  const RT r_fac = (RT)sc.r_fac, inv_r_fac = M::inv_r_fac(sc), rof_floor = (RT)sc.rof_min;

  // per-cell scalars, identical in all lanes of the group
  RT T = RT(1000), p = M::patm(), t = RT(0);
  int steps = 0, steps_in_pass = 0, slot = 0, cell_idx = -1;
  long long pos = -1;
  bool need = true, active = false, exhausted = false;

  for (;;) {
    // ---- a6: variable load.  Groups whose cell retired pull the next active cell: ballot the requests,
    //      one atomic per warp reserves that many queue positions, popc of the lower mask ranks them.
    const unsigned req = __ballot_sync(0xffffffffu, need && !exhausted && gl == 0);
    if (req) {
      int base = 0;
      if (lane == 0) base = atomicAdd(a.queue_head, __popc(req));
      base = __shfl_sync(0xffffffffu, base, 0);
      if (need && !exhausted) {
        pos = (long long)base + __popc(req & ((1u << (grp * G)) - 1u));
        if (pos < a.n_active) {
          cell_idx = a.list ? a.list[pos] : (int)pos;
          T = (RT)a.T[cell_idx];
          p = (RT)a.p[cell_idx];
          for (int i = gl; i < S; i += G) cY[i] = (RT)a.Y[(long long)i * a.ld + cell_idx];
          steps_in_pass = 0;
          if (a.restore) {
            const double *rec = a.spill + (long long)cell_idx * a.spill_stride;
            t = (RT)rec[0];
            steps = (int)rec[1];
            slot = (int)rec[2];
            for (int k = gl; k < Rrev; k += G) cRof[k] = (RT)rec[3 + k];
            for (int s = 0; s < kWindow; ++s)
              for (int k = gl; k < Rrev; k += G) cRing[s * rp + k] = (RT)rec[3 + Rrev + s * Rrev + k];
          } else {
            t = RT(0);
            steps = 0;
            slot = 0;
            for (int k = gl; k < Rrev; k += G) cRof[k] = RT(1);                     // Eq 11
            for (int s = 0; s < kWindow; ++s)
              for (int k = gl; k < Rrev; k += G) cRing[s * rp + k] = RT(0);         // R10
          }
          active = true;
        } else {
          exhausted = true;
          active = false;
        }
        need = false;
      }
      __syncwarp();
    }
    if (!__any_sync(0xffffffffu, active)) break;

    // ---- a1, a2, a3: right-hand side and limiter
    const RhsOut<RT> rhs = rhs_eval<G, RT>(tb, tv, cl, sc, cell, gl, T, p, true);

    // ---- a3: step size (Eq 5) and landing on t_f (R5)
    RT h = (rhs.t_star < dt_max) ? rhs.t_star : dt_max;
    bool last = false;
    const RT rem = t_f - t;
    if (rem - h < t_tol) {
      h = rem;
      last = true;
    }

    // ---- a4: forward Euler (Eq 18)
    int bad = 0;
    for (int i = gl; i < S; i += G) {
      const RT y = M::fma(h, cConc[i], cY[i]);
      cY[i] = y;
      bad |= !(y - y == RT(0));
    }
    T = M::fma(h, rhs.dTdt, T);
    t = last ? t_f : t + h;
    steps += 1;
    steps_in_pass += 1;
    bad |= !(T - T == RT(0));

    // ---- a5: DFT stabilisation (Eqs 8-14): store the applied change in progress (R8, R9), test, update rOF
    if (sc.dft_enable) {
      const RT inv_ctot = RT(1) / rhs.c_tot;
      for (int k = gl; k < Rrev; k += G) {
        cRing[slot * rp + k] = (cQ[k] * h) * inv_ctot;
        RT x[kWindow];
#pragma unroll
        for (int s = 0; s < kWindow; ++s) x[s] = cRing[s * rp + k];
        const bool ringing = dft_is_ringing<RT>(x, sc);
        RT rof = cRof[k] * (ringing ? inv_r_fac : r_fac);
        if (rof > RT(1)) rof = RT(1);
        if (rof < rof_floor) rof = rof_floor;
        cRof[k] = rof;
      }
      slot = (slot + 1 == kWindow) ? 0 : slot + 1;
    }

    // ---- a6: retirement (R20)
    bad = group_or<G>(bad);
    int st = -1;
    if (bad) st = 2;            // checked first: a landing step that produced a non-finite state is not "finished"
    else if (last) st = 0;
    else if (steps >= sc.max_steps) st = 1;
    const bool pause = (st < 0) && a.chunk_steps > 0 && steps_in_pass >= a.chunk_steps;
    if (active && (st >= 0 || pause)) {
      for (int i = gl; i < S; i += G) a.Y[(long long)i * a.ld + cell_idx] = (double)cY[i];
      if (gl == 0) {
        a.T[cell_idx] = (double)T;
        a.steps[cell_idx] = steps;
        if (st >= 0 && a.status) a.status[cell_idx] = (unsigned char)st;
        if (st > 0) atomicMax(a.worst_status, st);
        if (a.flags) a.flags[pos] = pause ? 1 : 0;
      }
      if (pause) {
        double *rec = a.spill + (long long)cell_idx * a.spill_stride;
        if (gl == 0) {
          rec[0] = (double)t;
          rec[1] = (double)steps;
          rec[2] = (double)slot;
        }
        for (int k = gl; k < Rrev; k += G) rec[3 + k] = (double)cRof[k];
        for (int s = 0; s < kWindow; ++s)
          for (int k = gl; k < Rrev; k += G) rec[3 + Rrev + s * Rrev + k] = (double)cRing[s * rp + k];
      }
      need = true;
      active = false;
    }
    group_sync<G>();
  }
}

// ---------------------------------------------------------------------------------------------------------
// Test export: one right-hand-side evaluation per cell with the same device code.
// ---------------------------------------------------------------------------------------------------------
template <int G, typename RT>
__global__ void __launch_bounds__(512) stev_rates_kernel(const __grid_constant__ RatesArgs a) {
  extern __shared__ __align__(128) unsigned char smem[];
  __shared__ unsigned long long mbar;
  stage_tables(smem, a.table, a.tb.bytes, &mbar);
  const DevTables &tb = a.tb;
  const CellLayout &cl = a.cl;
  const TableView<RT> tv(smem, tb);
  const int S = tb.S, R = tb.R, Rrev = tb.Rrev;
  const int gl = (threadIdx.x & 31) % G;
  RT *cell = (RT *)(smem + tb.bytes) + (size_t)(threadIdx.x / G) * cl.stride;
  const long long cells_per_block = blockDim.x / G;
  for (long long base = (long long)blockIdx.x * cells_per_block; base < a.n; base += (long long)gridDim.x * cells_per_block) {
    const long long c = base + threadIdx.x / G;
    const bool valid = c < a.n;
    const long long cc = valid ? c : a.n - 1;
    const RT T = (RT)a.T[cc], p = (RT)a.p[cc];
    for (int i = gl; i < S; i += G) cell[cl.oY + i] = (RT)a.Y[(long long)i * a.ld + cc];
    for (int k = gl; k < Rrev; k += G) cell[cl.oRof + k] = a.rOF ? (RT)a.rOF[(long long)tv.orig[k] * a.ld + cc] : RT(1);
    group_sync<G>();
    const RhsOut<RT> rhs = rhs_eval<G, RT>(tb, tv, cl, a.sc, cell, gl, T, p, true);
    if (valid) {
      for (int i = gl; i < S; i += G) a.dYdt[(long long)i * a.ld + c] = (double)cell[cl.oConc + i];
      for (int k = gl; k < R; k += G) a.q[(long long)tv.orig[k] * a.ld + c] = (double)cell[cl.oQ + k];
      if (gl == 0) a.dTdt[c] = (double)rhs.dTdt;
    }
    group_sync<G>();
  }
}

}  // namespace stev
