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

// min / or across the G lanes of a group (exact: min and or are associative and commutative)
template <int G>
__device__ __forceinline__ double group_min(double v) {
#pragma unroll
  for (int off = G / 2; off >= 1; off >>= 1) {
    double o = __shfl_xor_sync(0xffffffffu, v, off);
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
struct TableView {
  const double *invW, *W, *tmid, *nasa, *lnA, *b, *Ta, *dnu;
  const unsigned long long *part;
  const unsigned short *orig, *gptr;
  const unsigned *gent;
  const float *eshift, *escale, *W1T, *b1, *W2T, *b2;
  const double *rcoef, *rord, *gcoef;
  __device__ __forceinline__ TableView(const unsigned char *base, const DevTables &tb) {
    rcoef = (const double *)(base + tb.o_rcoef);
    rord = (const double *)(base + tb.o_rord);
    gcoef = (const double *)(base + tb.o_gcoef);
    invW = (const double *)(base + tb.o_invW);
    W = (const double *)(base + tb.o_W);
    tmid = (const double *)(base + tb.o_tmid);
    nasa = (const double *)(base + tb.o_nasa);
    lnA = (const double *)(base + tb.o_lnA);
    b = (const double *)(base + tb.o_b);
    Ta = (const double *)(base + tb.o_Ta);
    dnu = (const double *)(base + tb.o_dnu);
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
__device__ __forceinline__ double times_power(double f, double c, double x) {
  if (x == 1.0) return f * c;
  if (x == 2.0) return (f * c) * c;
  if (x == 3.0) return ((f * c) * c) * c;
  if (x == 0.0) return f;
  return f * ((c > 0.0) ? cexp(x * clog(c)) : 0.0);
}

// What one right-hand-side evaluation leaves in registers (identical in every lane of the group).
struct RhsOut {
  double c_tot, rho, dTdt, t_star;
};

// ---------------------------------------------------------------------------------------------------------
// Steps 1-6a of DESIGN.md section 2 for one cell, executed by the G lanes of a group.
//   in : T, p (registers, all lanes), cell[oY] mass fractions, cell[oRof] (if use_rof)
//   out: cell[oQ][k] effective progress rates (internal order), cell[oConc][i] := r_i = dY_i/dt,
//        cell[oG][i] := omega_i, RhsOut.  Ends with the group converged and all writes visible.
// ---------------------------------------------------------------------------------------------------------
template <int G>
__device__ __forceinline__ RhsOut rhs_eval(const DevTables &tb, const TableView &tv, const CellLayout &cl,
                                           const SolverConsts &sc, double *cell, int gl, double T, double p,
                                           bool use_rof) {
  const int S = tb.S, R = tb.R, Rrev = tb.Rrev;
  double *cY = cell + cl.oY, *cConc = cell + cl.oConc, *cG = cell + cl.oG, *cCp = cell + cl.oCp, *cH = cell + cl.oH;
  double *cQ = cell + cl.oQ;
  const double *cRof = cell + cl.oRof;

  // -- a1: thermo (Eqs 15-16, R17).  g/RT always from NASA-7.
  const double lnT = clog(T);
  const double invT = 1.0 / T;
  for (int i = gl; i < S; i += G) {
    const double *c = tv.nasa + ((T < tv.tmid[i]) ? 0 : kNasaRows * S) + i;
    const double a1 = c[0], a2 = c[S];
    double hp = fma_rn(fma_rn(fma_rn(fma_rn(c[8 * S], T, c[7 * S]), T, c[6 * S]), T, c[5 * S]), T, a1);
    double hRT = fma_rn(c[9 * S], invT, hp);
    double sp = fma_rn(fma_rn(fma_rn(c[12 * S], T, c[11 * S]), T, c[10 * S]), T, a2);
    double sR = fma_rn(a1, lnT, fma_rn(sp, T, c[13 * S]));
    cG[i] = hRT - sR;
    if (!tb.has_est) {
      cCp[i] = fma_rn(fma_rn(fma_rn(fma_rn(c[4 * S], T, c[3 * S]), T, c[2 * S]), T, a2), T, a1);
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
        double raw = (k == 0) ? T : ((k == 1) ? p : cY[k - 2]);
        float x = ((float)raw - tv.eshift[k]) * tv.escale[k];
        z = __fmaf_rn(tv.W1T[k * H + jh], x, z);
      }
      double zd = (double)z;
      float a;
      if (tb.act == 0) a = (float)(1.0 - 2.0 / (1.0 + cexp(2.0 * zd)));
      else a = (float)(1.0 / (1.0 + cexp(-zd)));
      hid[jh] = a;
    }
    group_sync<G>();
    for (int o = gl; o < n_out; o += G) {
      float y = tv.b2[o];
      for (int jh = 0; jh < H; ++jh) y = __fmaf_rn(tv.W2T[jh * n_out + o], hid[jh], y);
      if (o < S) cCp[o] = (double)y;
      else cH[o - S] = ((double)y * (double)tb.h_ref_T) * invT;
    }
  }
  group_sync<G>();

  // -- mixture sums, sequential in species order (contract 5.4); every lane computes them redundantly.
  double inv_wbar = 0.0, sum_cp = 0.0;
  for (int i = 0; i < S; ++i) {
    double y = cY[i], w = tv.invW[i];
    inv_wbar = fma_rn(y, w, inv_wbar);
    sum_cp = fma_rn(y * w, cCp[i], sum_cp);
  }
  RhsOut out;
  out.c_tot = p / (kRu * T);
  out.rho = out.c_tot / inv_wbar;
  // -- small-species stabilisation (Eqs 6-7, R7): C** = gamma(y) rho y / W
  for (int i = gl; i < S; i += G) {
    double y = cY[i];
    double yp = (y > 0.0) ? y : 0.0;
    double c = (out.rho * yp) * tv.invW[i];
    if (sc.alpha > 0.0) c = (yp / (sc.alpha + yp)) * c;
    cConc[i] = c;
  }
  group_sync<G>();

  // -- a2: rate constants and progress rates (Eqs 28-30; Eq 14).  Internal order:
  //    k < Rrev reversible, k >= Rrev irreversible, so the branch below is uniform except at one boundary.
  const double ln_c0 = clog(kPatm / (kRu * T));
  for (int k = gl; k < R; k += G) {
    const double ln_kf = fma_rn(-tv.Ta[k], invT, fma_rn(tv.b[k], lnT, tv.lnA[k]));
    double fwd = cexp(ln_kf);
    const unsigned long long pt = tv.part[k];
    const int r0 = (int)(pt & 0xff), n0 = (int)((pt >> 8) & 0xff), r1 = (int)((pt >> 16) & 0xff), n1 = (int)((pt >> 24) & 0xff);
    const int p0 = (int)((pt >> 32) & 0xff), m0 = (int)((pt >> 40) & 0xff), p1 = (int)((pt >> 48) & 0xff), m1 = (int)((pt >> 56) & 0xff);
    double qk;
    if (tb.has_real) {
      // real coefficients and exponents (Eqs 26-29): same order of operations as the integer case below
      const double *co = tv.rcoef + 4 * k, *od = tv.rord + 4 * k;
      fwd = times_power(fwd, cConc[r0], od[0]);
      if (n1) fwd = times_power(fwd, cConc[r1], od[1]);
      qk = fwd;
      if (k < Rrev) {
        double dg = 0.0 - co[0] * cG[r0];
        if (n1) dg = dg - co[1] * cG[r1];
        dg = dg + co[2] * cG[p0];
        if (m1) dg = dg + co[3] * cG[p1];
        const double ln_kc = fma_rn(tv.dnu[k], ln_c0, -dg);
        double rev = cexp(ln_kf - ln_kc);
        rev = times_power(rev, cConc[p0], od[2]);
        if (m1) rev = times_power(rev, cConc[p1], od[3]);
        qk = (fwd - rev) * (use_rof ? cRof[k] : 1.0);
      }
    } else {
      {
        const double c0 = cConc[r0];
        for (int n = 0; n < n0; ++n) fwd = fwd * c0;
        if (n1) {
          const double c1 = cConc[r1];
          for (int n = 0; n < n1; ++n) fwd = fwd * c1;
        }
      }
      qk = fwd;
      if (k < Rrev) {
        double dg = 0.0 - (double)n0 * cG[r0];
        if (n1) dg = dg - (double)n1 * cG[r1];
        dg = dg + (double)m0 * cG[p0];
        if (m1) dg = dg + (double)m1 * cG[p1];
        const double ln_kc = fma_rn(tv.dnu[k], ln_c0, -dg);
        double rev = cexp(ln_kf - ln_kc);
        const double d0 = cConc[p0];
        for (int n = 0; n < m0; ++n) rev = rev * d0;
        if (m1) {
          const double d1 = cConc[p1];
          for (int n = 0; n < m1; ++n) rev = rev * d1;
        }
        qk = (fwd - rev) * (use_rof ? cRof[k] : 1.0);
      }
    }
    cQ[k] = qk;
  }
  group_sync<G>();

  // -- source terms and the step limiter (Eqs 1-3): omega_i gathered in the caller's reaction
  //    order, r_i = W_i omega_i / rho, t* = min_i min(Y_step^max, y_i*) / r_i*.
  const double inv_rho = 1.0 / out.rho;
  double t_star = bits_to_double(0x7ff0000000000000ull);
  for (int i = gl; i < S; i += G) {
    double om = 0.0;
    const int e1 = tv.gptr[i + 1];
    for (int e = tv.gptr[i]; e < e1; ++e) {
      const unsigned ent = tv.gent[e];
      const double coef = tb.has_real ? tv.gcoef[e] : (double)(int)(signed char)(ent >> 16);
      om = om + coef * cQ[ent & 0xffffu];
    }
    const double r = (tv.W[i] * om) * inv_rho;
    const double y = cY[i];
    const double r_star = (-r > 1.0e-30) ? -r : 1.0e-30;
    const double y_star = (y < 1.0e-20) ? 1.0 : 0.9 * y;
    const double lim = ((sc.y_step_max < y_star) ? sc.y_step_max : y_star) / r_star;
    if (lim < t_star) t_star = lim;
    cConc[i] = r;   // concentrations are dead: reuse for dY_i/dt
    cG[i] = om;     // g/RT is dead: reuse for omega_i
  }
  out.t_star = group_min<G>(t_star);
  group_sync<G>();

  // -- temperature equation (R15), enthalpy sum sequential in species order.
  double sum_h = 0.0;
  for (int i = 0; i < S; ++i) sum_h = fma_rn(cH[i], cG[i], sum_h);
  out.dTdt = (sc.energy_mode == 0) ? -((sum_h * kRu) * T) / (out.rho * (kRu * sum_cp)) : 0.0;
  return out;
}

// ---------------------------------------------------------------------------------------------------------
// a5: DFT ringing detection for one reversible reaction (Eqs 8-13).  x[0..12] is the window in
// physical slot order.  Direct sums with the contract's twiddle literals; the largest high-bin magnitude is
// sqrt(max |.|^2), which equals max sqrt(|.|^2) bit for bit because IEEE sqrt is monotone.
// ---------------------------------------------------------------------------------------------------------
template <int M>
__device__ __forceinline__ double dft_bin_sq(const double (&x)[kWindow]) {
  double re = 0.0, im = 0.0;
#pragma unroll
  for (int k = 0; k < kWindow; ++k) {
    re = fma_rn(x[k], cos13((M * k) % kWindow), re);
    im = fma_rn(x[k], -sin13((M * k) % kWindow), im);
  }
  return fma_rn(re, re, im * im);
}

__device__ __forceinline__ bool dft_is_ringing(const double (&x)[kWindow], const SolverConsts &sc) {
  double d0 = 0.0;
#pragma unroll
  for (int k = 0; k < kWindow; ++k) d0 = d0 + x[k];
  d0 = fabs(d0);
  double m2 = 0.0, v;
  const int nhf = sc.nhf;
  if (nhf <= 1) { v = dft_bin_sq<1>(x); m2 = (v > m2) ? v : m2; }
  if (nhf <= 2) { v = dft_bin_sq<2>(x); m2 = (v > m2) ? v : m2; }
  if (nhf <= 3) { v = dft_bin_sq<3>(x); m2 = (v > m2) ? v : m2; }
  if (nhf <= 4) { v = dft_bin_sq<4>(x); m2 = (v > m2) ? v : m2; }
  if (nhf <= 5) { v = dft_bin_sq<5>(x); m2 = (v > m2) ? v : m2; }
  { v = dft_bin_sq<6>(x); m2 = (v > m2) ? v : m2; }
  const double d_hi = sqrt(m2);
  const double f_ring = d0 / ((d_hi > 1.0e-300) ? d_hi : 1.0e-300);
  return (d_hi > 1.0e-300) && (f_ring < sc.tol_ring) && (d0 < sc.tol_freq);   // no high-frequency content: not ringing
}

// ---------------------------------------------------------------------------------------------------------
// The integrator.  One launch = one pass over the active-cell list.
// ---------------------------------------------------------------------------------------------------------
template <int G>
__global__ void __launch_bounds__(512) stev_integrate_kernel(const __grid_constant__ IntegrateArgs a) {
  extern __shared__ __align__(128) unsigned char smem[];
  __shared__ unsigned long long mbar;
  stage_tables(smem, a.table, a.tb.bytes, &mbar);
  const DevTables &tb = a.tb;
  const CellLayout &cl = a.cl;
  const SolverConsts &sc = a.sc;
  const TableView tv(smem, tb);
  const int S = tb.S, Rrev = tb.Rrev;

  const int lane = threadIdx.x & 31;
  const int gl = lane % G;                    // lane within the group
  const int grp = lane / G;                   // group within the warp
  double *cell = (double *)(smem + tb.bytes) + (size_t)(threadIdx.x / G) * cl.stride;
  double *cY = cell + cl.oY, *cConc = cell + cl.oConc, *cQ = cell + cl.oQ, *cRof = cell + cl.oRof, *cRing = cell + cl.oRing;
  const int rp = cl.rrev_pad;

  const double dt_max = a.t_f * sc.delta_max;   // Eq 4
  const double t_tol = 1.0e-12 * a.t_f;         // R5

  // per-cell scalars, identical in all lanes of the group
  double T = 1000.0, p = kPatm, t = 0.0;
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
          T = a.T[cell_idx];
          p = a.p[cell_idx];
          for (int i = gl; i < S; i += G) cY[i] = a.Y[(long long)i * a.ld + cell_idx];
          steps_in_pass = 0;
          if (a.restore) {
            const double *rec = a.spill + (long long)cell_idx * a.spill_stride;
            t = rec[0];
            steps = (int)rec[1];
            slot = (int)rec[2];
            for (int k = gl; k < Rrev; k += G) cRof[k] = rec[3 + k];
            for (int s = 0; s < kWindow; ++s)
              for (int k = gl; k < Rrev; k += G) cRing[s * rp + k] = rec[3 + Rrev + s * Rrev + k];
          } else {
            t = 0.0;
            steps = 0;
            slot = 0;
            for (int k = gl; k < Rrev; k += G) cRof[k] = 1.0;                       // Eq 11
            for (int s = 0; s < kWindow; ++s)
              for (int k = gl; k < Rrev; k += G) cRing[s * rp + k] = 0.0;           // R10
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
    const RhsOut rhs = rhs_eval<G>(tb, tv, cl, sc, cell, gl, T, p, true);

    // ---- a3: step size (Eq 5) and landing on t_f (R5)
    double h = (rhs.t_star < dt_max) ? rhs.t_star : dt_max;
    bool last = false;
    const double rem = a.t_f - t;
    if (rem - h < t_tol) {
      h = rem;
      last = true;
    }

    // ---- a4: forward Euler (Eq 18)
    int bad = 0;
    for (int i = gl; i < S; i += G) {
      const double y = fma_rn(h, cConc[i], cY[i]);
      cY[i] = y;
      bad |= !(y - y == 0.0);
    }
    T = fma_rn(h, rhs.dTdt, T);
    t = last ? a.t_f : t + h;
    steps += 1;
    steps_in_pass += 1;
    bad |= !(T - T == 0.0);

    // ---- a5: DFT stabilisation (Eqs 8-14): store the applied change in progress (R8, R9), test, update rOF
    if (sc.dft_enable) {
      const double inv_ctot = 1.0 / rhs.c_tot;
      for (int k = gl; k < Rrev; k += G) {
        cRing[slot * rp + k] = (cQ[k] * h) * inv_ctot;
        double x[kWindow];
#pragma unroll
        for (int s = 0; s < kWindow; ++s) x[s] = cRing[s * rp + k];
        const bool ringing = dft_is_ringing(x, sc);
        double rof = cRof[k] * (ringing ? sc.inv_r_fac : sc.r_fac);
        if (rof > 1.0) rof = 1.0;
        if (rof < sc.rof_min) rof = sc.rof_min;
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
      for (int i = gl; i < S; i += G) a.Y[(long long)i * a.ld + cell_idx] = cY[i];
      if (gl == 0) {
        a.T[cell_idx] = T;
        a.steps[cell_idx] = steps;
        if (st >= 0 && a.status) a.status[cell_idx] = (unsigned char)st;
        if (st > 0) atomicMax(a.worst_status, st);
        if (a.flags) a.flags[pos] = pause ? 1 : 0;
      }
      if (pause) {
        double *rec = a.spill + (long long)cell_idx * a.spill_stride;
        if (gl == 0) {
          rec[0] = t;
          rec[1] = (double)steps;
          rec[2] = (double)slot;
        }
        for (int k = gl; k < Rrev; k += G) rec[3 + k] = cRof[k];
        for (int s = 0; s < kWindow; ++s)
          for (int k = gl; k < Rrev; k += G) rec[3 + Rrev + s * Rrev + k] = cRing[s * rp + k];
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
template <int G>
__global__ void __launch_bounds__(512) stev_rates_kernel(const __grid_constant__ RatesArgs a) {
  extern __shared__ __align__(128) unsigned char smem[];
  __shared__ unsigned long long mbar;
  stage_tables(smem, a.table, a.tb.bytes, &mbar);
  const DevTables &tb = a.tb;
  const CellLayout &cl = a.cl;
  const TableView tv(smem, tb);
  const int S = tb.S, R = tb.R, Rrev = tb.Rrev;
  const int gl = (threadIdx.x & 31) % G;
  double *cell = (double *)(smem + tb.bytes) + (size_t)(threadIdx.x / G) * cl.stride;
  const long long cells_per_block = blockDim.x / G;
  for (long long base = (long long)blockIdx.x * cells_per_block; base < a.n; base += (long long)gridDim.x * cells_per_block) {
    const long long c = base + threadIdx.x / G;
    const bool valid = c < a.n;
    const long long cc = valid ? c : a.n - 1;
    const double T = a.T[cc], p = a.p[cc];
    for (int i = gl; i < S; i += G) cell[cl.oY + i] = a.Y[(long long)i * a.ld + cc];
    for (int k = gl; k < Rrev; k += G) cell[cl.oRof + k] = a.rOF ? a.rOF[(long long)tv.orig[k] * a.ld + cc] : 1.0;
    group_sync<G>();
    const RhsOut rhs = rhs_eval<G>(tb, tv, cl, a.sc, cell, gl, T, p, true);
    if (valid) {
      for (int i = gl; i < S; i += G) a.dYdt[(long long)i * a.ld + c] = cell[cl.oConc + i];
      for (int k = gl; k < R; k += G) a.q[(long long)tv.orig[k] * a.ld + c] = cell[cl.oQ + k];
      if (gl == 0) a.dTdt[c] = rhs.dTdt;
    }
    group_sync<G>();
  }
}

}  // namespace stev
