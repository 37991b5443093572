// stev_pk_kernel.cuh -- the warp-pair STEV integrator for large mechanisms (rows a1-a7 of DESIGN.md section 1).
//
// One block per SM holds up to eight cells.  Each cell is served by a PAIR of warps that split every phase of a step
// between them (no idle role), meeting at a 64-thread named barrier between phases:
//   A  warp 0: scalars, ln T, ln(p_atm/R_u T), 1/Wbar, stabilised concentrations
//      warp 1: NASA-7 g/RT and the cp / h estimator (MLP on fp32 CUDA cores, or the NASA-7 polynomials)
//   B  both:   Arrhenius + equilibrium rates of their own 32-blocks of reactions, q_eff = q rOF, stored multiples
//   C  both:   source terms of their own species (one species per lane), step limiter, warp minimum
//   D  both:   step size, Euler update of their own species, DFT ringing filter of their own 32-blocks of
//              reversible reactions; warp 0 also evaluates the two sequential sums of the temperature equation
// The 13-deep history of every reversible reaction lives in TENSOR MEMORY (one lane-private row of TMEM columns per
// reaction, tcgen05.st / tcgen05.ld); each warp keeps the windows of its own blocks in its own TMEM lane quarter.
// Shared memory holds the mechanism tables (one TMA bulk copy per block) and ~17 KB of per-cell scratch; the hot loop
// has no HBM traffic.
// Arithmetic follows the contract of DESIGN.md section 5 exactly; every bit-equivalent deviation in evaluation order
// is explained where it occurs.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

#include "stev_device.cuh"
#include "stev_fast.cuh"
#include "stev_math.cuh"
#include "stev_pk.cuh"

namespace stev {

// 8-byte load at a 32-bit shared-memory address (warp-uniform base + per-lane table offset: one LDS with a
// register + uniform-register address, no separate add).  Volatile, no memory clobber: it keeps its order with the cell
// barriers (volatile asm / __syncwarp), which is all that is needed -- every value read this way was written in an
// earlier phase -- and leaves the compiler free to schedule the surrounding table loads and arithmetic.
__device__ __forceinline__ double lds_f64s(uint32_t base_s, unsigned off) {
  double v;
  asm volatile("ld.shared.f64 %0, [%1];" : "=d"(v) : "r"(base_s + off));
  return v;
}
// SA selects it; otherwise the plain C++ load, which the compiler may interleave freely (the large-mechanism kernels
// run four reactions per lane side by side and lose more to the fixed order than they gain from the saved adds)
template <bool SA>
__device__ __forceinline__ double lds_sel(const unsigned char *cell, uint32_t cell_s, unsigned off) {
  return SA ? lds_f64s(cell_s, off) : lds_f64(cell, off);
}

// ---------------------------------------------------------------------------------------------------------
// a1: NASA-7 (Eqs 15-16, R17) by one warp: g/RT (and 2 g/RT) always, cp/R and h/RT if CPH.
// Two species per lane side by side; lanes past the end recompute the last species and store nothing.
// ---------------------------------------------------------------------------------------------------------
template <bool CPH>
__device__ __forceinline__ void pk_nasa(const PkTables &tb, const unsigned char *tbl, double *cG, double2 *cYwCp, double2 *cHOm,
                                        double T, double invT, double lnT, int lane) {
  const int S = tb.S;
  const double *tmid = (const double *)(tbl + tb.o_tmid), *nasa = (const double *)(tbl + tb.o_nasa);
  for (int ia = lane; ia < S; ia += 64) {
    const int ib_ = ia + 32;
    const int ib = (ib_ < S) ? ib_ : S - 1;
    const double *ca = nasa + ((T < tmid[ia]) ? 0 : kNasaRows * S) + ia;
    const double *cb = nasa + ((T < tmid[ib]) ? 0 : kNasaRows * S) + ib;
    const double a1a = ca[0], a2a = ca[S], a1b = cb[0], a2b = cb[S];
    const double hpa = fma_rn(fma_rn(fma_rn(fma_rn(ca[8 * S], T, ca[7 * S]), T, ca[6 * S]), T, ca[5 * S]), T, a1a);
    const double hpb = fma_rn(fma_rn(fma_rn(fma_rn(cb[8 * S], T, cb[7 * S]), T, cb[6 * S]), T, cb[5 * S]), T, a1b);
    const double hRTa = fma_rn(ca[9 * S], invT, hpa), hRTb = fma_rn(cb[9 * S], invT, hpb);
    const double spa = fma_rn(fma_rn(fma_rn(ca[12 * S], T, ca[11 * S]), T, ca[10 * S]), T, a2a);
    const double spb = fma_rn(fma_rn(fma_rn(cb[12 * S], T, cb[11 * S]), T, cb[10 * S]), T, a2b);
    const double sRa = fma_rn(a1a, lnT, fma_rn(spa, T, ca[13 * S])), sRb = fma_rn(a1b, lnT, fma_rn(spb, T, cb[13 * S]));
    const double ga = hRTa - sRa, gb = hRTb - sRb;
    cG[1 + ia] = ga;
    cG[1 + S + ia] = ga + ga;
    if (ib_ < S) {
      cG[1 + ib] = gb;
      cG[1 + S + ib] = gb + gb;
    }
    if (CPH) {
      cYwCp[ia].y = fma_rn(fma_rn(fma_rn(fma_rn(ca[4 * S], T, ca[3 * S]), T, ca[2 * S]), T, a2a), T, a1a);
      cHOm[ia].x = hRTa;
      if (ib_ < S) {
        cYwCp[ib].y = fma_rn(fma_rn(fma_rn(fma_rn(cb[4 * S], T, cb[3 * S]), T, cb[2 * S]), T, a2b), T, a1b);
        cHOm[ib].x = hRTb;
      }
    }
  }
}

// The same with one species per lane (one warp per cell: at most 32 species, so the second slot would be idle).
template <bool CPH>
__device__ __forceinline__ void pk_nasa1(const PkTables &tb, const unsigned char *tbl, double *cG, double2 *cYwCp, double2 *cHOm,
                                         double T, double invT, double lnT, int lane) {
  const int S = tb.S;
  const double *tmid = (const double *)(tbl + tb.o_tmid), *nasa = (const double *)(tbl + tb.o_nasa);
  for (int ia = lane; ia < S; ia += 32) {
    const double *ca = nasa + ((T < tmid[ia]) ? 0 : kNasaRows * S) + ia;
    const double a1a = ca[0], a2a = ca[S];
    const double hpa = fma_rn(fma_rn(fma_rn(fma_rn(ca[8 * S], T, ca[7 * S]), T, ca[6 * S]), T, ca[5 * S]), T, a1a);
    const double hRTa = fma_rn(ca[9 * S], invT, hpa);
    const double spa = fma_rn(fma_rn(fma_rn(ca[12 * S], T, ca[11 * S]), T, ca[10 * S]), T, a2a);
    const double sRa = fma_rn(a1a, lnT, fma_rn(spa, T, ca[13 * S]));
    const double ga = hRTa - sRa;
    cG[1 + ia] = ga;
    cG[1 + S + ia] = ga + ga;
    if (CPH) {
      cYwCp[ia].y = fma_rn(fma_rn(fma_rn(fma_rn(ca[4 * S], T, ca[3 * S]), T, ca[2 * S]), T, a2a), T, a1a);
      cHOm[ia].x = hRTa;
    }
  }
}

// ---------------------------------------------------------------------------------------------------------
// a7 in the integrator (fp32 CUDA cores, R18): cp_i/R and h_i/(R T_ref) from the shallow MLP, by one warp.
// ---------------------------------------------------------------------------------------------------------
template <int MU>
__device__ __forceinline__ void pk_mlp(const PkTables &tb, const unsigned char *tbl, const double2 *cYp, double2 *cYwCp,
                                       double2 *cHOm, float *cHid, double T, double p, double invT, int lane, int o_lo, int o_hi) {
  const int S = tb.S;
  const float *eshift = (const float *)(tbl + tb.o_eshift), *escale = (const float *)(tbl + tb.o_escale);
  const float *W1T = (const float *)(tbl + tb.o_W1T), *b1 = (const float *)(tbl + tb.o_b1);
  const float *W2p = (const float *)(tbl + tb.o_W2p), *b2 = (const float *)(tbl + tb.o_b2);
  const int H = tb.H, Hpad = tb.Hpad, n_in = tb.n_in;
  // normalised inputs once (lane k: input k), then two hidden units per lane per pass; per unit the operations and
  // their order are the contract's (fmaf over the inputs in index order)
  float *cXn = cHid + H;
  for (int k = lane; k < n_in; k += 32) {
    const double raw = (k == 0) ? T : ((k == 1) ? p : cYp[k - 2].x);
    cXn[k] = ((float)raw - eshift[k]) * escale[k];
  }
  __syncwarp();
  auto activate = [&](float z) {
    const double zd = (double)z;
    if (tb.act == 0) return (float)(1.0 - 2.0 / (1.0 + ab_exp(2.0 * zd)));
    return (float)(1.0 / (1.0 + ab_exp(-zd)));
  };
  for (int jh0 = lane; jh0 < H; jh0 += 64) {
    const int jh1_ = jh0 + 32;
    const int jh1 = (jh1_ < H) ? jh1_ : jh0;
    float z0 = b1[jh0], z1 = b1[jh1];
    if (jh0 - lane + 32 < H) {   // warp-uniform: a second row of units exists
      const float *w = W1T + jh0;   // unit jh0 and, 32 floats on, unit jh0 + 32; one row of H floats per input
#pragma unroll 4
      for (int k = 0; k < n_in; ++k, w += H) {
        const float xk = cXn[k];
        z0 = __fmaf_rn(w[0], xk, z0);
        z1 = __fmaf_rn(w[32], xk, z1);
      }
    } else {
      const float *w = W1T + jh0;
#pragma unroll 4
      for (int k = 0; k < n_in; ++k, w += H) z0 = __fmaf_rn(w[0], cXn[k], z0);
    }
    cHid[jh0] = activate(z0);
    if (jh1_ < H) cHid[jh1] = activate(z1);
  }
  __syncwarp();
  const float4 *hid4 = (const float4 *)cHid;
  for (int o0 = o_lo; o0 < o_hi; o0 += 32 * MU) {
    float y[MU];
    const float4 *wrow[MU];
#pragma unroll
    for (int u = 0; u < MU; ++u) {
      int o = o0 + 32 * u + lane;
      o = (o < o_hi) ? o : o_hi - 1;
      y[u] = b2[o];
      wrow[u] = (const float4 *)(W2p + (size_t)o * Hpad);
    }
#pragma unroll 4
    for (int q4 = 0; q4 < H / 4; ++q4) {
      const float4 hv = hid4[q4];
#pragma unroll
      for (int u = 0; u < MU; ++u) {
        const float4 wv = wrow[u][q4];
        y[u] = __fmaf_rn(wv.x, hv.x, y[u]);
        y[u] = __fmaf_rn(wv.y, hv.y, y[u]);
        y[u] = __fmaf_rn(wv.z, hv.z, y[u]);
        y[u] = __fmaf_rn(wv.w, hv.w, y[u]);
      }
    }
#pragma unroll
    for (int u = 0; u < MU; ++u) {
      const int o = o0 + 32 * u + lane;
      if (o < o_hi) {
        if (o < S) cYwCp[o].y = (double)y[u];
        else cHOm[o - S].x = ((double)y[u] * (double)tb.h_ref_T) * invT;
      }
    }
  }
}

// ---------------------------------------------------------------------------------------------------------
// a5: the ringing filter (Eqs 8-13) of the 32-blocks [it_lo, it_hi) of reversible reactions, by one
// warp.  TMEM address of slot s of this lane's reaction in block `it`:  trow + it * 32 + 2 s.
// Two windows are processed side by side (independent dependency chains for the scheduler).
// ---------------------------------------------------------------------------------------------------------
template <int NHF, bool PAIRWIN>
__device__ __forceinline__ void pk_dft(const SolverConsts &sc, const double *cQ, double *cRof, int Rrev, int it_lo, int it_hi,
                                       uint32_t trow, int slot, double h, double inv_ctot, int lane) {
  auto update_rof = [&](int k, bool ringing) {
    double rof = cRof[k] * (ringing ? sc.inv_r_fac : sc.r_fac);   // Eqs 12-13
    if (rof > 1.0) rof = 1.0;
    if (rof < sc.rof_min) rof = sc.rof_min;
    cRof[k] = rof;
  };
  // Eq 8 with R8, R9: the applied change in progress / C_tot of every reversible reaction goes into its window
  for (int it = it_lo; it < it_hi; ++it) {
    const int k = it * 32 + lane;
    const double q = (k < Rrev) ? cQ[k] : 0.0;
    tmem_st2(trow + it * 32 + 2 * slot, (q * h) * inv_ctot);
  }
  tmem_wait_st();
  int it = it_lo;
  for (; PAIRWIN && it + 2 <= it_hi; it += 2) {
    uint32_t ra[26], rb[26];
    tmem_ld26(trow + it * 32, ra);
    tmem_ld26(trow + it * 32 + 32, rb);
    tmem_wait_ld();
    double xa[kWindow], xb[kWindow];
    unpack_window(ra, xa);
    unpack_window(rb, xb);
    double d0a, m2a, d0b, m2b;
    ab_window_stats<NHF>(xa, d0a, m2a);
    ab_window_stats<NHF>(xb, d0b, m2b);
    const int ka = it * 32 + lane, kb = ka + 32;
    bool sure_a, sure_b;
    bool ring_a = ab_ring_filter(d0a, m2a, sc, sure_a);
    bool ring_b = ab_ring_filter(d0b, m2b, sc, sure_b);
    if (__any_sync(0xffffffffu, (!sure_a && ka < Rrev) || (!sure_b && kb < Rrev))) {
      ring_a = ab_ring_exact(d0a, m2a, sc);
      ring_b = ab_ring_exact(d0b, m2b, sc);
    }
    if (ka < Rrev) update_rof(ka, ring_a);
    if (kb < Rrev) update_rof(kb, ring_b);
  }
  auto one_window = [&](int it) {
    uint32_t ra[26];
    tmem_ld26(trow + it * 32, ra);
    tmem_wait_ld();
    double xa[kWindow];
    unpack_window(ra, xa);
    double d0a, m2a;
    ab_window_stats<NHF>(xa, d0a, m2a);
    const int ka = it * 32 + lane;
    bool sure_a;
    bool ring_a = ab_ring_filter(d0a, m2a, sc, sure_a);
    if (__any_sync(0xffffffffu, !sure_a && ka < Rrev)) ring_a = ab_ring_exact(d0a, m2a, sc);
    if (ka < Rrev) update_rof(ka, ring_a);
  };
  if (PAIRWIN) {
    if (it < it_hi) one_window(it);
  } else {
#pragma unroll 1
    for (; it < it_hi; ++it) one_window(it);
  }
}

// ---------------------------------------------------------------------------------------------------------
// a2 for U reversible reactions per lane side by side (blocks b0, b0 + bs, ..): rate constants, equilibrium
// constants, effective progress rates and their stored multiples.  One pass = one trip through the latency chain
// table load -> g loads -> exponentials -> concentration loads -> stores, with 2 U independent exp chains in flight.
// Lanes past the end recompute the last reaction and store nothing.
// ---------------------------------------------------------------------------------------------------------
template <int U, bool SA>
__device__ __forceinline__ void pk_rev_batch(const unsigned char *cell, uint32_t cell_s, const double2 *rkA, const double2 *rkB, const uint4 *rfac,
                                             const uint4 *rdg, const double *cRof, double *cQ, int Rp, int Rrev, bool has2,
                                             double invT, double lnT, double ln_c0, int b0, int bs, int lane) {
  int k_[U], k[U];
  double lkf[U], lkr[U];
  uint4 f[U];
  bool oor = false;
#pragma unroll
  for (int u = 0; u < U; ++u) {
    k_[u] = (b0 + u * bs) * 32 + lane;
    k[u] = (k_[u] < Rrev) ? k_[u] : Rrev - 1;
  }
#pragma unroll
  for (int u = 0; u < U; ++u) {
    const double2 p0 = rkA[k[u]], p1 = rkB[k[u]];
    const uint4 d = rdg[k[u]];
    f[u] = rfac[k[u]];
    lkf[u] = fma_rn(-p1.x, invT, fma_rn(p0.y, lnT, p0.x));
    double dg = 0.0 - lds_sel<SA>(cell, cell_s, d.x);
    dg = dg - lds_sel<SA>(cell, cell_s, d.y);
    dg = dg + lds_sel<SA>(cell, cell_s, d.z);
    dg = dg + lds_sel<SA>(cell, cell_s, d.w);
    lkr[u] = lkf[u] - fma_rn(p1.y, ln_c0, -dg);
    oor = oor || ab_exp_out_of_range(lkf[u]) || ab_exp_out_of_range(lkr[u]);
  }
  double fwd[U], rev[U];
  if (__any_sync(0xffffffffu, oor)) {
#pragma unroll
    for (int u = 0; u < U; ++u) {
      fwd[u] = cexp(lkf[u]);
      rev[u] = cexp(lkr[u]);
    }
  } else {
#pragma unroll
    for (int u = 0; u < U; ++u) {
      fwd[u] = ab_exp_core(lkf[u]);
      rev[u] = ab_exp_core(lkr[u]);
    }
  }
#pragma unroll
  for (int u = 0; u < U; ++u) {
    fwd[u] = fwd[u] * lds_sel<SA>(cell, cell_s, f[u].x);
    rev[u] = rev[u] * lds_sel<SA>(cell, cell_s, f[u].z);
  }
#pragma unroll
  for (int u = 0; u < U; ++u) {
    fwd[u] = fwd[u] * lds_sel<SA>(cell, cell_s, f[u].y);
    rev[u] = rev[u] * lds_sel<SA>(cell, cell_s, f[u].w);
  }
#pragma unroll
  for (int u = 0; u < U; ++u) {
    const double q = (fwd[u] - rev[u]) * cRof[k[u]];   // Eq 14
    if (k_[u] < Rrev) {
      cQ[k[u]] = q;
      cQ[Rp + k[u]] = -q;
      if (has2) {
        const double q2 = q + q;
        cQ[2 * Rp + k[u]] = q2;
        cQ[3 * Rp + k[u]] = -q2;
      }
    }
  }
}

// a2 for IU irreversible reactions per lane side by side (reactions k0 + lane, k0 + ks + lane, ..): rate constants, progress
// rates and their stored multiples.  Lanes past the end recompute the last reaction and store nothing.
template <int IU, bool SA>
__device__ __forceinline__ void pk_irr_batch(const unsigned char *cell, uint32_t cell_s, const double2 *rkA, const double2 *rkB, const uint4 *rfac,
                                             double *cQ, int Rp, int R, bool has2, double invT, double lnT, int k0, int ks, int lane) {
  double lk[IU], fw[IU];
  uint4 f[IU];
  int kk[IU];
  bool oor = false;
#pragma unroll
  for (int u = 0; u < IU; ++u) {
    kk[u] = k0 + ks * u + lane;
    const int k = (kk[u] < R) ? kk[u] : R - 1;
    const double2 p0 = rkA[k];
    const double ta = rkB[k].x;
    f[u] = rfac[k];
    lk[u] = fma_rn(-ta, invT, fma_rn(p0.y, lnT, p0.x));
    oor = oor || ab_exp_out_of_range(lk[u]);
  }
  if (__any_sync(0xffffffffu, oor)) {
#pragma unroll
    for (int u = 0; u < IU; ++u) fw[u] = cexp(lk[u]);
  } else {
#pragma unroll
    for (int u = 0; u < IU; ++u) fw[u] = ab_exp_core(lk[u]);
  }
#pragma unroll
  for (int u = 0; u < IU; ++u) fw[u] = fw[u] * lds_sel<SA>(cell, cell_s, f[u].x);
#pragma unroll
  for (int u = 0; u < IU; ++u) fw[u] = fw[u] * lds_sel<SA>(cell, cell_s, f[u].y);
#pragma unroll
  for (int u = 0; u < IU; ++u) {
    if (kk[u] < R) {
      const int k = kk[u];
      cQ[k] = fw[u];
      cQ[Rp + k] = -fw[u];
      if (has2) {
        const double f2 = fw[u] + fw[u];
        cQ[2 * Rp + k] = f2;
        cQ[3 * Rp + k] = -f2;
      }
    }
  }
}

// unsigned-bit-pattern minimum of positive doubles (NaN patterns sort above +inf and are thereby ignored, like the
// contract's plain comparison `lim < t_star` ignores them)
__device__ __forceinline__ double pk_min_bits(double a, double b) {
  return (double_to_bits(b) < double_to_bits(a)) ? b : a;
}

// ---------------------------------------------------------------------------------------------------------
// One warp of the NW (1 or 2) warps that serve a cell.  `half` (0 .. NW-1) is warp-uniform.  With NW = 1 the pair
// barriers degenerate to __syncwarp and the warp walks both halves of every phase (mid-size mechanisms: 16 cells per SM).
// ---------------------------------------------------------------------------------------------------------
#ifdef PK_TIMING
__shared__ long long pk_tacc[32][8];
#define PKT(i)                                                        \
  if (lane == 0) {                                                    \
    const long long now_ = clock64();                                 \
    pk_tacc[threadIdx.x >> 5][i] += now_ - tlast_;                    \
    tlast_ = now_;                                                    \
  }
#else
#define PKT(i)
#endif

template <bool EST, int NW, bool DENSE>
__device__ __forceinline__ void pk_worker(const PkArgs &a, const unsigned char *tbl, unsigned char *cell, int j, int half,
                                          int tmem_quarter, uint32_t tmem_base, int lane) {
  const PkTables &tb = a.tb;
  const SolverConsts &sc = a.sc;
  const int S = tb.S, R = tb.R, Rrev = tb.Rrev, Rp = tb.Rp, n_it = tb.n_it;
  double2 *cYp = (double2 *)(cell + a.cl.oYp);
  double2 *cYwCp = (double2 *)(cell + a.cl.oYwCp);
  double2 *cHOm = (double2 *)(cell + a.cl.oHOm);
  double *cConc = (double *)(cell + a.cl.oConc);
  double *cG = (double *)(cell + a.cl.oG);
  double *cQ = (double *)(cell + a.cl.oQ);
  double *cRof = (double *)(cell + a.cl.oRof);
  float *cHid = (float *)(cell + a.cl.oHid);
  volatile PkScal *scal = (volatile PkScal *)(cell + a.cl.oSc);
  const uint32_t cell_s = (uint32_t)__cvta_generic_to_shared(cell);   // table-driven loads address shared memory directly
  constexpr bool kSA = (NW == 1), kGA = (NW == 1);

  const double *W = (const double *)(tbl + tb.o_W), *invW = (const double *)(tbl + tb.o_invW);
  const double2 *rkA = (const double2 *)(tbl + tb.o_rkA), *rkB = (const double2 *)(tbl + tb.o_rkB);
  const uint4 *rfac = (const uint4 *)(tbl + tb.o_rfac), *rdg = (const uint4 *)(tbl + tb.o_rdg);
  const unsigned char *gsp = tbl + tb.o_gsp;
  const bool has2 = tb.n_var > 2;

  const int bar = 1 + j;                        // named barrier of this cell's warps (0 is __syncthreads)
  auto cell_sync = [&]() {
    if (NW >= 2) asm volatile("bar.sync %0, %1;" ::"r"(bar), "n"(32 * NW) : "memory");
    else __syncwarp();
  };
  const double dt_max = a.t_f * sc.delta_max;   // Eq 4
  const double t_tol = 1.0e-12 * a.t_f;         // R5
  const int it_lo = (NW == 1 || half == 0) ? 0 : tb.it_split[half], it_hi = (NW == 1) ? n_it : tb.it_split[half + 1];   // DFT blocks of this warp (at most four)
  // TMEM: a warp reaches the lane quarter (warp id mod 4); it keeps the windows of its own blocks in 128 columns of
  // that quarter: columns [128 (j / 4), +128) for warp 0 of a cell (or the only warp), [256 + 128 (j / 4), +128) for warp 1.
  // (one warp per cell, dense: 32 cells per block, at most two blocks = 64 columns per cell)
  uint32_t tcol = DENSE ? (uint32_t)((j >> 2) * 64) : (uint32_t)((j >> 2) * 128 + half * 256);
  const uint32_t trow = tmem_base + ((uint32_t)((tmem_quarter & 3) * 32) << 16) + tcol - (uint32_t)(it_lo * 32);
  const int my_sp = (half < 2) ? half * 32 + lane : 0x7fff;   // species this lane loads, updates and writes back
  const int g_sp = gsp[half * 32 + lane];       // species whose source term this lane gathers (255 = none)
  const uint4 *ge = (const uint4 *)(tbl + tb.o_gent) + tb.g_row0[half] * 32 + lane;
  const int g_len4 = tb.g_len4[half];
  if (lane == 0) scal->t_star[half] = bits_to_double(0x7ff0000000000000ull);   // stays +inf for a warp without lists

  if (half == 0 && lane == 0) {
    cConc[0] = 1.0;
    cG[0] = 0.0;
  }
  // a5 for this warp's blocks: h_s and ictot_s are the step size and 1/C_tot of the step whose progress is stored
  constexpr bool kPairWin = (NW <= 2) && !DENSE;   // two windows side by side need ~125 registers
  auto run_dft = [&](int slot_s, double h_s, double ictot_s) __attribute__((always_inline)) {
    switch (sc.nhf) {
      case 1: pk_dft<1, kPairWin>(sc, cQ, cRof, Rrev, it_lo, it_hi, trow, slot_s, h_s, ictot_s, lane); break;
      case 2: pk_dft<2, kPairWin>(sc, cQ, cRof, Rrev, it_lo, it_hi, trow, slot_s, h_s, ictot_s, lane); break;
      case 3: pk_dft<3, kPairWin>(sc, cQ, cRof, Rrev, it_lo, it_hi, trow, slot_s, h_s, ictot_s, lane); break;
      case 4: pk_dft<4, kPairWin>(sc, cQ, cRof, Rrev, it_lo, it_hi, trow, slot_s, h_s, ictot_s, lane); break;
      case 5: pk_dft<5, kPairWin>(sc, cQ, cRof, Rrev, it_lo, it_hi, trow, slot_s, h_s, ictot_s, lane); break;
      default: pk_dft<6, kPairWin>(sc, cQ, cRof, Rrev, it_lo, it_hi, trow, slot_s, h_s, ictot_s, lane); break;
    }
  };
  // Pair: second named barrier of the cell (ids 9..15, and 0 -- free after the block-wide start-up -- for cell 7).
  // Warp 0 arrives when the new T and Y are in shared memory, warp 1 waits for that before the thermodynamics.
  const int xbar = (j < 7) ? 9 + j : 0;

  for (;;) {
    // ---- a6: variable load.  A pair whose cell retired pulls the next active cell from the global queue.
    if (half == 0 && lane == 0) scal->pos = atomicAdd(a.queue_head, 1);
    cell_sync();
    const int pos = scal->pos;
    if ((long long)pos >= a.n_active) return;
    const int cidx = a.list ? a.list[pos] : pos;
    double T = a.T[cidx];
    const double p = a.p[cidx];
    if (my_sp < S) cYp[my_sp] = make_double2(a.Y[(long long)my_sp * a.ld + cidx], invW[my_sp]);
    for (int it = it_lo; it < it_hi; ++it) {
#pragma unroll
      for (int s = 0; s < kWindow; ++s) tmem_st2(trow + it * 32 + 2 * s, 0.0);   // R10: zero-initialised window
      const int k = it * 32 + lane;
      if (k < Rrev) cRof[k] = 1.0;                                                // Eq 11
    }
    tmem_wait_st();
    double t = 0.0, h_prev = 0.0, ictot_prev = 0.0;
    int steps = 0, slot = 0;
    cell_sync();
#ifdef PK_TIMING
    long long tlast_ = clock64();
    if (lane == 0)
      for (int i_ = 0; i_ < 8; ++i_) pk_tacc[threadIdx.x >> 5][i_] = 0;
#endif

    for (;;) {
      // ================= phase A =================
      double lnT, ln_c0, invT, inv_ctot, rho;
      if (NW == 1 || half == 0) {
        // -- scalars.  ln T and ln(p_atm / (R_u T)) are evaluated side by side in the two half-warps.
        const double RuT = kRu * T;
        const double c_tot = p / RuT;
        invT = 1.0 / T;
        const double larg = (lane & 16) ? (kPatm / RuT) : T;
        const double lval = ab_log(larg);
        lnT = __shfl_sync(0xffffffffu, lval, 0);
        ln_c0 = __shfl_sync(0xffffffffu, lval, 16);
        inv_ctot = 1.0 / c_tot;
        if (NW == 1) {
          if (EST) pk_nasa1<false>(tb, tbl, cG, cYwCp, cHOm, T, invT, lnT, lane);
          else pk_nasa1<true>(tb, tbl, cG, cYwCp, cHOm, T, invT, lnT, lane);
        }
        // -- 1/Wbar = sum Y_i/W_i, sequential in species order (contract 5.4)
        double inv_wbar = 0.0;
#pragma unroll 8
        for (int i = 0; i < S; ++i) {
          const double2 v = cYp[i];
          inv_wbar = fma_rn(v.x, v.y, inv_wbar);
        }
        rho = c_tot / inv_wbar;
        if (lane == 0) {
          scal->lnT = lnT;
          scal->ln_c0 = ln_c0;
          scal->invT = invT;
          scal->inv_ctot = inv_ctot;
          scal->rho = rho;
        }
        // -- Y_i/W_i (for the cp sum) and the small-species stabilisation (Eqs 6-7, R7):
        //    C** = gamma(y) rho y / W
        if (NW == 1) {
          for (int ia = lane; ia < S; ia += 32) {
            const double2 va = cYp[ia];
            const double ypa = (va.x > 0.0) ? va.x : 0.0;
            double ca = (rho * ypa) * va.y;
            if (sc.alpha > 0.0) ca = (ypa / (sc.alpha + ypa)) * ca;
            cYwCp[ia].x = va.x * va.y;
            cConc[1 + ia] = ca;
          }
        } else
        for (int ia = lane; ia < S; ia += 64) {
          const int ib_ = ia + 32;
          const int ib = (ib_ < S) ? ib_ : S - 1;
          const double2 va = cYp[ia], vb = cYp[ib];
          const double ypa = (va.x > 0.0) ? va.x : 0.0, ypb = (vb.x > 0.0) ? vb.x : 0.0;
          double ca = (rho * ypa) * va.y, cb = (rho * ypb) * vb.y;
          if (sc.alpha > 0.0) {
            const double gam_a = ypa / (sc.alpha + ypa), gam_b = ypb / (sc.alpha + ypb);
            ca = gam_a * ca;
            cb = gam_b * cb;
          }
          cYwCp[ia].x = va.x * va.y;
          cConc[1 + ia] = ca;
          if (ib_ < S) {
            cYwCp[ib].x = vb.x * vb.y;
            cConc[1 + ib] = cb;
          }
        }
      }
      if (NW == 2 && half == 0 && steps > 0 && sc.dft_enable) {
        // warp 0 of the pair: its share of the ringing filter of the PREVIOUS step (it only feeds rOF, which phase B
        // reads), after the scalars of this step, so that no barrier separates the update from phase A
        run_dft(slot, h_prev, ictot_prev);
        slot = (slot + 1 == kWindow) ? 0 : slot + 1;
      }
      if (NW == 1) {
        if (EST) {
          // outputs per lane per pass sized to the output layer (config 4 has 40 outputs: two per lane, not four)
          if (tb.n_out <= 64) pk_mlp<2>(tb, tbl, cYp, cYwCp, cHOm, cHid, T, p, invT, lane, 0, tb.n_out);
          else pk_mlp<4>(tb, tbl, cYp, cYwCp, cHOm, cHid, T, p, invT, lane, 0, tb.n_out);
        }
      } else if (NW >= 2 && half == 1) {
        // warp 1 of the pair: all of the thermodynamics (its own ln T and 1/T: same operations, same bits)
        const double invT1 = 1.0 / T;
        if (EST) {
          pk_nasa<false>(tb, tbl, cG, cYwCp, cHOm, T, invT1, ab_log(T), lane);
          pk_mlp<4>(tb, tbl, cYp, cYwCp, cHOm, cHid, T, p, invT1, lane, 0, tb.n_out);
        } else {
          pk_nasa<true>(tb, tbl, cG, cYwCp, cHOm, T, invT1, ab_log(T), lane);
        }
      }
      PKT(0)
      cell_sync();
      PKT(1)
      if (NW >= 2 && half) {
        lnT = scal->lnT;
        ln_c0 = scal->ln_c0;
        invT = scal->invT;
        inv_ctot = scal->inv_ctot;
        rho = scal->rho;
      }

      // ================= phase B: a2, rate constants and effective progress rates (Eqs 28-30, Eq 14) =================
      // Reversible reactions occupy internal indices [0, Rrev) in 32-blocks; blocks b = half (mod 2) belong to this
      // warp and are evaluated four (small mechanisms: two) at a time, i.e. eight independent exp chains and one trip
      // through the load -> exp -> load -> store latency chain.  The stored multiples +q, -q, +2q, -2q (all exact) turn the sum
      // omega_i = sum_j nu_ij q_j into plain additions in the contract's order.
      if (!DENSE && n_it > 2 * NW) {
        for (int b0 = half; b0 < n_it; b0 += 4 * NW)
          pk_rev_batch<4, kSA>(cell, cell_s, rkA, rkB, rfac, rdg, cRof, cQ, Rp, Rrev, has2, invT, lnT, ln_c0, b0, NW, lane);
      } else {
        int b0 = half;
        for (; b0 + NW < n_it; b0 += 2 * NW)
          pk_rev_batch<2, kSA>(cell, cell_s, rkA, rkB, rfac, rdg, cRof, cQ, Rp, Rrev, has2, invT, lnT, ln_c0, b0, NW, lane);
        for (; b0 < n_it; b0 += NW)
          pk_rev_batch<1, kSA>(cell, cell_s, rkA, rkB, rfac, rdg, cRof, cQ, Rp, Rrev, has2, invT, lnT, ln_c0, b0, NW, lane);
      }
      // irreversible reactions [Rrev, R): 32-blocks c = half (mod NW), two at a time while two are left
      {
        int k0 = Rrev + half * 32;
        for (; k0 + 32 * NW < R; k0 += 64 * NW) pk_irr_batch<2, kSA>(cell, cell_s, rkA, rkB, rfac, cQ, Rp, R, has2, invT, lnT, k0, 32 * NW, lane);
        for (; k0 < R; k0 += 32 * NW) pk_irr_batch<1, kSA>(cell, cell_s, rkA, rkB, rfac, cQ, Rp, R, has2, invT, lnT, k0, 32 * NW, lane);
      }
      PKT(2)
      cell_sync();
      PKT(3)

      // ================= phase C: source terms and the limiter (Eqs 1-3) =================
      // One species per lane; the entry lists hold the byte offsets of the stored multiples in the caller's reaction
      // order and are padded with the 0.0 slot to the longest list of the warp, so the loop is warp-uniform.
      {
        const double inv_rho = 1.0 / rho;
        double om = 0.0;
        // Two rows of four entries per trip: the eight loads of a trip are independent and the offsets of the next
        // trip are fetched before the additions of this one (the table carries two spare rows).  Lists are sorted by
        // length over the lanes; padding entries read the 0.0 slot, and adding +0.0 changes nothing (om is never -0.0).
        uint4 o0 = ge[0], o1 = ge[32];
        for (int e4 = 0; e4 < g_len4; e4 += 2) {
          const double v0 = lds_sel<kGA>(cell, cell_s, o0.x), v1 = lds_sel<kGA>(cell, cell_s, o0.y), v2 = lds_sel<kGA>(cell, cell_s, o0.z), v3 = lds_sel<kGA>(cell, cell_s, o0.w);
          const double v4 = lds_sel<kGA>(cell, cell_s, o1.x), v5 = lds_sel<kGA>(cell, cell_s, o1.y), v6 = lds_sel<kGA>(cell, cell_s, o1.z), v7 = lds_sel<kGA>(cell, cell_s, o1.w);
          o0 = ge[(e4 + 2) * 32];
          o1 = ge[(e4 + 3) * 32];
          om = om + v0;
          om = om + v1;
          om = om + v2;
          om = om + v3;
          om = om + v4;
          om = om + v5;
          om = om + v6;
          om = om + v7;
        }
        // lanes without a species (255) work on species 0 and discard the result
        const int i0 = (g_sp < S) ? g_sp : 0;
        const double r0 = (W[i0] * om) * inv_rho;
        const double y0 = cYp[i0].x;
        const double rs0 = (-r0 > 1.0e-30) ? -r0 : 1.0e-30;
        const double ys0 = (y0 < 1.0e-20) ? 1.0 : 0.9 * y0;
        const double lim0 = ((sc.y_step_max < ys0) ? sc.y_step_max : ys0) / rs0;
        const double inf = bits_to_double(0x7ff0000000000000ull);
        double t_star = (g_sp < S && lim0 < inf) ? lim0 : inf;
        if (g_sp < S) {
          cConc[1 + g_sp] = r0;     // concentrations are dead: reuse for dY_i/dt
          cHOm[g_sp].y = om;
        }
        // min over lanes: every lim is a positive double or +inf, for which the ordering of the bit patterns as
        // unsigned integers is the ordering of the values
        const unsigned long long u = double_to_bits(t_star);
        const unsigned hi = (unsigned)(u >> 32), lo = (unsigned)u;
        const unsigned mhi = __reduce_min_sync(0xffffffffu, hi);
        const unsigned mlo = __reduce_min_sync(0xffffffffu, (hi == mhi) ? lo : 0xffffffffu);
        if (lane == 0) scal->t_star[half] = bits_to_double(((unsigned long long)mhi << 32) | mlo);
      }
      PKT(4)
      cell_sync();
      PKT(5)

      // ================= phase D =================
      // -- a3: step size (Eq 5) and landing on t_f (R5)
      double t_star = scal->t_star[0];
      if (NW >= 2) t_star = pk_min_bits(t_star, scal->t_star[1]);
      double h = (t_star < dt_max) ? t_star : dt_max;
      bool last = false;
      const double rem = a.t_f - t;
      if (rem - h < t_tol) {
        h = rem;
        last = true;
      }
      // -- a4: forward Euler (Eq 18), one species per lane (pair: warp 0 updates all species, two per lane,
      //    so that it depends on nothing of warp 1 between here and the end of phase A)
      int bad = 0;
      if (NW == 2) {
        if (half == 0) {
#pragma unroll
          for (int u = 0; u < 2; ++u) {
            const int i = lane + 32 * u;
            if (i < S) {
              const double y = fma_rn(h, cConc[1 + i], cYp[i].x);
              cYp[i].x = y;
              bad |= !(y - y == 0.0);
            }
          }
        }
      } else if (my_sp < S) {
        const double y = fma_rn(h, cConc[1 + my_sp], cYp[my_sp].x);
        cYp[my_sp].x = y;
        bad |= !(y - y == 0.0);
      }
      if (half == 0) {
        // temperature equation (R15): sum (Y_i/W_i) cp_i/R and sum (h_i/RT) omega_i, each sequential in species order
        // (contract 5.4); the two chains run in the even and the odd lanes of the same instruction stream
        const double2 *arr = (lane & 1) ? cHOm : cYwCp;
        double acc = 0.0;
#pragma unroll 8
        for (int i = 0; i < S; ++i) {
          const double2 v = arr[i];
          acc = fma_rn(v.x, v.y, acc);
        }
        const double sum_cp = __shfl_sync(0xffffffffu, acc, 0), sum_h = __shfl_sync(0xffffffffu, acc, 1);
        const double dTdt = (sc.energy_mode == 0) ? -((sum_h * kRu) * T) / (rho * (kRu * sum_cp)) : 0.0;
        T = fma_rn(h, dTdt, T);
        bad |= !(T - T == 0.0);
        if (lane == 0) scal->T_new = T;
      }
      bad = __any_sync(0xffffffffu, bad);
      if (lane == 0 && half < 2) scal->bad[half] = bad;
      PKT(6)
      if (NW == 2) {
        // -- a5 on warp 1 now (skipped on the landing step: the cell retires); warp 0 runs its share after the scalars of
        //    the next step.  Warp 0 announces the new T and Y (bar.arrive), warp 1 waits for them (bar.sync).
        if (half == 0) {
          __threadfence_block();
          asm volatile("bar.arrive %0, 64;" ::"r"(xbar) : "memory");
        } else {
          if (!last && sc.dft_enable) {
            run_dft(slot, h, inv_ctot);
            slot = (slot + 1 == kWindow) ? 0 : slot + 1;
          }
          asm volatile("bar.sync %0, 64;" ::"r"(xbar) : "memory");
          T = scal->T_new;
        }
      } else {
        // -- a5: DFT ringing filter of this warp's blocks (skipped on the landing step: the cell retires)
        if (!last && sc.dft_enable) {
          run_dft(slot, h, inv_ctot);
          slot = (slot + 1 == kWindow) ? 0 : slot + 1;
        }
        cell_sync();
        if (NW >= 2 && half) T = scal->T_new;
      }
      PKT(7)
      t = last ? a.t_f : t + h;
      steps += 1;
      h_prev = h;
      ictot_prev = inv_ctot;

      // -- a6: retirement (R20)
      int st = -1;
      if (scal->bad[0]) st = 2;   // checked first: a non-finite landing step is not "finished"
      else if (last) st = 0;
      else if (steps >= sc.max_steps) st = 1;
      if (st >= 0) {
#ifdef PK_TIMING
        if (blockIdx.x == 0 && j == 0 && lane == 0)
          printf("PKT half %d steps %d per step: A %lld w %lld | B %lld w %lld | C %lld w %lld | D %lld w %lld\n", half, steps,
                 pk_tacc[threadIdx.x >> 5][0] / steps, pk_tacc[threadIdx.x >> 5][1] / steps, pk_tacc[threadIdx.x >> 5][2] / steps,
                 pk_tacc[threadIdx.x >> 5][3] / steps, pk_tacc[threadIdx.x >> 5][4] / steps, pk_tacc[threadIdx.x >> 5][5] / steps,
                 pk_tacc[threadIdx.x >> 5][6] / steps, pk_tacc[threadIdx.x >> 5][7] / steps);
#endif
        if (my_sp < S) a.Y[(long long)my_sp * a.ld + cidx] = cYp[my_sp].x;
        if (half == 0 && lane == 0) {
          a.T[cidx] = T;
          a.steps[cidx] = steps;
          if (a.status) a.status[cidx] = (unsigned char)st;
          if (st > 0) atomicMax(a.worst_status, st);
        }
        break;
      }
    }
  }
}

template <int NW, bool DENSE = false>
__global__ void __launch_bounds__(DENSE ? kPkThreads4 : kPkThreads, 1) stev_pk_kernel(const __grid_constant__ PkArgs a) {
  extern __shared__ __align__(128) unsigned char smem[];
  __shared__ unsigned long long mbar;
  __shared__ uint32_t tmem_base_s;
  __shared__ int done_warps;
  const int warp = __shfl_sync(0xffffffffu, (int)(threadIdx.x >> 5), 0), lane = threadIdx.x & 31;   // warp-uniform for the compiler
  if (threadIdx.x == 0) done_warps = 0;
  stage_tables(smem, a.table, a.tb.bytes, &mbar);
  if (warp == 0) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 512;" ::"r"(
                     (uint32_t)__cvta_generic_to_shared(&tmem_base_s))
                 : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  __syncthreads();
  asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
  const uint32_t tmem_base = tmem_base_s;

  // NW = 1: warp j is cell slot j.  NW = 2: warps j and 8 + (j + 1) % 8 form the pair of cell slot j.  The two warps of a
  // pair run the same phase at the same time, so they are placed on DIFFERENT schedulers (warp id mod 4): a scheduler
  // then interleaves four cells in four different phases (fp64-bound DFT against latency-bound gather and rates).
  const int half = (NW == 2) ? (warp >> 3) : 0;
  const int j = (NW == 2) ? (half ? ((warp - 8 + 7) & 7) : warp) : warp;
  if (j < a.cells_per_block) {
    unsigned char *cell = smem + a.tb.bytes + (size_t)j * a.cl.stride;
    if (a.tb.has_est) pk_worker<true, NW, DENSE>(a, smem, cell, j, half, warp & 3, tmem_base, lane);
    else pk_worker<false, NW, DENSE>(a, smem, cell, j, half, warp & 3, tmem_base, lane);
  }
  __syncwarp();
  if (lane == 0) atomicAdd(&done_warps, 1);
  if (warp == 0) {
    if (lane == 0) {
      while (atomicAdd(&done_warps, 0) < (int)(blockDim.x >> 5)) __nanosleep(200);
    }
    __syncwarp();
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 512;" ::"r"(tmem_base) : "memory");
  }
}

}  // namespace stev
