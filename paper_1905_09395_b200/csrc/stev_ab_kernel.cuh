// stev_ab_kernel.cuh -- the warp-specialised STEV integrator for large mechanisms (rows a1-a6 of DESIGN.md section 1).
//
// One block per SM holds up to eight cells.  Each cell is served by a pair of warps:
//   * the RATE warp ("A") walks the critical path of a step: thermo (NASA-7 / MLP), mixture sums, stabilised
//     concentrations, Arrhenius + equilibrium rates, source terms, the step limiter, the Euler update and retirement;
//   * the DFT warp ("B") runs the ringing detector of the previous step concurrently: it keeps the 13-deep history of
//     every reversible reaction in TENSOR MEMORY (one lane-private row of TMEM columns per reaction, written with
//     tcgen05.st and read back with tcgen05.ld), evaluates the DFT bins and produces the rOF factors of the next step.
// The two warps hand over through two named barriers per cell (bar.arrive / bar.sync, producer-consumer):
//   S2: A -> B "step published (q_eff, h, 1/C_tot)"      S1: B -> A "rOF of the next step ready".
// The history never touches HBM or shared memory; shared memory holds the mechanism tables (staged once per block by
// one TMA bulk copy) and ~10 KB of per-cell scratch.  Arithmetic follows the contract of DESIGN.md section 5 exactly;
// every deviation in evaluation order that is bit-equivalent is explained where it occurs.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

#include "stev_ab.cuh"
#include "stev_device.cuh"
#include "stev_fast.cuh"
#include "stev_math.cuh"

namespace stev {
// ---------------------------------------------------------------------------------------------------------
// DFT warp: row a5 of DESIGN.md.  TMEM address of slot s of this lane's reaction `it`:
//   base + (lane quarter << 16) + cell_half * 256 + it * 32 + 2 s.
// Two windows are processed side by side (independent dependency chains for the scheduler).
// ---------------------------------------------------------------------------------------------------------
template <int NHF>
__device__ __forceinline__ void ab_dft_warp(const AbArgs &a, unsigned char *cell, int j, uint32_t tmem_base, int lane) {
  const AbTables &tb = a.tb;
  const SolverConsts &sc = a.sc;
  const int Rrev = tb.Rrev, n_it = tb.n_it;
  double *cRof = (double *)(cell + a.cl.oRof);
  const double *cQ = (const double *)(cell + a.cl.oQ);
  volatile AbCtrl *ctrl = (volatile AbCtrl *)(cell + a.cl.oCtrl);
  const uint32_t trow = tmem_base + ((uint32_t)((j & 3) * 32) << 16) + (uint32_t)((j >> 2) * 256);
  const int barS2 = 2 * j, barS1 = 2 * j + 1;
  int slot = 0;

  auto reset = [&]() {
    for (int it = 0; it < n_it; ++it)
      for (int s = 0; s < kWindow; ++s) tmem_st2(trow + it * 32 + 2 * s, 0.0);   // R10: zero-initialised window
    tmem_wait_st();
    for (int k = lane; k < Rrev; k += 32) cRof[k] = 1.0;                         // Eq 11
    slot = 0;
  };
  auto update_rof = [&](int k, bool ringing) {
    double rof = cRof[k] * (ringing ? sc.inv_r_fac : sc.r_fac);   // Eqs 12-13
    if (rof > 1.0) rof = 1.0;
    if (rof < sc.rof_min) rof = sc.rof_min;
    cRof[k] = rof;
  };

  reset();
  __threadfence_block();
  named_bar_arrive(barS1);
  for (;;) {
    named_bar_sync(barS2);
    const int cmd = ctrl->cmd;
    if (cmd == kCmdExit) break;
    if (cmd == kCmdFinal) {
      reset();   // the cell retired: its last DFT is unobservable; prepare the next cell
    } else {
      const double h = ctrl->h, inv_ctot = ctrl->inv_ctot;
      // Eq 8 with R8, R9: the applied change in progress / C_tot of every reversible reaction goes into its window
      for (int it = 0; it < n_it; ++it) {
        const int k = it * 32 + lane;
        const double q = (k < Rrev) ? cQ[k] : 0.0;
        tmem_st2(trow + it * 32 + 2 * slot, (q * h) * inv_ctot);
      }
      tmem_wait_st();
      int it = 0;
      for (; it + 2 <= n_it; it += 2) {
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
      if (it < n_it) {
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
      }
      slot = (slot + 1 == kWindow) ? 0 : slot + 1;
    }
    __threadfence_block();
    named_bar_arrive(barS1);
  }
}

// ---------------------------------------------------------------------------------------------------------
// Rate warp: rows a1-a4, a6.
// ---------------------------------------------------------------------------------------------------------
template <bool EST>
__device__ __forceinline__ void ab_rate_warp(const AbArgs &a, const unsigned char *tbl, unsigned char *cell, int j, int lane) {
  const AbTables &tb = a.tb;
  const SolverConsts &sc = a.sc;
  const int S = tb.S, R = tb.R, Rrev = tb.Rrev, Rp = tb.Rp;
  double2 *cYp = (double2 *)(cell + a.cl.oYp);
  double2 *cYwCp = (double2 *)(cell + a.cl.oYwCp);
  double2 *cHOm = (double2 *)(cell + a.cl.oHOm);
  double *cConc = (double *)(cell + a.cl.oConc);
  double *cG = (double *)(cell + a.cl.oG);
  double *cQ = (double *)(cell + a.cl.oQ);
  double *cQraw = (double *)(cell + a.cl.oQraw);
  const double *cRof = (const double *)(cell + a.cl.oRof);
  float *cHid = (float *)(cell + a.cl.oHid);
  volatile AbCtrl *ctrl = (volatile AbCtrl *)(cell + a.cl.oCtrl);

  const double *tmid = (const double *)(tbl + tb.o_tmid), *W = (const double *)(tbl + tb.o_W);
  const double *invW = (const double *)(tbl + tb.o_invW), *nasa = (const double *)(tbl + tb.o_nasa);
  const double2 *rkA = (const double2 *)(tbl + tb.o_rkA), *rkB = (const double2 *)(tbl + tb.o_rkB);
  const uint4 *rfac = (const uint4 *)(tbl + tb.o_rfac), *rdg = (const uint4 *)(tbl + tb.o_rdg);
  const unsigned char *gsp = tbl + tb.o_gsp;
  const unsigned short *gent = (const unsigned short *)(tbl + tb.o_gent);
  const bool has2 = tb.n_var > 2;

  const int barS2 = 2 * j, barS1 = 2 * j + 1;
  const double dt_max = a.t_f * sc.delta_max;   // Eq 4
  const double t_tol = 1.0e-12 * a.t_f;         // R5

  if (lane == 0) {
    cConc[0] = 1.0;
    cG[0] = 0.0;
  }

  for (;;) {
    // ---- a6: variable load.  A retired cell's warp pair pulls the next active cell from the global queue.
    int pos = 0;
    if (lane == 0) pos = atomicAdd(a.queue_head, 1);
    pos = __shfl_sync(0xffffffffu, pos, 0);
    if ((long long)pos >= a.n_active) {
      named_bar_sync(barS1);          // the DFT warp has consumed the previous command
      if (lane == 0) ctrl->cmd = kCmdExit;
      __threadfence_block();
      named_bar_arrive(barS2);
      return;
    }
    const int cidx = a.list ? a.list[pos] : pos;
    double T = a.T[cidx];
    const double p = a.p[cidx];
    for (int i = lane; i < S; i += 32) cYp[i] = make_double2(a.Y[(long long)i * a.ld + cidx], invW[i]);
    double t = 0.0;
    int steps = 0;
    __syncwarp();

    for (;;) {
      // ================= part 1: everything that does not need rOF =================
      // -- scalars.  ln T and ln(p_atm / (R_u T)) are evaluated side by side in the two half-warps.
      const double RuT = kRu * T;
      const double c_tot = p / RuT;
      const double invT = 1.0 / T;
      const double larg = (lane & 16) ? (kPatm / RuT) : T;
      const double lval = ab_log(larg);
      const double lnT = __shfl_sync(0xffffffffu, lval, 0);
      const double ln_c0 = __shfl_sync(0xffffffffu, lval, 16);

      // -- a1: NASA-7 (Eqs 15-16, R17); g/RT always, cp and h unless the MLP supplies them.
      //    Two species per lane side by side; lanes past the end recompute the last species and store nothing.
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
        if (!EST) {
          cYwCp[ia].y = fma_rn(fma_rn(fma_rn(fma_rn(ca[4 * S], T, ca[3 * S]), T, ca[2 * S]), T, a2a), T, a1a);
          cHOm[ia].x = hRTa;
          if (ib_ < S) {
            cYwCp[ib].y = fma_rn(fma_rn(fma_rn(fma_rn(cb[4 * S], T, cb[3 * S]), T, cb[2 * S]), T, a2b), T, a1b);
            cHOm[ib].x = hRTb;
          }
        }
      }
      // -- a7 in the integrator (fp32 CUDA cores, R18): cp_i/R and h_i/(R T_ref) from the shallow MLP.
      if (EST) {
        const float *eshift = (const float *)(tbl + tb.o_eshift), *escale = (const float *)(tbl + tb.o_escale);
        const float *W1T = (const float *)(tbl + tb.o_W1T), *b1 = (const float *)(tbl + tb.o_b1);
        const float *W2p = (const float *)(tbl + tb.o_W2p), *b2 = (const float *)(tbl + tb.o_b2);
        const int H = tb.H, Hpad = tb.Hpad, n_in = tb.n_in, n_out = tb.n_out;
        for (int jh = lane; jh < H; jh += 32) {
          float z = b1[jh];
          for (int k = 0; k < n_in; ++k) {
            const double raw = (k == 0) ? T : ((k == 1) ? p : cYp[k - 2].x);
            const float xk = ((float)raw - eshift[k]) * escale[k];
            z = __fmaf_rn(W1T[k * H + jh], xk, z);
          }
          const double zd = (double)z;
          float act;
          if (tb.act == 0) act = (float)(1.0 - 2.0 / (1.0 + ab_exp(2.0 * zd)));
          else act = (float)(1.0 / (1.0 + ab_exp(-zd)));
          cHid[jh] = act;
        }
        __syncwarp();
        const float4 *hid4 = (const float4 *)cHid;
        for (int o0 = 0; o0 < n_out; o0 += 128) {
          float y[4];
          const float4 *wrow[4];
#pragma unroll
          for (int u = 0; u < 4; ++u) {
            int o = o0 + 32 * u + lane;
            o = (o < n_out) ? o : n_out - 1;
            y[u] = b2[o];
            wrow[u] = (const float4 *)(W2p + (size_t)o * Hpad);
          }
#pragma unroll 4
          for (int q4 = 0; q4 < H / 4; ++q4) {
            const float4 hv = hid4[q4];
#pragma unroll
            for (int u = 0; u < 4; ++u) {
              const float4 wv = wrow[u][q4];
              y[u] = __fmaf_rn(wv.x, hv.x, y[u]);
              y[u] = __fmaf_rn(wv.y, hv.y, y[u]);
              y[u] = __fmaf_rn(wv.z, hv.z, y[u]);
              y[u] = __fmaf_rn(wv.w, hv.w, y[u]);
            }
          }
#pragma unroll
          for (int u = 0; u < 4; ++u) {
            const int o = o0 + 32 * u + lane;
            if (o < n_out) {
              if (o < S) cYwCp[o].y = (double)y[u];
              else cHOm[o - S].x = ((double)y[u] * (double)tb.h_ref_T) * invT;
            }
          }
        }
        __syncwarp();
      }

      // -- mixture sums, sequential in species order (contract 5.4): 1/Wbar = sum Y_i/W_i and sum (Y_i/W_i) cp_i/R,
      //    two independent chains walked together
      double inv_wbar = 0.0, sum_cp = 0.0;
#pragma unroll 8
      for (int i = 0; i < S; ++i) {
        const double2 v = cYp[i];
        const double cp = cYwCp[i].y;
        inv_wbar = fma_rn(v.x, v.y, inv_wbar);
        sum_cp = fma_rn(v.x * v.y, cp, sum_cp);
      }
      const double rho = c_tot / inv_wbar;
      // -- small-species stabilisation (Eqs 6-7, R7): C** = gamma(y) rho y / W
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
        cConc[1 + ia] = ca;
        if (ib_ < S) cConc[1 + ib] = cb;
      }
      __syncwarp();

      // -- a2: rate constants and raw progress rates (Eqs 28-30).  Reversible reactions occupy
      //    internal indices [0, Rrev).  Each lane evaluates two reversible reactions side by side (four independent
      //    exp chains for the scheduler); lanes past the end recompute the last reaction and store nothing.
      for (int k0 = 0; k0 < Rrev; k0 += 64) {
        const int ka_ = k0 + lane, kb_ = ka_ + 32;
        const int ka = (ka_ < Rrev) ? ka_ : Rrev - 1, kb = (kb_ < Rrev) ? kb_ : Rrev - 1;
        const double2 pa0 = rkA[ka], pa1 = rkB[ka], pb0 = rkA[kb], pb1 = rkB[kb];
        const uint4 fa = rfac[ka], da = rdg[ka], fb = rfac[kb], db = rdg[kb];
        const double lkf_a = fma_rn(-pa1.x, invT, fma_rn(pa0.y, lnT, pa0.x));
        const double lkf_b = fma_rn(-pb1.x, invT, fma_rn(pb0.y, lnT, pb0.x));
        double dga = 0.0 - lds_f64(cell, da.x), dgb = 0.0 - lds_f64(cell, db.x);
        dga = dga - lds_f64(cell, da.y);
        dgb = dgb - lds_f64(cell, db.y);
        dga = dga + lds_f64(cell, da.z);
        dgb = dgb + lds_f64(cell, db.z);
        dga = dga + lds_f64(cell, da.w);
        dgb = dgb + lds_f64(cell, db.w);
        const double lkr_a = lkf_a - fma_rn(pa1.y, ln_c0, -dga);
        const double lkr_b = lkf_b - fma_rn(pb1.y, ln_c0, -dgb);
        double fwd_a, rev_a, fwd_b, rev_b;
        if (__any_sync(0xffffffffu, ab_exp_out_of_range(lkf_a) || ab_exp_out_of_range(lkr_a) ||
                                        ab_exp_out_of_range(lkf_b) || ab_exp_out_of_range(lkr_b))) {
          fwd_a = cexp(lkf_a); rev_a = cexp(lkr_a); fwd_b = cexp(lkf_b); rev_b = cexp(lkr_b);
        } else {
          fwd_a = ab_exp_core(lkf_a); rev_a = ab_exp_core(lkr_a); fwd_b = ab_exp_core(lkf_b); rev_b = ab_exp_core(lkr_b);
        }
        fwd_a = fwd_a * lds_f64(cell, fa.x);
        fwd_b = fwd_b * lds_f64(cell, fb.x);
        rev_a = rev_a * lds_f64(cell, fa.z);
        rev_b = rev_b * lds_f64(cell, fb.z);
        fwd_a = fwd_a * lds_f64(cell, fa.y);
        fwd_b = fwd_b * lds_f64(cell, fb.y);
        rev_a = rev_a * lds_f64(cell, fa.w);
        rev_b = rev_b * lds_f64(cell, fb.w);
        if (ka_ < Rrev) cQraw[ka] = fwd_a - rev_a;
        if (kb_ < Rrev) cQraw[kb] = fwd_b - rev_b;
      }
      // irreversible reactions: four per lane side by side; q_eff = q, so the stored multiples are written right
      // away (the DFT warp never reads them)
      for (int k0 = Rrev; k0 < R; k0 += 128) {
        double lk[4], fw[4];
        uint4 f[4];
        int kk[4];
        bool oor = false;
#pragma unroll
        for (int u = 0; u < 4; ++u) {
          kk[u] = k0 + 32 * u + lane;
          const int k = (kk[u] < R) ? kk[u] : R - 1;
          const double2 p0 = rkA[k];
          const double ta = rkB[k].x;
          f[u] = rfac[k];
          lk[u] = fma_rn(-ta, invT, fma_rn(p0.y, lnT, p0.x));
          oor = oor || ab_exp_out_of_range(lk[u]);
        }
        if (__any_sync(0xffffffffu, oor)) {
#pragma unroll
          for (int u = 0; u < 4; ++u) fw[u] = cexp(lk[u]);
        } else {
#pragma unroll
          for (int u = 0; u < 4; ++u) fw[u] = ab_exp_core(lk[u]);
        }
#pragma unroll
        for (int u = 0; u < 4; ++u) fw[u] = fw[u] * lds_f64(cell, f[u].x);
#pragma unroll
        for (int u = 0; u < 4; ++u) fw[u] = fw[u] * lds_f64(cell, f[u].y);
#pragma unroll
        for (int u = 0; u < 4; ++u) {
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

      // ================= part 2: needs rOF of this step (produced by the DFT warp) =================
      named_bar_sync(barS1);
      // effective rates (Eq 14) and their stored multiples +q, -q, +2q, -2q (all exact), which turn the sum
      // omega_i = sum_j nu_ij q_j into plain additions in the contract's order
      for (int k = lane; k < Rrev; k += 32) {
        const double q = cQraw[k] * cRof[k];
        cQ[k] = q;
        cQ[Rp + k] = -q;
        if (has2) {
          const double q2 = q + q;
          cQ[2 * Rp + k] = q2;
          cQ[3 * Rp + k] = -q2;
        }
      }
      __syncwarp();

      // -- source terms and the limiter (Eqs 1-3).  Lane l owns species gsp[l] and gsp[32+l]; the
      //    entry lists are padded with the 0.0 slot to a common length per round, so the loops are warp-uniform.
      const double inv_rho = 1.0 / rho;
      double t_star;
      {
        const int len0 = tb.g_len[0], len1 = tb.g_len[1];   // len1 <= len0 (the longest lists are in round 0)
        const unsigned short *ge0 = gent + lane, *ge1 = gent + len0 * 32 + lane;
        const int i0 = gsp[lane], i1 = gsp[32 + lane];
        double om0 = 0.0, om1 = 0.0;
        int e = 0;
#pragma unroll 4
        for (; e < len1; ++e) {
          om0 = om0 + lds_f64(cell, ge0[e * 32]);
          om1 = om1 + lds_f64(cell, ge1[e * 32]);
        }
#pragma unroll 8
        for (; e < len0; ++e) om0 = om0 + lds_f64(cell, ge0[e * 32]);
        // lanes without a species (i = 255) work on species 0 and discard the result
        const int j0 = (i0 < S) ? i0 : 0, j1 = (i1 < S) ? i1 : 0;
        const double r0 = (W[j0] * om0) * inv_rho, r1 = (W[j1] * om1) * inv_rho;
        const double y0 = cYp[j0].x, y1 = cYp[j1].x;
        const double rs0 = (-r0 > 1.0e-30) ? -r0 : 1.0e-30, rs1 = (-r1 > 1.0e-30) ? -r1 : 1.0e-30;
        const double ys0 = (y0 < 1.0e-20) ? 1.0 : 0.9 * y0, ys1 = (y1 < 1.0e-20) ? 1.0 : 0.9 * y1;
        const double lim0 = ((sc.y_step_max < ys0) ? sc.y_step_max : ys0) / rs0;
        const double lim1 = ((sc.y_step_max < ys1) ? sc.y_step_max : ys1) / rs1;
        const double inf = bits_to_double(0x7ff0000000000000ull);
        const double l0 = (i0 < S && lim0 < inf) ? lim0 : inf, l1 = (i1 < S) ? lim1 : inf;
        t_star = (l1 < l0) ? l1 : l0;
        if (i0 < S) {
          cConc[1 + i0] = r0;     // concentrations are dead: reuse for dY_i/dt
          cHOm[i0].y = om0;
        }
        if (i1 < S) {
          cConc[1 + i1] = r1;
          cHOm[i1].y = om1;
        }
      }
      // min over lanes: every lim is a positive double (or +inf / NaN), for which the ordering of the bit patterns
      // as unsigned integers is the ordering of the values; NaN patterns sort above +inf and are ignored like the
      // plain comparison `lim < t_star` ignores them.
      {
        const unsigned long long u = double_to_bits(t_star);
        const unsigned hi = (unsigned)(u >> 32), lo = (unsigned)u;
        const unsigned mhi = __reduce_min_sync(0xffffffffu, hi);
        const unsigned mlo = __reduce_min_sync(0xffffffffu, (hi == mhi) ? lo : 0xffffffffu);
        t_star = bits_to_double(((unsigned long long)mhi << 32) | mlo);
      }
      __syncwarp();

      // -- a3: step size (Eq 5) and landing on t_f (R5)
      double h = (t_star < dt_max) ? t_star : dt_max;
      bool last = false;
      const double rem = a.t_f - t;
      if (rem - h < t_tol) {
        h = rem;
        last = true;
      }
      // -- a4: forward Euler (Eq 18) for the species; the enthalpy sum of the temperature equation
      //    (R15) is sequential in species order
      int bad = 0;
      for (int i = lane; i < S; i += 32) {
        const double y = fma_rn(h, cConc[1 + i], cYp[i].x);
        cYp[i].x = y;
        bad |= !(y - y == 0.0);
      }
      double sum_h = 0.0;
#pragma unroll 8
      for (int i = 0; i < S; ++i) {
        const double2 v = cHOm[i];
        sum_h = fma_rn(v.x, v.y, sum_h);
      }
      const double dTdt = (sc.energy_mode == 0) ? -((sum_h * kRu) * T) / (rho * (kRu * sum_cp)) : 0.0;
      T = fma_rn(h, dTdt, T);
      t = last ? a.t_f : t + h;
      steps += 1;
      bad |= !(T - T == 0.0);
      bad = __any_sync(0xffffffffu, bad);

      // -- a6: retirement (R20)
      int st = -1;
      if (last) st = 0;
      else if (bad) st = 2;
      else if (steps >= sc.max_steps) st = 1;

      if (lane == 0) {
        ctrl->h = h;
        ctrl->inv_ctot = 1.0 / c_tot;
        ctrl->cmd = (st >= 0) ? kCmdFinal : kCmdStep;
      }
      __threadfence_block();
      named_bar_arrive(barS2);

      __syncwarp();
      if (st >= 0) {
        for (int i = lane; i < S; i += 32) a.Y[(long long)i * a.ld + cidx] = cYp[i].x;
        if (lane == 0) {
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

__global__ void __launch_bounds__(kAbThreads, 1) stev_ab_kernel(const __grid_constant__ AbArgs a) {
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

  // warps 0..7: DFT warp of cell slot j = warp (TMEM lane quarter j & 3 = warp & 3); warps 8..15: rate warp of j = warp - 8
  const bool is_dft = warp < kAbMaxCells;
  const int j = is_dft ? warp : warp - kAbMaxCells;
  if (j < a.cells_per_block) {
    unsigned char *cell = smem + a.tb.bytes + (size_t)j * a.cl.stride;
    if (is_dft) {
      switch (a.sc.nhf) {
        case 1: ab_dft_warp<1>(a, cell, j, tmem_base, lane); break;
        case 2: ab_dft_warp<2>(a, cell, j, tmem_base, lane); break;
        case 3: ab_dft_warp<3>(a, cell, j, tmem_base, lane); break;
        case 4: ab_dft_warp<4>(a, cell, j, tmem_base, lane); break;
        case 5: ab_dft_warp<5>(a, cell, j, tmem_base, lane); break;
        default: ab_dft_warp<6>(a, cell, j, tmem_base, lane); break;
      }
    }
    else if (a.tb.has_est) ab_rate_warp<true>(a, smem, cell, j, lane);
    else ab_rate_warp<false>(a, smem, cell, j, lane);
  }
  __syncwarp();
  if (lane == 0) atomicAdd(&done_warps, 1);
  if (warp == 0) {
    if (lane == 0) {
      while (atomicAdd(&done_warps, 0) < kAbThreads / 32) __nanosleep(200);
    }
    __syncwarp();
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 512;" ::"r"(tmem_base) : "memory");
  }
}

}  // namespace stev
