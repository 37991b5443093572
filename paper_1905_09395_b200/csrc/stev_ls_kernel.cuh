// stev_ls_kernel.cuh -- the lock-step STEV integrator (rows a1-a7 of DESIGN.md section 1); design in stev_ls.cuh.
//
// A step of the block (all C cell slots together) is five phases separated by block barriers:
//   0  scalar warp, one cell per lane: retirement / refill from the queue (a6), T-dependent scalars, 1/Wbar (sequential
//      sum), estimator inputs;  all warps: the ringing filter (a5) of the step just taken, over (cell, reversible
//      reaction) pairs -- it only feeds rOF, which phase 2 reads
//   1  (cell, species) pairs: NASA-7 g/RT (+ cp, h without estimator), stabilised concentrations;
//      (cell, hidden unit) pairs: first estimator layer (a7)
//   2  (cell, output) pairs: second estimator layer;  (cell, reaction) pairs: rates (a2), q_eff = q rOF, stored multiples
//   3  (cell, species) pairs: source terms gathered in the caller's reaction order, limiter (a3), atomicMin per cell
//   4  (cell, species) pairs: step size, Euler update (a4);  scalar warp: the two sequential sums of the temperature
//      equation, T, t, step count
// The 13-deep history of every reversible reaction lives in TENSOR MEMORY: pass p of 32 consecutive (cell, reaction)
// pairs belongs to warp p % 16 and sits in one 32-column slot of that warp's TMEM lane quarter.  tcgen05.st writes one
// column pair for all 32 lanes at once, so all cells of a block share the ring position: a slot is refilled only when
// the block's step counter is a multiple of 13 (the new cell then starts at physical slot 0, as the contract's R10 wants;
// a landed cell waits at most 12 steps, < 1.5 % of the shortest integrations of the five configurations).
// Arithmetic follows the contract of DESIGN.md section 5 exactly; the per-item arithmetic is the one of
// stev_pk_kernel.cuh, operation for operation.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

#include "stev_device.cuh"
#include "stev_fast.cuh"
#include "stev_ls.cuh"
#include "stev_math.cuh"

namespace stev {

// x / d for the small item counts of this kernel (x * d < 2^32): by a compile-time divisor when the shape is static,
// else through m = ceil(2^32 / d) (0 for d = 1)
template <class SH>
__device__ __forceinline__ unsigned ls_div(unsigned x, int d, unsigned m) {
  if (SH::kStatic) return x / (unsigned)(d > 0 ? d : 1);
  return m ? __umulhi(x, m) : x;
}
template <class SH>
struct LsConst {
  static constexpr LsLayout L = ls_layout_of(SH::D);
};
// dimension / layout field: a compile-time constant for a static shape, else read from the kernel arguments
#define LS_D(f) (SH::kStatic ? SH::D.f : a.tb.d.f)
#define LS_L(f) (SH::kStatic ? LsConst<SH>::L.f : a.lay.f)

constexpr unsigned kFull = 0xffffffffu;

// 26 consecutive columns of this lane back to tensor memory (x16 + x8 + x2)
__device__ __forceinline__ void tmem_st26(uint32_t taddr, const uint32_t (&r)[26]) {
  asm volatile(
      "tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16};" ::"r"(taddr),
      "r"(r[0]), "r"(r[1]), "r"(r[2]), "r"(r[3]), "r"(r[4]), "r"(r[5]), "r"(r[6]), "r"(r[7]), "r"(r[8]), "r"(r[9]), "r"(r[10]),
      "r"(r[11]), "r"(r[12]), "r"(r[13]), "r"(r[14]), "r"(r[15])
      : "memory");
  asm volatile("tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};" ::"r"(taddr + 16), "r"(r[16]),
               "r"(r[17]), "r"(r[18]), "r"(r[19]), "r"(r[20]), "r"(r[21]), "r"(r[22]), "r"(r[23])
               : "memory");
  asm volatile("tcgen05.st.sync.aligned.32x32b.x2.b32 [%0], {%1,%2};" ::"r"(taddr + 24), "r"(r[24]), "r"(r[25]) : "memory");
}

// ---------------------------------------------------------------------------------------------------------
// a5: the ringing filter (Eqs 8-13) of this warp's passes over the (cell, reversible reaction) pairs.
// slot13: ring position of the step whose applied change in progress is stored (the same for every cell of the block).
// ---------------------------------------------------------------------------------------------------------
template <class SH, int NHF>
__device__ __forceinline__ void ls_dft_passes(const LsArgs &a, unsigned char *cells, uint32_t trow, int slot13, int warp, int lane) {
  const SolverConsts &sc = a.sc;
  const int Rrev = LS_D(Rrev), n_rev_pass = LS_L(n_rev_pass);
  const unsigned n_items = (unsigned)(LS_D(C) * Rrev);
#pragma unroll
  for (int s = 0; s < kLsSlots; ++s) {
    const int p = warp + s * kLsWarps;
    if (p >= n_rev_pass) break;
    unsigned f = (unsigned)(p * 32 + lane);
    const bool valid = f < n_items;
    f = valid ? f : n_items - 1;
    const unsigned c = ls_div<SH>(f, Rrev, a.mRrev), k = f - c * (unsigned)Rrev;
    unsigned char *cell = cells + c * (unsigned)LS_L(stride);
    const LsScal *scl = (const LsScal *)(cell + LS_L(oSc));
    const bool on = valid && scl->dft_on;
    if (!__any_sync(kFull, on)) continue;   // landing steps and empty slots store nothing
    double *cRof = (double *)(cell + LS_L(oRof));
    const double q = ((const double *)(cell + LS_L(oQ)))[k];
    const uint32_t tw = trow + (uint32_t)(s * 32);
    // Eq 8 with R8, R9: the applied change in progress / C_tot.  (Lanes whose cell is not `on` overwrite a window that is
    // zeroed before its next use.)
    tmem_st2(tw + 2 * slot13, (q * scl->h_dft) * scl->ictot_dft);
    tmem_wait_st();
    uint32_t ra[26];
    tmem_ld26(tw, ra);
    tmem_wait_ld();
    double x[kWindow];
    unpack_window(ra, x);
    double d0, m2;
    ab_window_stats<NHF>(x, d0, m2);
    bool sure;
    bool ringing = ab_ring_filter(d0, m2, sc, sure);
    if (__any_sync(kFull, !sure && on)) ringing = ab_ring_exact(d0, m2, sc);
    if (on) {
      double rof = cRof[k] * (ringing ? sc.inv_r_fac : sc.r_fac);   // Eqs 12-13
      if (rof > 1.0) rof = 1.0;
      if (rof < sc.rof_min) rof = sc.rof_min;
      cRof[k] = rof;
    }
  }
}

// ---------------------------------------------------------------------------------------------------------
// a2: rates of this warp's passes over the (cell, reversible reaction) and (cell, irreversible reaction) pairs.
// The owner of a (cell, reaction) pair also owns its DFT window and its rOF: on the first step of a new cell it zeroes
// the window (R10) and sets rOF = 1 (Eq 11).
// ---------------------------------------------------------------------------------------------------------
template <class SH>
__device__ __forceinline__ void ls_rate_passes(const LsArgs &a, const unsigned char *tbl, unsigned char *cells, uint32_t trow, int warp,
                                               int lane) {
  const int Rrev = LS_D(Rrev), Rp = LS_L(Rp), Rirr = LS_D(R) - LS_D(Rrev);
  const int n_rev_pass = LS_L(n_rev_pass), n_irr_pass = LS_L(n_irr_pass);
  const bool has2 = LS_D(n_var) > 2;
  const double2 *rkA = (const double2 *)(tbl + LS_L(o_rkA)), *rkB = (const double2 *)(tbl + LS_L(o_rkB));
  const uint4 *rfac = (const uint4 *)(tbl + LS_L(o_rfac)), *rdg = (const uint4 *)(tbl + LS_L(o_rdg));
  const unsigned n_rev = (unsigned)(LS_D(C) * Rrev), n_irr = (unsigned)(LS_D(C) * Rirr);
#pragma unroll
  for (int s = 0; s < kLsSlots; ++s) {
    const int p = warp + s * kLsWarps;
    if (p >= n_rev_pass) break;
    unsigned f = (unsigned)(p * 32 + lane);
    const bool valid = f < n_rev;
    f = valid ? f : n_rev - 1;
    const unsigned c = ls_div<SH>(f, Rrev, a.mRrev), k = f - c * (unsigned)Rrev;
    unsigned char *cell = cells + c * (unsigned)LS_L(stride);
    const LsScal *scl = (const LsScal *)(cell + LS_L(oSc));
    double *cRof = (double *)(cell + LS_L(oRof)), *cQ = (double *)(cell + LS_L(oQ));
    const bool fresh = valid && scl->fresh;
    if (__any_sync(kFull, fresh)) {   // rare: once per cell
      const uint32_t tw = trow + (uint32_t)(s * 32);
      uint32_t ra[26];
      tmem_ld26(tw, ra);
      tmem_wait_ld();
      if (fresh) {
#pragma unroll
        for (int n = 0; n < 26; ++n) ra[n] = 0u;
        cRof[k] = 1.0;
      }
      tmem_st26(tw, ra);
      tmem_wait_st();
    }
    const double invT = scl->invT, lnT = scl->lnT, ln_c0 = scl->ln_c0;
    const double2 p0 = rkA[k], p1 = rkB[k];
    const uint4 d = rdg[k], fo = rfac[k];
    const double lkf = fma_rn(-p1.x, invT, fma_rn(p0.y, lnT, p0.x));
    double dg = 0.0 - lds_f64(cell, d.x);
    dg = dg - lds_f64(cell, d.y);
    dg = dg + lds_f64(cell, d.z);
    dg = dg + lds_f64(cell, d.w);
    const double lkr = lkf - fma_rn(p1.y, ln_c0, -dg);
    double fwd, rev;
    if (__any_sync(kFull, ab_exp_out_of_range(lkf) || ab_exp_out_of_range(lkr))) {
      fwd = cexp(lkf);
      rev = cexp(lkr);
    } else {
      fwd = ab_exp_core(lkf);
      rev = ab_exp_core(lkr);
    }
    fwd = fwd * lds_f64(cell, fo.x);
    rev = rev * lds_f64(cell, fo.z);
    fwd = fwd * lds_f64(cell, fo.y);
    rev = rev * lds_f64(cell, fo.w);
    const double q = (fwd - rev) * cRof[k];   // Eq 14
    if (valid) {
      cQ[k] = q;
      cQ[Rp + k] = -q;
      if (has2) {
        const double q2 = q + q;
        cQ[2 * Rp + k] = q2;
        cQ[3 * Rp + k] = -q2;
      }
    }
  }
  // irreversible reactions: passes continue round robin after the reversible ones, so the warps that had one pass less get these first
  for (int p = (warp - n_rev_pass) & (kLsWarps - 1); p < n_irr_pass; p += kLsWarps) {
    unsigned f = (unsigned)(p * 32 + lane);
    const bool valid = f < n_irr;
    f = valid ? f : n_irr - 1;
    const unsigned c = ls_div<SH>(f, Rirr, a.mRirr), k = (unsigned)Rrev + f - c * (unsigned)Rirr;
    unsigned char *cell = cells + c * (unsigned)LS_L(stride);
    const LsScal *scl = (const LsScal *)(cell + LS_L(oSc));
    double *cQ = (double *)(cell + LS_L(oQ));
    const double2 p0 = rkA[k];
    const double ta = rkB[k].x;
    const uint4 fo = rfac[k];
    const double lk = fma_rn(-ta, scl->invT, fma_rn(p0.y, scl->lnT, p0.x));
    double fw;
    if (__any_sync(kFull, ab_exp_out_of_range(lk))) fw = cexp(lk);
    else fw = ab_exp_core(lk);
    fw = fw * lds_f64(cell, fo.x);
    fw = fw * lds_f64(cell, fo.y);
    if (valid) {
      cQ[k] = fw;
      cQ[Rp + k] = -fw;
      if (has2) {
        const double f2 = fw + fw;
        cQ[2 * Rp + k] = f2;
        cQ[3 * Rp + k] = -f2;
      }
    }
  }
}

// ---------------------------------------------------------------------------------------------------------
// The kernel.
// ---------------------------------------------------------------------------------------------------------
template <class SH, bool EST>
__global__ void __launch_bounds__(kLsThreads, 1) stev_ls_kernel(const __grid_constant__ LsArgs a) {
  extern __shared__ __align__(128) unsigned char smem[];
  __shared__ unsigned long long mbar;
  __shared__ uint32_t tmem_base_s;
  __shared__ int s_go;
  const int tid = threadIdx.x;
  const int warp = __shfl_sync(kFull, tid >> 5, 0), lane = tid & 31;   // warp-uniform for the compiler
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
  const uint32_t trow = tmem_base + ((uint32_t)((warp & 3) * 32) << 16) + (uint32_t)((warp >> 2) * (32 * kLsSlots));

  const LsTables &tb = a.tb;
  const SolverConsts &sc = a.sc;
  const unsigned char *tbl = smem;
  unsigned char *cells = smem + tb.bytes;
  const int S = LS_D(S), C = LS_D(C);
  const double *W = (const double *)(tbl + LS_L(o_W)), *invW = (const double *)(tbl + LS_L(o_invW));
  const double *tmid = (const double *)(tbl + LS_L(o_tmid)), *nasa = (const double *)(tbl + LS_L(o_nasa));
  const double dt_max = a.t_f * sc.delta_max;   // Eq 4
  const double t_tol = 1.0e-12 * a.t_f;         // R5
  const unsigned n_cs = (unsigned)(C * S);
  const unsigned long long kInfBits = 0x7ff0000000000000ull;
  constexpr int SW = kLsWarps - 1;              // the scalar warp: it has the fewest reaction passes

  // the scalar lane of cell slot `lane` keeps the cell's own scalars in registers for the whole integration
  const bool my_slot = (warp == SW) && lane < C;
  unsigned char *my_cell = cells + (unsigned)(my_slot ? lane : 0) * (unsigned)LS_L(stride);
  LsScal *my_sc = (LsScal *)(my_cell + LS_L(oSc));
  double T = 1000.0, p = kPatm, t = 0.0, inv_ctot = 0.0, rho = 1.0;
  int steps = 0, cidx = -1, pending_st = -1;
  bool active = false, exhausted = false, last = false, bad_T = false;
  if (my_slot) {
    // a slot without a cell computes on a harmless finite state and commits nothing
    double2 *cYp = (double2 *)(my_cell + LS_L(oYp));
    for (int i = 0; i < S; ++i) cYp[i] = make_double2(1.0 / (double)S, invW[i]);
    ((double *)(my_cell + LS_L(oConc)))[0] = 1.0;
    ((double *)(my_cell + LS_L(oG)))[0] = 0.0;
    my_sc->active = 0;
    my_sc->fresh = 0;
    my_sc->dft_on = 0;
    my_sc->bad = 0;
    my_sc->h_dft = 0.0;
    my_sc->ictot_dft = 0.0;
  }
  __syncthreads();

  int g13 = 0;   // ring position of the step about to be taken (block-uniform)
  for (;;) {
    // =========================== phase 0 ===========================
    if (warp == SW) {
      // ---- a6: retirement (R20) of the step just taken
      if (my_slot && active) {
        int st = -1;
        if (bad_T || my_sc->bad) st = 2;            // checked first: a non-finite landing step is not "finished"
        else if (last) st = 0;
        else if (steps >= sc.max_steps) st = 1;
        if (st >= 0) {
          active = false;
          pending_st = st;
        }
      }
      if (g13 == 0) {
        // ---- results leave and new cells enter only at ring position 0 (see the header): write back ...
        if (my_slot && pending_st >= 0) {
          const double2 *cYp = (const double2 *)(my_cell + LS_L(oYp));
          for (int i = 0; i < S; ++i) a.Y[(long long)i * a.ld + cidx] = cYp[i].x;
          a.T[cidx] = T;
          a.steps[cidx] = steps;
          if (a.status) a.status[cidx] = (unsigned char)pending_st;
          if (pending_st > 0) atomicMax(a.worst_status, pending_st);
          pending_st = -1;
        }
        // ... and pull the next cells: ballot the requests, one atomic per warp reserves that many queue positions,
        // popc of the lower mask ranks them (variable load)
        const bool want = my_slot && !active && !exhausted;
        const unsigned req = __ballot_sync(kFull, want);
        if (req) {
          int base = 0;
          if (lane == 0) base = atomicAdd(a.queue_head, __popc(req));
          base = __shfl_sync(kFull, base, 0);
          if (want) {
            const long long pos = (long long)base + __popc(req & ((1u << lane) - 1u));
            if (pos < a.n_active) {
              cidx = a.list ? a.list[pos] : (int)pos;
              T = a.T[cidx];
              p = a.p[cidx];
              double2 *cYp = (double2 *)(my_cell + LS_L(oYp));
              for (int i = 0; i < S; ++i) cYp[i].x = a.Y[(long long)i * a.ld + cidx];
              t = 0.0;
              steps = 0;
              active = true;
              my_sc->fresh = 1;
            } else {
              exhausted = true;
            }
          }
        }
      }
      const int go = __any_sync(kFull, my_slot && (active || pending_st >= 0));
      if (lane == 0) s_go = go;
      if (my_slot) {
        // ---- scalars of this step
        const double RuT = kRu * T;
        const double c_tot = p / RuT;
        const double invT = 1.0 / T;
        const double lnT = ab_log(T);
        const double ln_c0 = ab_log(kPatm / RuT);
        inv_ctot = 1.0 / c_tot;
        // 1/Wbar = sum Y_i/W_i, sequential in species order (contract 5.4); estimator inputs on the way (R18)
        const double2 *cYp = (const double2 *)(my_cell + LS_L(oYp));
        double inv_wbar = 0.0;
        if (EST && LS_D(n_in) > 1) {
          float *cXn = (float *)(my_cell + LS_L(oHid)) + LS_D(H);
          const float *eshift = (const float *)(tbl + LS_L(o_eshift)), *escale = (const float *)(tbl + LS_L(o_escale));
          cXn[1] = ((float)p - eshift[1]) * escale[1];
          for (int i = 0; i < S; ++i) {
            const double2 v = cYp[i];
            inv_wbar = fma_rn(v.x, v.y, inv_wbar);
            cXn[2 + i] = ((float)v.x - eshift[2 + i]) * escale[2 + i];
          }
        } else {
#pragma unroll 4
          for (int i = 0; i < S; ++i) {
            const double2 v = cYp[i];
            inv_wbar = fma_rn(v.x, v.y, inv_wbar);
          }
        }
        if (EST) {
          float *cXn = (float *)(my_cell + LS_L(oHid)) + LS_D(H);
          cXn[0] = ((float)T - ((const float *)(tbl + LS_L(o_eshift)))[0]) * ((const float *)(tbl + LS_L(o_escale)))[0];
        }
        rho = c_tot / inv_wbar;
        my_sc->T = T;
        my_sc->p = p;
        my_sc->lnT = lnT;
        my_sc->ln_c0 = ln_c0;
        my_sc->invT = invT;
        my_sc->inv_ctot = inv_ctot;
        my_sc->rho = rho;
        my_sc->rem = a.t_f - t;
        my_sc->tstar_bits = kInfBits;
        my_sc->active = active ? 1 : 0;
        my_sc->bad = 0;
      }
    }
    // ---- a5 of the step just taken (its ring position is the one before g13)
    if (sc.dft_enable) {
      const int sl = (g13 == 0) ? kWindow - 1 : g13 - 1;
      switch (sc.nhf) {
        case 1: ls_dft_passes<SH, 1>(a, cells, trow, sl, warp, lane); break;
        case 2: ls_dft_passes<SH, 2>(a, cells, trow, sl, warp, lane); break;
        case 3: ls_dft_passes<SH, 3>(a, cells, trow, sl, warp, lane); break;
        case 4: ls_dft_passes<SH, 4>(a, cells, trow, sl, warp, lane); break;
        case 5: ls_dft_passes<SH, 5>(a, cells, trow, sl, warp, lane); break;
        default: ls_dft_passes<SH, 6>(a, cells, trow, sl, warp, lane); break;
      }
    }
    __syncthreads();
    if (!s_go) break;

    // =========================== phase 1: a1 thermo, concentrations, first estimator layer ===========================
    for (unsigned it = (unsigned)tid; it < n_cs; it += kLsThreads) {
      const unsigned c = ls_div<SH>(it, S, a.mS), i = it - c * (unsigned)S;
      unsigned char *cell = cells + c * (unsigned)LS_L(stride);
      const LsScal *scl = (const LsScal *)(cell + LS_L(oSc));
      const double Tc = scl->T, invT = scl->invT, lnT = scl->lnT, rho_c = scl->rho;
      double *cG = (double *)(cell + LS_L(oG)), *cConc = (double *)(cell + LS_L(oConc));
      double2 *cYwCp = (double2 *)(cell + LS_L(oYwCp)), *cHOm = (double2 *)(cell + LS_L(oHOm));
      // NASA-7 (Eqs 15-16, R17): g/RT and 2 g/RT always, cp/R and h/RT without an estimator
      const double *ca = nasa + ((Tc < tmid[i]) ? 0 : kNasaRows * S) + i;
      const double a1a = ca[0], a2a = ca[S];
      const double hpa = fma_rn(fma_rn(fma_rn(fma_rn(ca[8 * S], Tc, ca[7 * S]), Tc, ca[6 * S]), Tc, ca[5 * S]), Tc, a1a);
      const double hRTa = fma_rn(ca[9 * S], invT, hpa);
      const double spa = fma_rn(fma_rn(fma_rn(ca[12 * S], Tc, ca[11 * S]), Tc, ca[10 * S]), Tc, a2a);
      const double sRa = fma_rn(a1a, lnT, fma_rn(spa, Tc, ca[13 * S]));
      const double ga = hRTa - sRa;
      cG[1 + i] = ga;
      cG[1 + S + i] = ga + ga;
      if (!EST) {
        cYwCp[i].y = fma_rn(fma_rn(fma_rn(fma_rn(ca[4 * S], Tc, ca[3 * S]), Tc, ca[2 * S]), Tc, a2a), Tc, a1a);
        cHOm[i].x = hRTa;
      }
      // Y_i/W_i (for the cp sum) and the small-species stabilisation (Eqs 6-7, R7): C** = gamma(y) rho y / W
      const double2 va = ((const double2 *)(cell + LS_L(oYp)))[i];
      const double ypa = (va.x > 0.0) ? va.x : 0.0;
      double cc = (rho_c * ypa) * va.y;
      if (sc.alpha > 0.0) cc = (ypa / (sc.alpha + ypa)) * cc;
      cYwCp[i].x = va.x * va.y;
      cConc[1 + i] = cc;
    }
    if (EST) {
      // hidden units, dealt from the last thread downwards (the first threads have the species above)
      const int H = LS_D(H), n_in = LS_D(n_in);
      const float *W1T = (const float *)(tbl + LS_L(o_W1T)), *b1 = (const float *)(tbl + LS_L(o_b1));
      for (unsigned it = (unsigned)(kLsThreads - 1 - tid); it < (unsigned)(C * H); it += kLsThreads) {
        const unsigned c = ls_div<SH>(it, H, a.mH), j = it - c * (unsigned)H;
        float *cHid = (float *)(cells + c * (unsigned)LS_L(stride) + LS_L(oHid));
        const float *cXn = cHid + H;
        float z = b1[j];
        const float *w = W1T + j;
        for (int k = 0; k < n_in; ++k, w += H) z = __fmaf_rn(w[0], cXn[k], z);
        const double zd = (double)z;
        cHid[j] = (tb.act == 0) ? (float)(1.0 - 2.0 / (1.0 + ab_exp(2.0 * zd))) : (float)(1.0 / (1.0 + ab_exp(-zd)));
      }
    }
    __syncthreads();

    // =========================== phase 2: second estimator layer, a2 rates ===========================
    if (EST) {
      const int H = LS_D(H), n_out = LS_D(n_out);
      const float *W2p = (const float *)(tbl + LS_L(o_W2p)), *b2 = (const float *)(tbl + LS_L(o_b2));
      for (unsigned it = (unsigned)tid; it < (unsigned)(C * n_out); it += kLsThreads) {
        const unsigned c = ls_div<SH>(it, n_out, a.mNout), o = it - c * (unsigned)n_out;
        unsigned char *cell = cells + c * (unsigned)LS_L(stride);
        const float4 *hid4 = (const float4 *)(cell + LS_L(oHid));
        const float4 *wrow = (const float4 *)(W2p + (size_t)o * LS_L(Hpad));
        float y = b2[o];
#pragma unroll 4
        for (int q4 = 0; q4 < H / 4; ++q4) {
          const float4 hv = hid4[q4], wv = wrow[q4];
          y = __fmaf_rn(wv.x, hv.x, y);
          y = __fmaf_rn(wv.y, hv.y, y);
          y = __fmaf_rn(wv.z, hv.z, y);
          y = __fmaf_rn(wv.w, hv.w, y);
        }
        if (o < (unsigned)S) ((double2 *)(cell + LS_L(oYwCp)))[o].y = (double)y;
        else ((double2 *)(cell + LS_L(oHOm)))[o - S].x = ((double)y * (double)tb.h_ref_T) * ((const LsScal *)(cell + LS_L(oSc)))->invT;
      }
    }
    ls_rate_passes<SH>(a, tbl, cells, trow, warp, lane);
    __syncthreads();

    // =========================== phase 3: source terms and the limiter (Eqs 1-3) ===========================
    {
      const unsigned char *gsp = tbl + LS_L(o_gsp);
      const unsigned short *grow = (const unsigned short *)(tbl + LS_L(o_grow)), *glen = (const unsigned short *)(tbl + LS_L(o_glen));
      const uint4 *gent = (const uint4 *)(tbl + LS_L(o_gent));
      for (unsigned base = (unsigned)(warp * 32); base < n_cs; base += kLsThreads) {
        unsigned it = base + (unsigned)lane;
        const bool valid = it < n_cs;
        it = valid ? it : n_cs - 1;
        const unsigned r = ls_div<SH>(it, C, a.mC), c = it - r * (unsigned)C;   // lanes of one species (same list) side by side
        unsigned char *cell = cells + c * (unsigned)LS_L(stride);
        const int i = gsp[r];
        const int row0 = grow[r], rows = glen[r];
        const int max_rows = __reduce_max_sync(kFull, rows);
        double om = 0.0;
        // entries in the caller's reaction order; a shorter list reads the all-padding row (the 0.0 slot; om is never -0.0)
        uint4 o = gent[(0 < rows) ? row0 : tb.g_zero_row];
        for (int e = 0; e < max_rows; ++e) {
          const double v0 = lds_f64(cell, o.x), v1 = lds_f64(cell, o.y), v2 = lds_f64(cell, o.z), v3 = lds_f64(cell, o.w);
          o = gent[(e + 1 < rows) ? row0 + e + 1 : tb.g_zero_row];
          om = om + v0;
          om = om + v1;
          om = om + v2;
          om = om + v3;
        }
        LsScal *scl = (LsScal *)(cell + LS_L(oSc));
        const double inv_rho = 1.0 / scl->rho;
        const double r0 = (W[i] * om) * inv_rho;
        const double y0 = ((const double2 *)(cell + LS_L(oYp)))[i].x;
        const double rs0 = (-r0 > 1.0e-30) ? -r0 : 1.0e-30;                       // Eq 1
        const double ys0 = (y0 < 1.0e-20) ? 1.0 : 0.9 * y0;                       // Eq 2 (R2)
        const double lim0 = ((sc.y_step_max < ys0) ? sc.y_step_max : ys0) / rs0;  // Eq 3
        if (valid) {
          ((double *)(cell + LS_L(oConc)))[1 + i] = r0;     // concentrations are dead: reuse for dY_i/dt
          ((double2 *)(cell + LS_L(oHOm)))[i].y = om;
          // min over species: every lim is a positive double, for which the ordering of the bit patterns as unsigned
          // integers is the ordering of the values; NaN is ignored like the contract's plain comparison ignores it
          if (lim0 < bits_to_double(kInfBits)) atomicMin(&scl->tstar_bits, double_to_bits(lim0));
        }
      }
    }
    __syncthreads();

    // =========================== phase 4: a3 step size, a4 update ===========================
    for (unsigned it = (unsigned)tid; it < n_cs; it += kLsThreads) {
      const unsigned c = ls_div<SH>(it, S, a.mS), i = it - c * (unsigned)S;
      unsigned char *cell = cells + c * (unsigned)LS_L(stride);
      LsScal *scl = (LsScal *)(cell + LS_L(oSc));
      const double t_star = bits_to_double(scl->tstar_bits);
      double h = (t_star < dt_max) ? t_star : dt_max;       // Eq 5
      const double rem = scl->rem;
      if (rem - h < t_tol) h = rem;                          // landing on t_f (R5)
      if (scl->active) {
        double2 *cYp = (double2 *)(cell + LS_L(oYp));
        const double y = fma_rn(h, ((const double *)(cell + LS_L(oConc)))[1 + i], cYp[i].x);   // Eq 18
        cYp[i].x = y;
        if (!(y - y == 0.0)) atomicOr(&scl->bad, 1);
      }
    }
    if (my_slot) {
      const double t_star = bits_to_double(my_sc->tstar_bits);
      double h = (t_star < dt_max) ? t_star : dt_max;
      const double rem = a.t_f - t;
      bool lst = false;
      if (rem - h < t_tol) {
        h = rem;
        lst = true;
      }
      // temperature equation (R15): sum (Y_i/W_i) cp_i/R and sum (h_i/RT) omega_i, each sequential in species order
      const double2 *cYwCp = (const double2 *)(my_cell + LS_L(oYwCp)), *cHOm = (const double2 *)(my_cell + LS_L(oHOm));
      double sum_cp = 0.0, sum_h = 0.0;
#pragma unroll 4
      for (int i = 0; i < S; ++i) {
        const double2 u = cYwCp[i], v = cHOm[i];
        sum_cp = fma_rn(u.x, u.y, sum_cp);
        sum_h = fma_rn(v.x, v.y, sum_h);
      }
      const double dTdt = (sc.energy_mode == 0) ? -((sum_h * kRu) * T) / (rho * (kRu * sum_cp)) : 0.0;
      my_sc->fresh = 0;
      my_sc->h_dft = h;
      my_sc->ictot_dft = inv_ctot;
      my_sc->dft_on = (active && !lst) ? 1 : 0;   // the landing step's change is never looked at: the cell retires
      if (active) {
        T = fma_rn(h, dTdt, T);
        bad_T = !(T - T == 0.0);
        t = lst ? a.t_f : t + h;
        steps += 1;
        last = lst;
      }
    }
    __syncthreads();
    g13 = (g13 + 1 == kWindow) ? 0 : g13 + 1;
  }

  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  __syncthreads();
  if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 512;" ::"r"(tmem_base) : "memory");
}

}  // namespace stev
