// stev_ls_kernel.cuh -- the lock-step STEV integrator (rows a1-a7 of DESIGN.md section 1); design in stev_ls.cuh.
//
// A step of the block (all C cell slots together) is four phases separated by block barriers:
//   1  (species, cell) pairs: NASA-7 g/RT (+ cp, h without estimator), stabilised concentrations;
//      (hidden unit, cell) pairs: first estimator layer (a7)
//   2  (reaction, cell) pairs: rates (a2), q_eff = q rOF, stored multiples
//   3  (species, cell) pairs: source terms gathered in the caller's reaction order, limiter (a3), atomicMin per cell;
//      (output, cell) pairs: second estimator layer (it only feeds the temperature equation)
//   4  the serial chain of the method on the SCALAR WARP, one cell per lane -- step size and landing, one loop over the
//      species that carries the two sequential sums of the temperature equation and, behind the update of each mass
//      fraction (a4), 1/Wbar of the new state, then T, t, step count, retirement / refill from the queue (a6) and for
//      the NEXT step the two logarithms and the divisions (spread over lane groups) -- while the fifteen other warps run
//      the whole ringing filter (a5) of the step: the filter only feeds rOF, which the rates of the next step read, so
//      the fp64-bound filter hides the chain.  The scalars exist in two sets used by alternate steps, so the scalar
//      warp can write the next step's while the filter still reads this step's.  The scalar warp owns no reversible
//      (reaction, cell) pairs; beside the three filter warps of its scheduler it gets one issue slot in four, so its chain
//      is bound by its instruction count.
// The 13-deep history of every reversible reaction lives in TENSOR MEMORY: pass p of 32 consecutive (reaction, cell)
// pairs belongs to the pass warp of rank p % 15 and sits in one 32-column slot of that warp's TMEM lane quarter.  tcgen05.st writes one
// column pair for all 32 lanes at once, so all cells of a block share the ring position: a slot is refilled only when
// the block's step counter is a multiple of 13 (the new cell then starts at physical slot 0, as the contract's R10 wants;
// a landed cell waits at most 12 steps, < 1.5 % of the shortest integrations of the five configurations).
// Arithmetic follows the contract of DESIGN.md section 5 exactly.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

#include "stev_device.cuh"
#include "stev_fast.cuh"
#include "stev_ls.cuh"
#include "stev_math.cuh"

namespace stev {

template <class SH>
struct LsConst {
  static constexpr LsLayout L = ls_layout_of(SH::D);
};
// dimension / layout field: a compile-time constant for a static shape, else read from the kernel arguments
#define LS_D(f) (SH::kStatic ? SH::D.f : a.tb.d.f)
#define LS_L(f) (SH::kStatic ? LsConst<SH>::L.f : a.lay.f)
// element (idx, c) of the cell-region array of reals at byte offset `off` (index-major, cell-minor)
#define LS_AT(type, off, idx, c) (*(type *)(cells + (off) + (unsigned)((idx) * C + (c)) * (unsigned)sizeof(type)))
// scalar `field` of cell c in the scalar set at byte offset sc_set: eight-byte entries whatever the type
#define LS_SC(type, field, c) (*(type *)(cells + sc_set + ((unsigned)((int)(field) * C + (c)) << 3)))

constexpr unsigned kFull = 0xffffffffu;

// x / C for the small item counts of this kernel (x * C < 2^32): by a compile-time divisor when the shape is static,
// else through m = ceil(2^32 / C) (0 for C = 1)
template <class SH>
__device__ __forceinline__ unsigned ls_div_c(unsigned x, int C, unsigned m) {
  if (SH::kStatic) return x / (unsigned)(C > 0 ? C : 1);
  return m ? __umulhi(x, m) : x;
}

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

// the thirteen floats of a binary32 window: 13 consecutive columns of this lane (x8 + x4 + x1)
__device__ __forceinline__ void tmem_ld13(uint32_t taddr, uint32_t (&r)[13]) {
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
               : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7])
               : "r"(taddr)
               : "memory");
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x4.b32 {%0,%1,%2,%3}, [%4];"
               : "=r"(r[8]), "=r"(r[9]), "=r"(r[10]), "=r"(r[11])
               : "r"(taddr + 8)
               : "memory");
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x1.b32 {%0}, [%1];" : "=r"(r[12]) : "r"(taddr + 12) : "memory");
}
__device__ __forceinline__ void tmem_st13(uint32_t taddr, const uint32_t (&r)[13]) {
  asm volatile("tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};" ::"r"(taddr), "r"(r[0]), "r"(r[1]),
               "r"(r[2]), "r"(r[3]), "r"(r[4]), "r"(r[5]), "r"(r[6]), "r"(r[7])
               : "memory");
  asm volatile("tcgen05.st.sync.aligned.32x32b.x4.b32 [%0], {%1,%2,%3,%4};" ::"r"(taddr + 8), "r"(r[8]), "r"(r[9]), "r"(r[10]),
               "r"(r[11])
               : "memory");
  asm volatile("tcgen05.st.sync.aligned.32x32b.x1.b32 [%0], {%1};" ::"r"(taddr + 12), "r"(r[12]) : "memory");
}
__device__ __forceinline__ void tmem_st1(uint32_t taddr, float v) {
  asm volatile("tcgen05.st.sync.aligned.32x32b.x1.b32 [%0], {%1};" ::"r"(taddr), "r"(__float_as_uint(v)) : "memory");
}

// Shared-memory store the compiler does not see as a memory access: the loads of the following loop iterations (other
// addresses, by construction) may be scheduled above it.  The caller closes the loop with a compiler barrier.
__device__ __forceinline__ void ls_sts_unordered(double *p, double v) {
  asm volatile("st.shared.f64 [%0], %1;" ::"r"((uint32_t)__cvta_generic_to_shared(p)), "d"(v));
}
__device__ __forceinline__ void ls_sts_unordered(float *p, float v) {
  asm volatile("st.shared.f32 [%0], %1;" ::"r"((uint32_t)__cvta_generic_to_shared(p)), "f"(v));
}

// The pieces of a step that differ between the two precisions (DESIGN.md sections 5 and 5b).
template <typename RT> struct LsReal;
template <> struct LsReal<double> {
  using bits_t = unsigned long long;
  static __device__ __forceinline__ bits_t inf_bits() { return 0x7ff0000000000000ull; }
  // v is infinite or NaN, i.e. !(v - v == 0): the exponent field is all ones (no fp64 instruction)
  static __device__ __forceinline__ bool nonfinite(double v) { return ((unsigned)__double2hiint(v) & 0x7ff00000u) == 0x7ff00000u; }
  static __device__ __forceinline__ double from_bits(bits_t u) { return bits_to_double(u); }
  static __device__ __forceinline__ bits_t to_bits(double v) { return double_to_bits(v); }
  // forward and reverse exponentials of a batch: the generic routine only if any lane of the warp is out of range
  template <int U>
  static __device__ __forceinline__ void exp_pairs(const double (&lkf)[U], const double (&lkr)[U], double (&fwd)[U], double (&rev)[U]) {
    bool oor = false;
#pragma unroll
    for (int u = 0; u < U; ++u) oor = oor || ab_exp_out_of_range(lkf[u]) || ab_exp_out_of_range(lkr[u]);
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
  }
  static __device__ __forceinline__ double exp1(double x) {
    if (__any_sync(0xffffffffu, ab_exp_out_of_range(x))) return cexp(x);
    return ab_exp_core(x);
  }
  static __device__ __forceinline__ float activation(float z, int act) {
    const double zd = (double)z;
    return (act == 0) ? (float)(1.0 - 2.0 / (1.0 + ab_exp(2.0 * zd))) : (float)(1.0 / (1.0 + ab_exp(-zd)));
  }
  // stores the new sample in column pair `slot13` of the window at tw, reads the window back, decides Eq 12
  template <int NHF>
  static __device__ __forceinline__ bool window_rings(uint32_t tw, int slot13, double v, bool on, const SolverConsts &sc) {
    tmem_st2(tw + 2 * slot13, v);
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
    if (__any_sync(0xffffffffu, !sure && on)) ringing = ab_ring_exact(d0, m2, sc);
    return ringing;
  }
  static __device__ __forceinline__ void window_zero_if(uint32_t tw, bool fresh) {
    uint32_t ra[26];
    tmem_ld26(tw, ra);
    tmem_wait_ld();
    if (fresh) {
#pragma unroll
      for (int n = 0; n < 26; ++n) ra[n] = 0u;
    }
    tmem_st26(tw, ra);
    tmem_wait_st();
  }
};
template <> struct LsReal<float> {
  using bits_t = unsigned int;
  static __device__ __forceinline__ bits_t inf_bits() { return 0x7f800000u; }
  static __device__ __forceinline__ bool nonfinite(float v) { return (__float_as_uint(v) & 0x7f800000u) == 0x7f800000u; }
  static __device__ __forceinline__ float from_bits(bits_t u) { return __uint_as_float(u); }
  static __device__ __forceinline__ bits_t to_bits(float v) { return __float_as_uint(v); }
  template <int U>
  static __device__ __forceinline__ void exp_pairs(const float (&lkf)[U], const float (&lkr)[U], float (&fwd)[U], float (&rev)[U]) {
#pragma unroll
    for (int u = 0; u < U; ++u) {
      fwd[u] = cexpf32(lkf[u]);
      rev[u] = cexpf32(lkr[u]);
    }
  }
  static __device__ __forceinline__ float exp1(float x) { return cexpf32(x); }
  static __device__ __forceinline__ float activation(float z, int act) {
    return (act == 0) ? 1.0f - 2.0f / (1.0f + cexpf32(2.0f * z)) : 1.0f / (1.0f + cexpf32(-z));
  }
  template <int NHF>
  static __device__ __forceinline__ bool window_rings(uint32_t tw, int slot13, float v, bool on, const SolverConsts &sc) {
    tmem_st1(tw + slot13, v);
    tmem_wait_st();
    uint32_t ra[13];
    tmem_ld13(tw, ra);
    tmem_wait_ld();
    float x[kWindow];
#pragma unroll
    for (int n = 0; n < kWindow; ++n) x[n] = __uint_as_float(ra[n]);
    return dft_is_ringing<float>(x, sc);   // Eqs 9-12 as written (float sqrt and division are cheap)
  }
  static __device__ __forceinline__ void window_zero_if(uint32_t tw, bool fresh) {
    uint32_t ra[13];
    tmem_ld13(tw, ra);
    tmem_wait_ld();
    if (fresh) {
#pragma unroll
      for (int n = 0; n < 13; ++n) ra[n] = 0u;
    }
    tmem_st13(tw, ra);
    tmem_wait_st();
  }
};

// ---------------------------------------------------------------------------------------------------------
// a5: the ringing filter (Eqs 8-13) of pass `s` of this warp over the (reversible reaction, cell) pairs,
// run in phase 4 of the step whose applied change in progress it stores: the step size follows from the limiter's
// minimum exactly as in the update.  slot13: ring position of the step (the same for every cell of the block).
// ---------------------------------------------------------------------------------------------------------
template <class SH, typename RT, int NHF>
__device__ __forceinline__ void ls_dft_all(const LsArgs &a, unsigned char *cells, int sc_set, uint32_t trow, int slot13, int prank,
                                           int lane, RT dt_max, RT t_tol) {
  using LR = LsReal<RT>;
  const SolverConsts &sc = a.sc;
  const int C = LS_D(C);
  const unsigned n_items = (unsigned)(C * LS_D(Rrev));
  // what a pass needs of its cell: the step size (from the limiter's minimum, exactly as the update forms it), 1/C_tot,
  // and whether the step's change is looked at -- not on the landing step (the cell retires), not in an empty slot
  RT h = RT(0), ic = RT(0);
  bool cell_on = false;
  auto load_cell = [&](unsigned c) {
    const RT t_star = LR::from_bits(LS_SC(typename LR::bits_t, kF_TSTAR, c));
    h = (t_star < dt_max) ? t_star : dt_max;
    const RT rem = LS_SC(RT, kF_REM, c);
    const bool lst = rem - h < t_tol;
    h = lst ? rem : h;
    ic = LS_SC(RT, kF_ICTOT, c);
    cell_on = LS_SC(int, kF_ACTIVE, c) && !lst;
  };
  const bool fixed_cell = (32 % C) == 0;   // then a lane holds the same cell in every pass
  if (fixed_cell) load_cell((unsigned)lane % (unsigned)C);
#pragma unroll 1
  for (int s = 0; s < ls_slots((int)sizeof(RT)); ++s) {
    const int p = prank + s * kLsPassWarps;
    if (p >= LS_L(n_rev_pass)) break;
    unsigned f = (unsigned)(p * 32 + lane);
    const bool valid = f < n_items;
    f = valid ? f : n_items - 1;
    const unsigned k = ls_div_c<SH>(f, C, a.mC), c = f - k * (unsigned)C;
    if (!fixed_cell) load_cell(c);
    const bool on = valid && cell_on;
    if (!__any_sync(kFull, on)) continue;   // landing steps and empty slots store nothing
    const RT q = LS_AT(RT, LS_L(oQ), k, c);
    // Eq 8 with R8, R9: the applied change in progress / C_tot.  (Lanes whose cell is not `on` overwrite a window that is
    // zeroed before its next use.)
    const bool ringing = LR::template window_rings<NHF>(trow + (uint32_t)(s * ls_slot_pitch((int)sizeof(RT))), slot13, (q * h) * ic, on, sc);
    if (on) {
      RT &rof_ref = LS_AT(RT, LS_L(oRof), k, c);
      RT rof = rof_ref * (ringing ? MathT<RT>::inv_r_fac(sc) : (RT)sc.r_fac);   // Eqs 12-13
      if (rof > RT(1)) rof = RT(1);
      if (rof < (RT)sc.rof_min) rof = (RT)sc.rof_min;
      rof_ref = rof;
    }
  }
}

template <class SH, typename RT>
__device__ __forceinline__ void ls_dft(const LsArgs &a, unsigned char *cells, int sc_set, uint32_t trow, int slot13, int prank, int lane,
                                       RT dt_max, RT t_tol) {
  if (!a.sc.dft_enable) return;
  if (sizeof(RT) == 4) {   // the binary32 filter reads the first high bin at run time
    ls_dft_all<SH, RT, 0>(a, cells, sc_set, trow, slot13, prank, lane, dt_max, t_tol);
    return;
  }
  switch (a.sc.nhf) {
    case 1: ls_dft_all<SH, RT, 1>(a, cells, sc_set, trow, slot13, prank, lane, dt_max, t_tol); break;
    case 2: ls_dft_all<SH, RT, 2>(a, cells, sc_set, trow, slot13, prank, lane, dt_max, t_tol); break;
    case 3: ls_dft_all<SH, RT, 3>(a, cells, sc_set, trow, slot13, prank, lane, dt_max, t_tol); break;
    case 4: ls_dft_all<SH, RT, 4>(a, cells, sc_set, trow, slot13, prank, lane, dt_max, t_tol); break;
    case 5: ls_dft_all<SH, RT, 5>(a, cells, sc_set, trow, slot13, prank, lane, dt_max, t_tol); break;
    default: ls_dft_all<SH, RT, 6>(a, cells, sc_set, trow, slot13, prank, lane, dt_max, t_tol); break;
  }
}

// two reals / four table offsets of a reaction
template <typename RT> struct alignas(2 * sizeof(RT)) LsPair { RT x, y; };

// What the rate passes need of a cell.  When C divides 32 a lane holds the same cell (lane % C) in every pass, and the
// caller loads these once per step (fixed = true); otherwise every pass loads its own.
template <typename RT> struct LsCellScalars {
  bool fixed;
  unsigned c;
  RT invT, lnT, ln_c0;
  int fresh;
};
template <typename RT>
__device__ __forceinline__ LsCellScalars<RT> ls_cell_scalars(const unsigned char *cells, int sc_set, int C, unsigned c) {
  LsCellScalars<RT> v;
  v.fixed = true;
  v.c = c;
  v.invT = *(const RT *)(cells + sc_set + ((unsigned)((int)kF_INVT * C + (int)c) << 3));
  v.lnT = *(const RT *)(cells + sc_set + ((unsigned)((int)kF_LNT * C + (int)c) << 3));
  v.ln_c0 = *(const RT *)(cells + sc_set + ((unsigned)((int)kF_LNC0 * C + (int)c) << 3));
  v.fresh = *(const int *)(cells + sc_set + ((unsigned)((int)kF_FRESH * C + (int)c) << 3));
  return v;
}

// ---------------------------------------------------------------------------------------------------------
// a2: rates of passes s0 .. s0 + U - 1 of this warp over the (reversible reaction, cell) pairs, side by side (2 U
// independent exponential chains in flight).  The owner of a pair also owns its DFT window and its rOF: on the first
// step of a new cell it zeroes the window (R10) and sets rOF = 1 (Eq 11).
// ---------------------------------------------------------------------------------------------------------
template <class SH, typename RT, int U>
__device__ __forceinline__ void ls_rev_batch(const LsArgs &a, const unsigned char *tbl, unsigned char *cells, int sc_set, uint32_t trow,
                                             int s0, int warp, int lane, const LsCellScalars<RT> &cs) {
  using M = MathT<RT>;
  using LR = LsReal<RT>;
  const int C = LS_D(C), Rrev = LS_D(Rrev), Rp = LS_L(Rp);
  const bool has2 = LS_D(n_var) > 2;
  const unsigned n_rev = (unsigned)(C * Rrev);
  unsigned k[U], c[U];
  bool valid[U];
  RT lkf[U], lkr[U], cx[U], cy[U], cz[U], cw[U], rof[U];
  uint4 fo[U];
#pragma unroll
  for (int u = 0; u < U; ++u) {
    const int p = warp + (s0 + u) * kLsPassWarps;
    unsigned f = (unsigned)(p * 32 + lane);
    valid[u] = f < n_rev;
    f = valid[u] ? f : n_rev - 1;
    k[u] = ls_div_c<SH>(f, C, a.mC);
    c[u] = cs.fixed ? cs.c : f - k[u] * (unsigned)C;   // (a lane beyond the last pair computes on (R_rev - 1, its own cell) and stores nothing)
    const bool fresh = valid[u] && (cs.fixed ? cs.fresh : LS_SC(int, kF_FRESH, c[u]));
    if (__any_sync(kFull, fresh)) {   // rare: once per cell
      LR::window_zero_if(trow + (uint32_t)((s0 + u) * ls_slot_pitch((int)sizeof(RT))), fresh);
      if (fresh) LS_AT(RT, LS_L(oRof), k[u], c[u]) = RT(1);
    }
  }
#pragma unroll
  for (int u = 0; u < U; ++u) {
    const unsigned char *cc = cells + c[u] * (unsigned)sizeof(RT);   // this lane's cell column
    const RT invT = cs.fixed ? cs.invT : LS_SC(RT, kF_INVT, c[u]), lnT = cs.fixed ? cs.lnT : LS_SC(RT, kF_LNT, c[u]);
    const RT ln_c0 = cs.fixed ? cs.ln_c0 : LS_SC(RT, kF_LNC0, c[u]);
    const LsPair<RT> p0 = ((const LsPair<RT> *)(tbl + LS_L(o_rkA)))[k[u]], p1 = ((const LsPair<RT> *)(tbl + LS_L(o_rkB)))[k[u]];
    const uint4 d = ((const uint4 *)(tbl + LS_L(o_rdg)))[k[u]];
    fo[u] = ((const uint4 *)(tbl + LS_L(o_rfac)))[k[u]];
    lkf[u] = M::fma(-p1.x, invT, M::fma(p0.y, lnT, p0.x));
    RT dg = RT(0) - *(const RT *)(cc + d.x);
    dg = dg - *(const RT *)(cc + d.y);
    dg = dg + *(const RT *)(cc + d.z);
    dg = dg + *(const RT *)(cc + d.w);
    lkr[u] = lkf[u] - M::fma(p1.y, ln_c0, -dg);
    // the concentration factors and rOF are fetched here, under the exponentials, not behind them
    cx[u] = *(const RT *)(cc + fo[u].x);
    cy[u] = *(const RT *)(cc + fo[u].y);
    cz[u] = *(const RT *)(cc + fo[u].z);
    cw[u] = *(const RT *)(cc + (fo[u].w & 0x7fffffffu));
    rof[u] = LS_AT(RT, LS_L(oRof), k[u], c[u]);
  }
  RT fwd[U], rev[U];
  LR::template exp_pairs<U>(lkf, lkr, fwd, rev);
#pragma unroll
  for (int u = 0; u < U; ++u) {
    fwd[u] = fwd[u] * cx[u];
    rev[u] = rev[u] * cz[u];
    fwd[u] = fwd[u] * cy[u];
    rev[u] = rev[u] * cw[u];
    const RT q = (fwd[u] - rev[u]) * rof[u];   // Eq 14
    if (valid[u]) {
      LS_AT(RT, LS_L(oQ), k[u], c[u]) = q;
      LS_AT(RT, LS_L(oQ), Rp + k[u], c[u]) = -q;
      if (has2 && (fo[u].w >> 31)) {   // only a reaction with a coefficient of 2 has readers of these
        const RT q2 = q + q;
        LS_AT(RT, LS_L(oQ), 2 * Rp + k[u], c[u]) = q2;
        LS_AT(RT, LS_L(oQ), 3 * Rp + k[u], c[u]) = -q2;
      }
    }
  }
}

// passes [s0, s1) of this warp, two at a time while two are left
template <class SH, typename RT>
__device__ __forceinline__ void ls_rev_range(const LsArgs &a, const unsigned char *tbl, unsigned char *cells, int sc_set, uint32_t trow,
                                             int s0, int s1, int warp, int lane, const LsCellScalars<RT> &cs) {
  const int n_mine = (LS_L(n_rev_pass) - warp + kLsPassWarps - 1) / kLsPassWarps;   // passes of this warp
  s1 = (s1 < n_mine) ? s1 : n_mine;
  int s = s0;
  for (; s + 2 <= s1; s += 2) ls_rev_batch<SH, RT, 2>(a, tbl, cells, sc_set, trow, s, warp, lane, cs);
  if (s < s1) ls_rev_batch<SH, RT, 1>(a, tbl, cells, sc_set, trow, s, warp, lane, cs);
}

// irreversible reactions: passes continue round robin after the reversible ones, so the warps that had one pass less get
// these first
template <class SH, typename RT>
__device__ __forceinline__ void ls_irr_passes(const LsArgs &a, const unsigned char *tbl, unsigned char *cells, int sc_set, int warp, int lane,
                                              const LsCellScalars<RT> &cs) {
  using M = MathT<RT>;
  const int C = LS_D(C), Rrev = LS_D(Rrev), Rp = LS_L(Rp), Rirr = LS_D(R) - LS_D(Rrev);
  const int n_irr_pass = LS_L(n_irr_pass);
  const bool has2 = LS_D(n_var) > 2;
  const unsigned n_irr = (unsigned)(C * Rirr);
  (void)n_irr_pass;
  for (int p = a.tb.irr_start[warp], p_end = p + a.tb.irr_count[warp]; p < p_end; ++p) {
    unsigned f = (unsigned)(p * 32 + lane);
    const bool valid = f < n_irr;
    f = valid ? f : n_irr - 1;
    const unsigned kk = ls_div_c<SH>(f, C, a.mC), c = cs.fixed ? cs.c : f - kk * (unsigned)C, k = (unsigned)Rrev + kk;
    const unsigned char *cc = cells + c * (unsigned)sizeof(RT);
    const LsPair<RT> p0 = ((const LsPair<RT> *)(tbl + LS_L(o_rkA)))[k];
    const RT ta = ((const LsPair<RT> *)(tbl + LS_L(o_rkB)))[k].x;
    const uint4 fo = ((const uint4 *)(tbl + LS_L(o_rfac)))[k];
    const RT lk = M::fma(-ta, cs.fixed ? cs.invT : LS_SC(RT, kF_INVT, c), M::fma(p0.y, cs.fixed ? cs.lnT : LS_SC(RT, kF_LNT, c), p0.x));
    const RT cx = *(const RT *)(cc + fo.x), cy = *(const RT *)(cc + fo.y);   // fetched under the exponential
    RT fw = LsReal<RT>::exp1(lk);
    fw = fw * cx;
    fw = fw * cy;
    if (valid) {
      LS_AT(RT, LS_L(oQ), k, c) = fw;
      LS_AT(RT, LS_L(oQ), Rp + k, c) = -fw;
      if (has2 && (fo.w >> 31)) {
        const RT f2 = fw + fw;
        LS_AT(RT, LS_L(oQ), 2 * Rp + k, c) = f2;
        LS_AT(RT, LS_L(oQ), 3 * Rp + k, c) = -f2;
      }
    }
  }
}

// ---------------------------------------------------------------------------------------------------------
// The kernel.
// ---------------------------------------------------------------------------------------------------------
#ifdef LS_TIMING
#define LST(i) { const long long now_ = clock64(); tph[i] += now_ - tl_; tl_ = now_; }
#else
#define LST(i)
#endif

template <class SH, bool EST, typename RT>
__global__ void __launch_bounds__(kLsThreads, 1) stev_ls_kernel(const __grid_constant__ LsArgs a) {
  using M = MathT<RT>;
  using LR = LsReal<RT>;
  using bits_t = typename LR::bits_t;
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
  const uint32_t trow = tmem_base + ((uint32_t)((warp & 3) * 32) << 16) + (uint32_t)((warp >> 2) * 128);

  const LsTables &tb = a.tb;
  const SolverConsts &sc = a.sc;
  const unsigned char *tbl = smem;
  unsigned char *cells = smem + tb.bytes;
  const int S = LS_D(S), C = LS_D(C);
  const RT *W = (const RT *)(tbl + LS_L(o_W)), *invW = (const RT *)(tbl + LS_L(o_invW));
  const RT *tmid = (const RT *)(tbl + LS_L(o_tmid)), *nasa = (const RT *)(tbl + LS_L(o_nasa));
  const RT t_f = (RT)a.t_f;
  const RT dt_max = t_f * (RT)sc.delta_max;     // Eq 4
  const RT t_tol = M::land_tol() * t_f;         // R5 (R26 in binary32)
  const RT alpha = (RT)sc.alpha, y_step_max = (RT)sc.y_step_max;
  const unsigned n_cs = (unsigned)(C * S);
  const bits_t kInfBits = LR::inf_bits();
  constexpr int SW = kLsWarps - 1;              // the scalar warp
  // Passes over the (reversible reaction, cell) pairs are dealt in the order 0 1 2 4 5 6 8 9 10 12 13 14 3 7 11: when the
  // count is not a multiple of fifteen, the warps that share a scheduler (warp % 4) with the scalar warp get one less.
  const int prank = ((warp & 3) == 3) ? 12 + (warp >> 2) : (warp >> 2) * 3 + (warp & 3);

  // the scalar lane of cell slot `lane` keeps the cell's own scalars in registers for the whole integration
  const bool my_slot = (warp == SW) && lane < C;
  const int mc = my_slot ? lane : 0;
  RT T = RT(1000), p = M::patm(), t = RT(0), inv_ctot = RT(0), rho = RT(1);
  int steps = 0, cidx = -1, pending_st = -1;
  bool active = false, exhausted = false, last = false, bad_T = false;
  int sc_set = LS_L(oSc);   // scalar set of the current step; the other one is at LS_L(oSc) + LS_L(sc_bytes)
  if (my_slot) {
    // a slot without a cell computes on a harmless finite state and commits nothing
    for (int i = 0; i < S; ++i) LS_AT(RT, LS_L(oY), i, mc) = RT(1) / (RT)S;
    LS_AT(RT, LS_L(oConc), 0, mc) = RT(1);
    LS_AT(RT, LS_L(oG), 0, mc) = RT(0);
  }
#ifdef LS_TIMING
  long long tph[6] = {0, 0, 0, 0, 0, 0}, tl_ = clock64(), n_steps_ = 0;
#endif

  // What the scalar warp does between two steps: retirement of the step just taken (a6), write-back and refill at ring
  // position 0, and the scalars of the next step into scalar set `set_next`.  g_next: ring position of the next step.
  // inv_wbar: sum Y_i/W_i of the updated mass fractions (from the fused loop of phase 4; recomputed here for a new cell).
  auto scalar_warp_prepare = [&](int set_next, int g_next, bool first, RT inv_wbar, bool bad_y) {
    const int sc_keep = sc_set;
    if (!first) {
      // ---- a6: retirement (R20) of the step just taken
      if (my_slot && active) {
        int st = -1;
        if (bad_T || bad_y) st = 2;   // checked first: a non-finite landing step is not "finished"
        else if (last) st = 0;
        else if (steps >= sc.max_steps) st = 1;
        if (st >= 0) {
          active = false;
          pending_st = st;
        }
      }
    }
    sc_set = set_next;
    int fresh = 0;
    if (g_next == 0) {
      // ---- results leave and new cells enter only at ring position 0 (see the header): write back ...
      if (my_slot && pending_st >= 0) {
        for (int i = 0; i < S; ++i) a.Y[(long long)i * a.ld + cidx] = (double)LS_AT(RT, LS_L(oY), i, mc);
        a.T[cidx] = (double)T;
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
            T = (RT)a.T[cidx];
            p = (RT)a.p[cidx];
            for (int i = 0; i < S; ++i) LS_AT(RT, LS_L(oY), i, mc) = (RT)a.Y[(long long)i * a.ld + cidx];
            t = RT(0);
            steps = 0;
            active = true;
            fresh = 1;
          } else {
            exhausted = true;
          }
        }
      }
    }
    const int go = __any_sync(kFull, my_slot && (active || pending_st >= 0));
    if (lane == 0) s_go = go;
    // ---- scalars of the next step.  The chain per cell is five divisions and two logarithms; the lanes of the scalar warp
    // beyond the C cell lanes take their share: with C <= 8 four lane groups (lane = group * 8 + cell), with C <= 16 two,
    // each evaluating one quotient / logarithm of the cell at a time with the same instructions on different operands.
    // 1/Wbar = sum Y_i/W_i, sequential in species order (contract 5.4), comes from the fused loop of phase 4; a new cell
    // (and the very first call) computes it here, with the estimator inputs on the way (R18).
    if (my_slot && (first || fresh)) {
      inv_wbar = RT(0);
      if (EST && LS_D(n_in) > 1) {
        float *cXn = (float *)(cells + LS_L(oXn));
        const float *eshift = (const float *)(tbl + LS_L(o_eshift)), *escale = (const float *)(tbl + LS_L(o_escale));
        for (int i = 0; i < S; ++i) {
          const RT y = LS_AT(RT, LS_L(oY), i, mc);
          inv_wbar = M::fma(y, invW[i], inv_wbar);
          cXn[(2 + i) * C + mc] = ((float)y - eshift[2 + i]) * escale[2 + i];
        }
      } else {
#pragma unroll 4
        for (int i = 0; i < S; ++i) inv_wbar = M::fma(LS_AT(RT, LS_L(oY), i, mc), invW[i], inv_wbar);
      }
    }
    RT lnT, ln_c0, invT, c_tot, inv_rho;
    const int cp = (C <= 8) ? 8 : ((C <= 16) ? 16 : 32);   // lanes per group
    const int src = lane & (cp - 1);                        // the cell's own lane (group 0)
    const int grp = lane / cp;
    const RT Tb = __shfl_sync(kFull, T, src), pb = __shfl_sync(kFull, p, src), iwb = __shfl_sync(kFull, inv_wbar, src);
    const RT RuT = M::ru() * Tb;
    if (cp == 8) {
      // group 0: p_atm / (R_u T), ln of it;  group 1: c_tot = p / (R_u T), 1 / c_tot;  group 2: 1 / T;  groups 1-3: ln T;
      // groups 0, 2, 3: rho = c_tot / (1/Wbar)
      const RT q1 = ((grp == 1) ? pb : ((grp == 2) ? RT(1) : M::patm())) / ((grp == 2) ? Tb : RuT);
      const RT lv = M::log((grp == 0) ? q1 : Tb);
      c_tot = __shfl_sync(kFull, q1, src + 8);
      const RT q3 = ((grp == 1) ? RT(1) : c_tot) / ((grp == 1) ? q1 : iwb);
      ln_c0 = lv;
      lnT = __shfl_sync(kFull, lv, src + 8);
      invT = __shfl_sync(kFull, q1, src + 16);
      inv_ctot = __shfl_sync(kFull, q3, src + 8);
      rho = q3;
      inv_rho = RT(1) / rho;
    } else if (cp == 16) {
      // group 0: p_atm / (R_u T), ln of it, 1 / T;  group 1: c_tot, ln T, 1 / c_tot;  both: rho
      const RT q1 = ((grp == 1) ? pb : M::patm()) / RuT;
      const RT lv = M::log((grp == 0) ? q1 : Tb);
      const RT q2 = RT(1) / ((grp == 1) ? q1 : Tb);
      c_tot = __shfl_sync(kFull, q1, src + 16);
      ln_c0 = lv;
      lnT = __shfl_sync(kFull, lv, src + 16);
      invT = q2;
      inv_ctot = __shfl_sync(kFull, q2, src + 16);
      rho = c_tot / iwb;
      inv_rho = RT(1) / rho;
    } else {
      lnT = M::log(Tb);
      ln_c0 = M::log(M::patm() / RuT);
      c_tot = pb / RuT;
      invT = RT(1) / Tb;
      inv_ctot = RT(1) / c_tot;
      rho = c_tot / iwb;
      inv_rho = RT(1) / rho;
    }
    if (my_slot) {
      if (EST) {
        float *cXn = (float *)(cells + LS_L(oXn));
        const float *eshift = (const float *)(tbl + LS_L(o_eshift)), *escale = (const float *)(tbl + LS_L(o_escale));
        cXn[mc] = ((float)T - eshift[0]) * escale[0];
        if (LS_D(n_in) > 1) cXn[1 * C + mc] = ((float)p - eshift[1]) * escale[1];
      }
      LS_SC(RT, kF_T, mc) = T;
      LS_SC(RT, kF_P, mc) = p;
      LS_SC(RT, kF_LNT, mc) = lnT;
      LS_SC(RT, kF_LNC0, mc) = ln_c0;
      LS_SC(RT, kF_INVT, mc) = invT;
      LS_SC(RT, kF_ICTOT, mc) = inv_ctot;
      LS_SC(RT, kF_RHO, mc) = rho;
      LS_SC(RT, kF_INVRHO, mc) = inv_rho;
      LS_SC(RT, kF_REM, mc) = t_f - t;
      LS_SC(bits_t, kF_TSTAR, mc) = kInfBits;
      LS_SC(int, kF_ACTIVE, mc) = active ? 1 : 0;
      LS_SC(int, kF_FRESH, mc) = fresh;
    }
    sc_set = sc_keep;
  };

  // ---- before the first step: the scalar warp fills the slots and prepares scalar set 0
  if (warp == SW) scalar_warp_prepare(LS_L(oSc), 0, true, RT(0), false);
  __syncthreads();

  // The thread's first (species, cell) item of phase 3 never changes: its species, the rows of its source-term list and
  // the longest list of its warp are looked up once, not at the head of every step's gather.
  unsigned g_c = 0;
  int g_i = 0, g_row0 = 0, g_rows = 0, g_max = 0;
  {
    unsigned it = (unsigned)(warp * 32 + lane);
    it = (it < n_cs) ? it : n_cs - 1;
    const unsigned r = ls_div_c<SH>(it, C, a.mC);
    g_c = it - r * (unsigned)C;
    g_i = (tbl + LS_L(o_gsp))[r];
    g_row0 = ((const unsigned short *)(tbl + LS_L(o_grow)))[r];
    g_rows = ((const unsigned short *)(tbl + LS_L(o_glen)))[r];
    g_max = __reduce_max_sync(kFull, g_rows);
  }

  int g13 = 0;   // ring position of the step being taken (block-uniform)
  while (s_go) {
    // =========================== phase 1: a1 thermo, concentrations, first estimator layer ===========================
    for (unsigned it = (unsigned)tid; it < n_cs; it += kLsThreads) {
      const unsigned i = ls_div_c<SH>(it, C, a.mC), c = it - i * (unsigned)C;
      const RT Tc = LS_SC(RT, kF_T, c), invT = LS_SC(RT, kF_INVT, c), lnT = LS_SC(RT, kF_LNT, c);
      const RT rho_c = LS_SC(RT, kF_RHO, c);
      // NASA-7 (Eqs 15-16, R17): g/RT and 2 g/RT always, cp/R and h/RT without an estimator
      const RT *ca = nasa + ((Tc < tmid[i]) ? 0 : kNasaRows * S) + i;
      const RT a1a = ca[0], a2a = ca[S];
      const RT hpa = M::fma(M::fma(M::fma(M::fma(ca[8 * S], Tc, ca[7 * S]), Tc, ca[6 * S]), Tc, ca[5 * S]), Tc, a1a);
      const RT hRTa = M::fma(ca[9 * S], invT, hpa);
      const RT spa = M::fma(M::fma(M::fma(ca[12 * S], Tc, ca[11 * S]), Tc, ca[10 * S]), Tc, a2a);
      const RT sRa = M::fma(a1a, lnT, M::fma(spa, Tc, ca[13 * S]));
      const RT ga = hRTa - sRa;
      LS_AT(RT, LS_L(oG), 1 + i, c) = ga;
      LS_AT(RT, LS_L(oG), 1 + S + i, c) = ga + ga;
      if (!EST) {
        LS_AT(RT, LS_L(oCp), i, c) = M::fma(M::fma(M::fma(M::fma(ca[4 * S], Tc, ca[3 * S]), Tc, ca[2 * S]), Tc, a2a), Tc, a1a);
        LS_AT(RT, LS_L(oH), i, c) = hRTa;
      }
      // Y_i/W_i (for the cp sum) and the small-species stabilisation (Eqs 6-7, R7): C** = gamma(y) rho y / W
      const RT y = LS_AT(RT, LS_L(oY), i, c), iw = invW[i];
      const RT ypa = (y > RT(0)) ? y : RT(0);
      RT cc = (rho_c * ypa) * iw;
      if (alpha > RT(0)) cc = (ypa / (alpha + ypa)) * cc;
      LS_AT(RT, LS_L(oYw), i, c) = y * iw;
      LS_AT(RT, LS_L(oConc), 1 + i, c) = cc;
    }
    if (EST) {
      const int H = LS_D(H), n_in = LS_D(n_in);
      const float *W1T = (const float *)(tbl + LS_L(o_W1T)), *b1 = (const float *)(tbl + LS_L(o_b1));
      const float *cXn = (const float *)(cells + LS_L(oXn));
      float *cHid = (float *)(cells + LS_L(oHid));
      if (C * H >= 4 * kLsThreads) {
        // many hidden units (config 4: 2,048 (unit, cell) pairs): a thread takes FOUR CONSECUTIVE units of one cell
        // (n_hidden is a multiple of 8), dealt from the last thread downwards -- one 16-byte load per weight row, one
        // load of the input, four independent fmaf / tanh chains side by side (config 4: +5.5 %)
        const unsigned n_grp4 = (unsigned)(C * (H >> 2));
        for (unsigned it0 = (unsigned)(kLsThreads - 1 - tid); it0 < n_grp4; it0 += kLsThreads) {
          const unsigned g = ls_div_c<SH>(it0, C, a.mC), c = it0 - g * (unsigned)C;
          const float4 bz = ((const float4 *)b1)[g];
          float z0 = bz.x, z1 = bz.y, z2 = bz.z, z3 = bz.w;
          const float4 *w4 = (const float4 *)W1T + g;
          const float *xc = cXn + c;
          for (int k = 0; k < n_in; ++k) {
            const float xk = xc[k * C];
            const float4 wv = w4[k * (H >> 2)];
            z0 = __fmaf_rn(wv.x, xk, z0);
            z1 = __fmaf_rn(wv.y, xk, z1);
            z2 = __fmaf_rn(wv.z, xk, z2);
            z3 = __fmaf_rn(wv.w, xk, z3);
          }
          float4 hv;
          hv.x = LR::activation(z0, tb.act);
          hv.y = LR::activation(z1, tb.act);
          hv.z = LR::activation(z2, tb.act);
          hv.w = LR::activation(z3, tb.act);
          *(float4 *)(cHid + c * (unsigned)LS_L(Hs) + 4 * g) = hv;
        }
      } else {
        // few hidden units (config 3: 256 pairs): one unit per thread from the last thread downwards, so that the tanh
        // chains (latency-bound) are spread over as many warps as there are (four chains on two warps: -10 %)
        for (unsigned it = (unsigned)(kLsThreads - 1 - tid); it < (unsigned)(C * H); it += kLsThreads) {
          const unsigned j = ls_div_c<SH>(it, C, a.mC), c = it - j * (unsigned)C;
          float z = b1[j];
          const float *w = W1T + j;
          const float *xc = cXn + c;
          for (int k = 0; k < n_in; ++k) z = __fmaf_rn(w[k * H], xc[k * C], z);
          cHid[c * LS_L(Hs) + j] = LR::activation(z, tb.act);
        }
      }
    }
    LST(1)
    __syncthreads();
    LST(5)

    // =========================== phase 2: a2 rates ===========================
    {
      LsCellScalars<RT> cs{};
      if ((32 % C) == 0) cs = ls_cell_scalars<RT>(cells, sc_set, C, (unsigned)lane % (unsigned)C);
      if (warp != SW) ls_rev_range<SH, RT>(a, tbl, cells, sc_set, trow, 0, ls_slots((int)sizeof(RT)), prank, lane, cs);
      ls_irr_passes<SH, RT>(a, tbl, cells, sc_set, prank, lane, cs);
    }
    LST(2)
    __syncthreads();
    LST(5)

    // =========================== phase 3: source terms and the limiter (Eqs 1-3) ===========================
    {
      const unsigned char *gsp = tbl + LS_L(o_gsp);
      const unsigned short *grow = (const unsigned short *)(tbl + LS_L(o_grow)), *glen = (const unsigned short *)(tbl + LS_L(o_glen));
      const uint4 *gent = (const uint4 *)(tbl + LS_L(o_gent));
      for (unsigned base = (unsigned)(warp * 32); base < n_cs; base += kLsThreads) {
        unsigned it = base + (unsigned)lane;
        const bool valid = it < n_cs;
        it = valid ? it : n_cs - 1;
        // lanes of one species (same list) side by side
        unsigned c;
        int i, row0, rows, max_rows;
        if (base == (unsigned)(warp * 32)) {
          c = g_c; i = g_i; row0 = g_row0; rows = g_rows; max_rows = g_max;
        } else {
          const unsigned r = ls_div_c<SH>(it, C, a.mC);
          c = it - r * (unsigned)C;
          i = gsp[r];
          row0 = grow[r];
          rows = glen[r];
          max_rows = __reduce_max_sync(kFull, rows);
        }
        const unsigned char *cc = cells + c * (unsigned)sizeof(RT);
        // what the limiter needs besides the sum is fetched before the gather, not behind it
        const RT inv_rho = LS_SC(RT, kF_INVRHO, c), w_i = W[i], y0 = LS_AT(RT, LS_L(oY), i, c);
        RT om = RT(0);
        // entries in the caller's reaction order; a shorter list reads the all-padding row (the 0.0 slot; om is never -0.0).
        // The values of the next row are fetched before this row is added.
        uint4 o = gent[(0 < rows) ? row0 : tb.g_zero_row];
        RT v0 = *(const RT *)(cc + o.x), v1 = *(const RT *)(cc + o.y), v2 = *(const RT *)(cc + o.z), v3 = *(const RT *)(cc + o.w);
        o = gent[(1 < rows) ? row0 + 1 : tb.g_zero_row];
        for (int e = 0; e < max_rows; ++e) {
          const RT u0 = v0, u1 = v1, u2 = v2, u3 = v3;
          v0 = *(const RT *)(cc + o.x);
          v1 = *(const RT *)(cc + o.y);
          v2 = *(const RT *)(cc + o.z);
          v3 = *(const RT *)(cc + o.w);
          o = gent[(e + 2 < rows) ? row0 + e + 2 : tb.g_zero_row];
          om = om + u0;
          om = om + u1;
          om = om + u2;
          om = om + u3;
        }
        const RT r0 = (w_i * om) * inv_rho;
        const RT rs0 = (-r0 > M::r_floor()) ? -r0 : M::r_floor();                 // Eq 1
        const RT ys0 = (y0 < M::y_small()) ? RT(1) : M::ninety() * y0;            // Eq 2 (R2)
        const RT lim0 = ((y_step_max < ys0) ? y_step_max : ys0) / rs0;            // Eq 3
        if (valid) {
          LS_AT(RT, LS_L(oConc), 1 + i, c) = r0;     // concentrations are dead: reuse for dY_i/dt
          LS_AT(RT, LS_L(oOm), i, c) = om;
        }
        // min over species: every lim is a positive real, for which the ordering of the bit patterns as unsigned
        // integers is the ordering of the values; NaN is ignored like the contract's plain comparison ignores it.
        // When C divides 32 the lanes lane, lane + C, lane + 2C ... hold the same cell: they reduce by shuffles and
        // one lane per cell goes to the shared atomic.
        bits_t lb = (valid && lim0 < M::inf()) ? LR::to_bits(lim0) : kInfBits;
        if ((32 % C) == 0) {
          for (int off = C; off < 32; off <<= 1) {
            const bits_t o2 = __shfl_xor_sync(kFull, lb, off);
            lb = (o2 < lb) ? o2 : lb;
          }
          if (lane < C && lb != kInfBits) atomicMin(&LS_SC(bits_t, kF_TSTAR, c), lb);
        } else if (lb != kInfBits) {
          atomicMin(&LS_SC(bits_t, kF_TSTAR, c), lb);
        }
      }
    }
    if (EST) {
      // second estimator layer: a thread owns output o for a GROUP of CG cells, so a row of weights is read once per group
      // (the hidden activations of a cell are read by broadcast); per output the fmaf chain runs in index order (R18).
      // Dealt from the last thread downwards (the first warps hold the longest lists above).
      constexpr int CG = 4;
      const int H = LS_D(H), n_out = LS_D(n_out);
      const int n_grp = (C + CG - 1) / CG;
      const float *W2p = (const float *)(tbl + LS_L(o_W2p)), *b2 = (const float *)(tbl + LS_L(o_b2));
      for (unsigned it = (unsigned)(kLsThreads - 1 - tid); it < (unsigned)(n_grp * n_out); it += kLsThreads) {
        const unsigned g = it / (unsigned)n_out;
        const unsigned o = it - g * (unsigned)n_out;
        const int c0 = (int)g * CG;
        const float4 *wrow = (const float4 *)(W2p + o * (unsigned)LS_L(Hpad));
        const float bias = b2[o];
        float y[CG];
        const float4 *hid4[CG];
#pragma unroll
        for (int u = 0; u < CG; ++u) {
          y[u] = bias;
          const int cu = (c0 + u < C) ? c0 + u : C - 1;
          hid4[u] = (const float4 *)(cells + LS_L(oHid) + (unsigned)cu * (unsigned)(4 * LS_L(Hs)));
        }
#pragma unroll 2
        for (int q4 = 0; q4 < H / 4; ++q4) {
          const float4 wv = wrow[q4];
#pragma unroll
          for (int u = 0; u < CG; ++u) {
            const float4 hv = hid4[u][q4];
            y[u] = __fmaf_rn(wv.x, hv.x, y[u]);
            y[u] = __fmaf_rn(wv.y, hv.y, y[u]);
            y[u] = __fmaf_rn(wv.z, hv.z, y[u]);
            y[u] = __fmaf_rn(wv.w, hv.w, y[u]);
          }
        }
#pragma unroll
        for (int u = 0; u < CG; ++u) {
          const int c = c0 + u;
          if (c < C) {
            if (o < (unsigned)S) LS_AT(RT, LS_L(oCp), o, c) = (RT)y[u];
            else LS_AT(RT, LS_L(oH), o - S, c) = ((RT)y[u] * (RT)tb.h_ref_T) * LS_SC(RT, kF_INVT, c);
          }
        }
      }
    }
    LST(3)
    __syncthreads();
    LST(5)

    // =========================== phase 4: a3 step size, a4 update, a5 ringing filter, and the scalar chain ===========================
    const int set_next = (sc_set == LS_L(oSc)) ? LS_L(oSc) + LS_L(sc_bytes) : LS_L(oSc);
    const int g_next = (g13 + 1 == kWindow) ? 0 : g13 + 1;
    if (warp == SW) {
      RT inv_wbar = RT(0);
      bool bad_y = false;
      if (my_slot) {
        const RT t_star = LR::from_bits(LS_SC(bits_t, kF_TSTAR, mc));
        RT h = (t_star < dt_max) ? t_star : dt_max;       // Eq 5
        const RT rem = t_f - t;
        bool lst = false;
        if (rem - h < t_tol) {                            // landing on t_f (R5)
          h = rem;
          lst = true;
        }
        // One loop over the species carries the three sequential sums of the step side by side: the temperature
        // equation's sum (Y_i/W_i) cp_i/R and sum (h_i/RT) omega_i (R15), and, behind the update of the mass fractions
        // (Eq 18), 1/Wbar of the new state -- each in species order (contract 5.4).
        // The loop body is branch-free (a slot without a cell stores its mass fractions back unchanged), so the loads
        // of the next species are issued under the fused multiply-adds of this one.
        // The scalar warp gets one issue slot in four while the three filter warps of its scheduler stream their
        // multiply-adds, so what counts here is the number of instructions: a slot without a cell takes a step of
        // length zero (fma(0, dY, y) = y exactly: its dY is finite, or y is already not) instead of a select, and the
        // non-finite test reads the exponent field instead of forming y - y.
        RT sum_cp = RT(0), sum_h = RT(0);
        const RT h_upd = active ? h : RT(0);
        bool bad_any = false;
#pragma unroll 4
        for (int i = 0; i < S; ++i) {
          sum_cp = M::fma(LS_AT(RT, LS_L(oYw), i, mc), LS_AT(RT, LS_L(oCp), i, mc), sum_cp);
          sum_h = M::fma(LS_AT(RT, LS_L(oH), i, mc), LS_AT(RT, LS_L(oOm), i, mc), sum_h);
          const RT y = M::fma(h_upd, LS_AT(RT, LS_L(oConc), 1 + i, mc), LS_AT(RT, LS_L(oY), i, mc));
          ls_sts_unordered(&LS_AT(RT, LS_L(oY), i, mc), y);
          bad_any = bad_any | LR::nonfinite(y);
          inv_wbar = M::fma(y, invW[i], inv_wbar);
        }
        bad_y = active && bad_any;
        asm volatile("" ::: "memory");
        if (EST && LS_D(n_in) > 1) {   // estimator inputs of the new state (R18)
          const float *eshift = (const float *)(tbl + LS_L(o_eshift)), *escale = (const float *)(tbl + LS_L(o_escale));
          float *cXn = (float *)(cells + LS_L(oXn));
#pragma unroll 4
          for (int i = 0; i < S; ++i) cXn[(2 + i) * C + mc] = ((float)LS_AT(RT, LS_L(oY), i, mc) - eshift[2 + i]) * escale[2 + i];
        }
        const RT dTdt = (sc.energy_mode == 0) ? -((sum_h * M::ru()) * T) / (rho * (M::ru() * sum_cp)) : RT(0);
        if (active) {
          T = M::fma(h, dTdt, T);
          bad_T = LR::nonfinite(T);
          t = lst ? t_f : t + h;
          steps += 1;
          last = lst;
        }
      }
      scalar_warp_prepare(set_next, g_next, false, inv_wbar, bad_y);
    } else {
      ls_dft<SH, RT>(a, cells, sc_set, trow, g13, prank, lane, dt_max, t_tol);
    }
    LST(4)
    __syncthreads();
    LST(5)
    sc_set = set_next;
    g13 = g_next;
#ifdef LS_TIMING
    n_steps_ += 1;
#endif
  }
#ifdef LS_TIMING
  if (blockIdx.x == 0 && lane == 0 && (warp == 0 || warp == 7 || warp == SW))
    printf("LST warp %d steps %lld per step: P1 %lld P2 %lld P3 %lld P4 %lld barrier-wait %lld\n", warp, n_steps_, tph[1] / n_steps_,
           tph[2] / n_steps_, tph[3] / n_steps_, tph[4] / n_steps_, tph[5] / n_steps_);
#endif

  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  __syncthreads();
  if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 512;" ::"r"(tmem_base) : "memory");
}

}  // namespace stev
