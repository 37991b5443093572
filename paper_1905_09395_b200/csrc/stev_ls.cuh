// stev_ls.cuh -- types shared by the host and device side of the lock-step integrator (stev_ls_kernel.cuh).
//
// One block per SM holds C cells that advance in LOCK STEP: every step of the method costs the same work whatever the
// state (all reactions, all DFT windows), so cells that step together never diverge; what differs between cells is the
// NUMBER of steps, and a slot whose cell has landed on t_f is refilled from the global queue.  Stepping
// together lets the block flatten its work over (cell, reaction) and (cell, species) pairs, so no lane idles because a
// mechanism does not fill a multiple of 32 lanes, and lets ONE warp evaluate the scalar chains (logarithms, divisions,
// the sequential species sums of the arithmetic contract) of all C cells at once, one cell per lane.
//
// Every size and byte offset of the kernel follows from LsDims through ONE constexpr function (ls_layout_of) that the host
// uses to build the table image and the kernel uses to address it.  The kernel is instantiated once with the dimensions
// read at run time (any mechanism) and once per entry of the shape list in stev_ls.cu with the dimensions as compile-time
// constants (offsets become immediates, item loops unroll, divisions by S / R_rev / C become multiplications).
#pragma once
#include <cstdint>

#include "stev_device.cuh"

namespace stev {

constexpr int kLsThreads = 512;                 // 16 warps; warp w reaches TMEM lane quarter w % 4
constexpr int kLsWarps = kLsThreads / 32;
constexpr int kLsPassWarps = kLsWarps - 1;      // the last warp is the scalar warp: it owns no reversible (reaction, cell) passes; pass p belongs to warp p % 15
// A warp owns 128 tensor-memory columns of its lane quarter (4 warps per quarter x 128 = 512): four 32-column slots of
// thirteen doubles, or eight 16-column slots of thirteen floats (stev_params.state_precision = STEV_STATE_FP32).
__host__ __device__ constexpr int ls_slot_pitch(int es) { return es == 8 ? 32 : 16; }
__host__ __device__ constexpr int ls_slots(int es) { return 128 / ls_slot_pitch(es); }
__host__ __device__ constexpr int ls_max_passes(int es) { return kLsPassWarps * ls_slots(es); }   // 60 (1920 windows) / 120 (3840)
constexpr int kLsMaxCells = 32;                 // one lane of the scalar warp per cell

// Scalars of the cell slots, one array of C eight-byte entries per field (entry (f, c) at set + (f C + c) 8).  There are
// TWO sets, used by alternate steps: while the block still reads the set of step n (update, ringing filter), the scalar
// warp already writes the set of step n + 1.  Written by the cell's lane of the scalar warp unless stated.
enum LsField {
  kF_T, kF_P,                          // state of the step
  kF_LNT, kF_LNC0, kF_INVT, kF_ICTOT, kF_RHO, kF_INVRHO,
  kF_REM,                              // t_f - t before the step
  kF_TSTAR,                            // u64: running minimum of the limiter (atomicMin of the bit patterns, phase 3)
  kF_ACTIVE,                           // int: 1 the slot integrates a cell; 0 it waits for a refill (or the queue is empty)
  kF_FRESH,                            // int: 1 during the first step of a new cell: window owners zero the history, rOF = 1
  kF_COUNT
};

struct LsDims {
  int S, R, Rrev;
  int n_var;                           // stored multiples of q: 2 (+q, -q) or 4 (+q, -q, +2q, -2q)
  int has_est, H, n_in, n_out;
  int C;                               // cell slots per block
  int es;                              // bytes per real: 8 (binary64 state) or 4 (binary32 state)
};

// Byte offsets; "real" is double or float (LsDims.es bytes).  The working set of the block's C cells is stored INDEX-MAJOR,
// CELL-MINOR: element (idx, c) of a real array at offset o sits at o + (idx C + c) es, so that lanes holding consecutive cells of the same species / reaction read
// consecutive addresses (and the per-reaction tables are read by broadcast).  From the start of the cell region:
//   oY [S] | oYw [S] Y_i/W_i | oCp [S] cp_i/R | oH [S] h_i/RT | oOm [S] omega_i
//   oConc [1+S] ([0] = 1.0, then C_i**, later dY_i/dt) | oG [1+2S] ([0] = 0.0, g_i/RT, 2 g_i/RT)
//   oQ [n_var][Rp] multiples of q_eff | oRof [Rrev] | oSc [2][kF_COUNT] the two sets of scalars
//   oHid float [C][Hs] hidden activations, cell-major with Hs = H + 4 | oXn float [n_in][C] normalised estimator inputs
// Table image (from the image base):
//   o_tmid, o_W, o_invW real [S] | o_nasa real [2][14][S] | o_rkA real2 [R] {ln A, b} | o_rkB real2 [R] {Ea/R_cal, dnu}
//   o_rfac uint4 [R] offsets (from the cell region, for cell 0) of the two reactant and two product concentration factors
//          (the 1.0 slot if absent); top bit of .w: the reaction has a coefficient of 2, its doubled multiples are read
//   o_rdg uint4 [Rrev] offsets of nu*g of the <= 2 reactant / <= 2 product entries (0.0 slot if absent)
//   o_gsp uint8 [S] species with the r-th longest source-term list | o_grow, o_glen uint16 [S] first row / rows of that list
//   o_eshift, o_escale float [n_in] | o_W1T float [n_in][H] | o_b1 float [H] | o_W2p float [n_out][Hpad] | o_b2 float [n_out]
//   o_gent uint4 [rows + 1] (LAST: its length depends on the mechanism's lists) offsets of the stored multiples coef*q_j in
//          the caller's reaction order, padded with the 0.0 slot; the last row is all padding
struct LsLayout {
  int Rp, Hpad, Hs;
  int oY, oYw, oCp, oH, oOm, oConc, oG, oQ, oRof, oSc, sc_bytes, oHid, oXn, cell_bytes;
  int o_tmid, o_W, o_invW, o_nasa, o_rkA, o_rkB, o_rfac, o_rdg, o_gsp, o_grow, o_glen;
  int o_eshift, o_escale, o_W1T, o_b1, o_W2p, o_b2, o_gent;
  int n_rev_pass, n_irr_pass;          // warp passes over the flattened (reversible reaction, cell) / (irreversible, cell) pairs
};

__host__ __device__ constexpr int ls_align(int x, int a) { return (x + a - 1) / a * a; }

__host__ __device__ constexpr LsLayout ls_layout_of(const LsDims &d) {
  LsLayout L{};
  L.Rp = (d.R + 1) & ~1;
  L.Hpad = d.H + 4;
  L.Hs = d.H + 4;
  const int C = d.C, es = d.es;
  int o = 0;
  L.oY = o; o = ls_align(o + es * C * d.S, 16);
  L.oYw = o; o = ls_align(o + es * C * d.S, 16);
  L.oCp = o; o = ls_align(o + es * C * d.S, 16);
  L.oH = o; o = ls_align(o + es * C * d.S, 16);
  L.oOm = o; o = ls_align(o + es * C * d.S, 16);
  L.oConc = o; o = ls_align(o + es * C * (1 + d.S), 16);
  L.oG = o; o = ls_align(o + es * C * (1 + 2 * d.S), 16);
  L.oQ = o; o = ls_align(o + es * C * d.n_var * L.Rp, 16);
  L.oRof = o; o = ls_align(o + es * C * (d.Rrev > 0 ? d.Rrev : 1), 16);
  L.oSc = o; o = ls_align(o + 2 * 8 * C * (int)kF_COUNT, 16);
  L.sc_bytes = 8 * C * (int)kF_COUNT;
  L.oHid = o; o = ls_align(o + 4 * C * (d.has_est ? L.Hs : 0), 16);
  L.oXn = o; o = ls_align(o + 4 * C * (d.has_est ? d.n_in : 0), 16);
  L.cell_bytes = o;
  int t = 0;
  L.o_tmid = t; t = ls_align(t + es * d.S, 16);
  L.o_W = t; t = ls_align(t + es * d.S, 16);
  L.o_invW = t; t = ls_align(t + es * d.S, 16);
  L.o_nasa = t; t = ls_align(t + es * 2 * kNasaRows * d.S, 16);
  L.o_rkA = t; t = ls_align(t + 2 * es * d.R, 16);
  L.o_rkB = t; t = ls_align(t + 2 * es * d.R, 16);
  L.o_rfac = t; t = ls_align(t + 16 * d.R, 16);
  L.o_rdg = t; t = ls_align(t + 16 * (d.Rrev > 0 ? d.Rrev : 1), 16);
  L.o_gsp = t; t = ls_align(t + d.S, 16);
  L.o_grow = t; t = ls_align(t + 2 * d.S, 16);
  L.o_glen = t; t = ls_align(t + 2 * d.S, 16);
  L.o_eshift = t; t = ls_align(t + 4 * d.n_in, 16);
  L.o_escale = t; t = ls_align(t + 4 * d.n_in, 16);
  L.o_W1T = t; t = ls_align(t + 4 * d.n_in * d.H, 16);
  L.o_b1 = t; t = ls_align(t + 4 * d.H, 16);
  L.o_W2p = t; t = ls_align(t + 4 * d.n_out * L.Hpad, 16);
  L.o_b2 = t; t = ls_align(t + 4 * d.n_out, 16);
  L.o_gent = t;
  L.n_rev_pass = (C * d.Rrev + 31) / 32;
  L.n_irr_pass = (C * (d.R - d.Rrev) + 31) / 32;
  return L;
}

// What the host keeps per (mechanism, estimator): the dimensions, the image size and the few values that are not sizes.
struct LsTables {
  LsDims d;
  int act, input_map;
  float h_ref_T;
  int g_zero_row;                      // index of the all-padding row of o_gent
  // passes over the (irreversible reaction, cell) pairs of the warp of rank r: irr_start[r] .. + irr_count[r]; dealt on the
  // host so that every warp carries about the same rate work (the scalar warp, which owns no reversible passes, the most)
  unsigned char irr_start[16], irr_count[16];
  int bytes;                           // image size
};

struct LsArgs {
  LsTables tb;
  LsLayout lay;                        // ls_layout_of(tb.d)
  unsigned mC;                         // ceil(2^32 / C) for the run-time shape: x / C = umulhi(x, mC) (0 for C = 1)
  const unsigned char *table;
  SolverConsts sc;
  double t_f;
  long long n_active;
  const int *list;
  long long ld;
  double *T;
  const double *p;
  double *Y;
  int *steps;
  unsigned char *status;
  int *queue_head;
  int *worst_status;
};

// Dimensions known at compile time (an entry of the shape list) or read from the arguments.
struct LsDyn {
  static constexpr bool kStatic = false;
  static constexpr LsDims D{};
};
template <int S_, int R_, int RREV_, int NVAR_, int EST_, int H_, int NIN_, int NOUT_, int C_, int ES_ = 8>
struct LsFix {
  static constexpr bool kStatic = true;
  static constexpr LsDims D{S_, R_, RREV_, NVAR_, EST_, H_, NIN_, NOUT_, C_, ES_};
};

}  // namespace stev
