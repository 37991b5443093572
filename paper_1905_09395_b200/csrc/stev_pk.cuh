// stev_pk.cuh -- types shared by the host and device side of the warp-pair integrator (stev_pk_kernel.cuh).
#pragma once
#include <cstdint>

#include "stev_device.cuh"

namespace stev {

constexpr int kPkMaxCells = 8;       // cells per block with two warps per cell: 2 per TMEM lane quarter x 4 quarters
                                     // (one warp per cell: 16 cells, 4 per quarter)
constexpr int kPkMaxIt = 8;          // 32-blocks of reversible reactions per cell with two warps per cell (32 TMEM columns
                                     // each, 256 columns per cell); 4 with one warp per cell
constexpr int kPkThreads = 64 * kPkMaxCells;   // block size with one or two warps per cell
constexpr int kPkThreads4 = 128 * kPkMaxCells;  // block size of the dense one-warp-per-cell kernel (32 cells, 64 registers per thread)
constexpr int kPkMaxNw = 2;

// Table image of the pair kernel (one contiguous buffer, copied verbatim to shared memory).  Byte offsets.
struct PkTables {
  int nw;                              // warps per cell: 2 (pair): 8 cells per block; 1: 16 cells (dense: 32)
  int S, R, Rrev, n_it, Rp;            // n_it: 32-blocks of reversible reactions; Rp: row length of the q-variant array
  int has_est, H, Hpad, n_in, n_out, act, input_map;
  float h_ref_T;
  int n_var;                           // stored multiples of q: 2 (+q, -q) or 4 (+q, -q, +2q, -2q)
  int g_len4[kPkMaxNw];                // per warp of the cell: rows of four gather entries per lane (longest list, rounded up)
  int g_row0[kPkMaxNw];                // first row of that warp's entries in o_gent
  int it_split[kPkMaxNw + 1];          // DFT blocks [it_split[h], it_split[h + 1]) belong to warp h of the cell
  int o_tmid, o_W, o_invW, o_nasa;     // double [S] each; nasa [2][14][S]
  int o_rkA, o_rkB;                    // double2 [R]: {ln A, b}, {Ea/R_cal, dnu}
  int o_rfac;                          // uint4 [R]: byte offsets (from the cell base) of the two reactant and two
                                       //            product concentration factors (the 1.0 slot if absent)
  int o_rdg;                           // uint4 [Rrev]: byte offsets of nu*g of the <=2 reactant / <=2 product entries
  int o_gsp;                           // uint8 [128]: species whose source term lane l of warp h gathers ([32 h + l]); 255 = none
  int o_glen;                          // uint16 [128]: number of entries of that species' list
  int o_gent;                          // uint4 [sum of g_len4 + 2][32]: byte offsets (from the cell base) of the
                                       //            stored multiples coef*q_j, or of the 0.0 slot (padding)
  int o_eshift, o_escale, o_W1T, o_b1, o_W2p, o_b2;  // float: [n_in],[n_in],[n_in][H],[H],[n_out][Hpad],[n_out]
  int bytes;
};

// Per-cell shared-memory scratch, byte offsets from the cell base (multiples of 16).
struct PkCell {
  int oYp;     // double2 [S]  {Y_i, 1/W_i}
  int oYwCp;   // double2 [S]  {Y_i/W_i, cp_i/R}
  int oHOm;    // double2 [S]  {h_i/RT, omega_i}
  int oConc;   // double [1+S] [0] = 1.0, then C_i**  (later dY_i/dt)
  int oG;      // double [1+2S] [0] = 0.0, then g_i/RT, then 2 g_i/RT
  int oQ;      // double [n_var][Rp]  multiples of the effective progress rates (variant 0 = q_eff itself)
  int oRof;    // double [Rrev]
  int oHid;    // float [H]
  int oSc;     // PkScal
  int stride;
};

// Scalars the two warps of a pair hand to each other (each field has one writer per step, read after a pair barrier).
struct PkScal {
  double lnT, ln_c0, invT, inv_ctot, rho;
  double t_star[kPkMaxNw];
  double T_new;
  int bad[kPkMaxNw];
  int pos;
  int pad;
};

struct PkArgs {
  PkTables tb;
  const unsigned char *table;
  PkCell cl;
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
  int cells_per_block;
};

}  // namespace stev
