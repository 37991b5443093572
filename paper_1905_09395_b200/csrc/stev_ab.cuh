// stev_ab.cuh -- types shared by the host and device side of the warp-specialised integrator (stev_ab_kernel.cuh).
#pragma once
#include <cstdint>

#include "stev_device.cuh"

namespace stev {

constexpr int kAbMaxCells = 8;       // cells per block: 2 per TMEM lane quarter x 4 quarters
constexpr int kAbMaxIt = 8;          // reversible reactions per lane (32 TMEM columns each, 256 columns per cell)
constexpr int kAbThreads = 64 * kAbMaxCells;

// Table image of the AB kernel (one contiguous buffer, copied verbatim to shared memory).  Byte offsets.
struct AbTables {
  int S, R, Rrev, n_it, Rp;            // Rp: row length of the q-variant array (R rounded up to even)
  int has_est, H, Hpad, n_in, n_out, act, input_map;
  float h_ref_T;
  int n_var;                           // stored multiples of q: 2 (+q, -q) or 4 (+q, -q, +2q, -2q)
  int g_len[2];                        // padded entries per lane in gather round 0 / 1 (species lane, lane + 32)
  int o_tmid, o_W, o_invW, o_nasa;     // double [S] each; nasa [2][14][S]
  int o_rkA, o_rkB;                    // double2 [R]: {ln A, b}, {Ea/R_cal, dnu}
  int o_rfac;                          // uint4 [R]: byte offsets (from the cell base) of the two reactant and two
                                       //            product concentration factors (the 1.0 slot if absent)
  int o_rdg;                           // uint4 [Rrev]: byte offsets of nu*g of the <=2 reactant / <=2 product entries
  int o_gsp;                           // uint8 [64]: species handled by lane l in round 0 ([l]) and round 1 ([32+l]); 255 = none
  int o_gent;                          // uint16 [(g_len[0]+g_len[1])][32]: byte offsets (from the cell base) of the
                                       //            stored multiple coef*q_j, or of the 0.0 slot (padding)
  int o_eshift, o_escale, o_W1T, o_b1, o_W2p, o_b2;  // float: [n_in],[n_in],[n_in][H],[H],[n_out][Hpad],[n_out]
  int bytes;
};

// Per-cell shared-memory scratch, byte offsets from the cell base (multiples of 16).
struct AbCell {
  int oYp;     // double2 [S]  {Y_i, 1/W_i}
  int oYwCp;   // double2 [S]  {Y_i/W_i, cp_i/R}
  int oHOm;    // double2 [S]  {h_i/RT, omega_i}
  int oConc;   // double [1+S] [0] = 1.0, then C_i**  (later dY_i/dt)
  int oG;      // double [1+2S] [0] = 0.0, then g_i/RT, then 2 g_i/RT
  int oQ;      // double [n_var][Rp]  multiples of the effective progress rates (variant 0 = q_eff itself)
  int oQraw;   // double [R]  raw progress rates of the step being prepared (the DFT warp still reads oQ)
  int oRof;    // double [Rrev]
  int oHid;    // float [H]
  int oCtrl;   // AbCtrl
  int stride;
};

struct AbCtrl {
  double h, inv_ctot;
  int cmd;
  int pad;
};
enum { kCmdStep = 0, kCmdFinal = 1, kCmdExit = 2 };

struct AbArgs {
  AbTables tb;
  const unsigned char *table;
  AbCell cl;
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
