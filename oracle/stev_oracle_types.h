/*
 * stev_oracle_types.h -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.  The plain structs the oracle's two modes
 * (stev_oracle.c: binary64, stev_oracle_f32.c: binary32) take; nothing under paper_1905_09395_b200/ includes it.
 */
#ifndef STEV_ORACLE_TYPES_H
#define STEV_ORACLE_TYPES_H
#include <stdint.h>

/* ------------------------------------------------------------------------------------------
 * Mechanism, estimator and parameter descriptions (plain structs, host pointers, borrowed).
 * ---------------------------------------------------------------------------------------- */
typedef struct {
  int32_t n_species, n_reactions;
  const double *mol_weight;           /* [S] g/mol */
  const double *nasa_lo, *nasa_hi;    /* [S*7] a1..a7; low range iff T < t_mid (R17) */
  const double *t_mid;                /* [S] */
  const double *A, *b, *Ea;           /* [R] Arrhenius k = A T^b exp(-Ea/(R_cal T)) */
  const uint8_t *reversible;          /* [R] */
  const int32_t *reac_ptr, *reac_species, *reac_nu; /* CSR, integer nu >= 1 */
  const int32_t *prod_ptr, *prod_species, *prod_nu;
  /* Optional (NULL = absent), one value per CSR entry.  PAPER.md:205-229 (BFER): CH4 + 1.5 O2 -> CO + 2 H2O with the
   * rate k C_CH4^0.5 C_O2^0.65 (Eqs 26, 28) and CO + 0.5 O2 <=> CO2 (Eqs 27, 29) need real stoichiometric coefficients
   * and forward orders that differ from them.  coef: stoichiometric coefficient (default (double)nu); order: exponent
   * of the concentration in the rate law (default coef). */
  const double *reac_coef, *prod_coef, *reac_order, *prod_order;
} ora_mechanism;

typedef struct {
  int32_t n_in, n_hidden, n_out;
  int32_t activation;                 /* 0 = tanh, 1 = sigmoid (paper: sigmoid) */
  int32_t input_map;                  /* 0 = (T), 1 = (T, p, Y_0..Y_{S-1}) */
  const float *in_shift, *in_scale;   /* [n_in]  x = (raw - shift) * scale */
  const float *W1, *b1, *W2, *b2;     /* [H*n_in], [H], [n_out*H], [n_out] row-major */
  float h_ref_temperature;            /* outputs: cp_i/R (first S), h_i/(R*h_ref_temperature) (next S) */
} ora_estimator;

typedef struct {
  double y_step_max;   /* Y_step^max, PAPER.md:51 (R3, default 1e-2) */
  double delta_max;    /* delta^max,  PAPER.md:57 (R4, default 1e-2) */
  double alpha;        /* PAPER.md:67 (default 1e-5; 0 => gamma == 1) */
  double tol_ring;     /* PAPER.md:95 (R12, default 0.5) */
  double tol_freq;     /* PAPER.md:95 (R12, default 0.1) */
  double r_fac;        /* PAPER.md:95 (R12, default 2) */
  double rof_min;      /* R13, default 2^-100 */
  int32_t dft_first_high_bin; /* n of Eq 10 (R10, default 4; high bins are n..6) */
  int32_t dft_enable;
  int32_t max_steps;   /* R20 */
  int32_t energy_mode; /* 0 = adiabatic constant pressure (R15), 1 = isothermal */
} ora_params;

#endif
