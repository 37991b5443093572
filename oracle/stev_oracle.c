/*
 * stev_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * A plain, slow, fp64 CPU implementation of the STEV integrator (Buchheit et al.,
 * arxiv 1905.09395), written step by step from /root/reference/PAPER.md in the paper's
 * order and notation.  It is the oracle the CUDA path is checked against.  Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may load it.
 * It shares no code, header, table generator or helper with paper_1905_09395_b200/.
 *
 * Citations are "PAPER.md:LINE (section / equation)".  Where the paper is silent the reading
 * "R<n>" of DESIGN.md section 3 is taken (the same numbering as SURVEY.md section 8c).
 *
 * Parity status: the paper prints no value of any solver quantity, so parity WITH THE PAPER is
 * unpinned; every function below is pinned by closed forms, invariants, library routines or
 * brute force in tests/test_oracle_*.py (pins P1..P12 of DESIGN.md section 4).
 *
 * Arithmetic: DESIGN.md section 5 ("arithmetic contract").  STEV trajectories on stiff
 * mechanisms amplify one-ulp differences, so every floating-point operation below is written
 * out: `fma(a,b,c)` where the contract says fused, plain `*`/`+` elsewhere, sums sequential in
 * index order, exp/log from the two routines at the top of this file (built from fma, *, +, /
 * and bit operations only).  Compile with -ffp-contract=off.
 *
 * Units: cgs-mol (R21): concentrations mol/cm^3, p dyn/cm^2, Ea cal/mol.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define ORA_RU 8.31446261815324e7   /* erg/(mol K)  (R21) */
#define ORA_RCAL 1.98720425864083   /* cal/(mol K)  (R21) */
#define ORA_PATM 1.01325e6          /* dyn/cm^2     (R21) */
#define ORA_WINDOW 13               /* "thirteen most recent changes" */

/* When the host has FMA hardware gcc inlines fma(); otherwise libm's (exact) fma is called. */
#if defined(__x86_64__)
#define ORA_CLONES __attribute__((target_clones("fma", "default")))
#else
#define ORA_CLONES
#endif

#include "stev_oracle_types.h"

/* ------------------------------------------------------------------------------------------
 * Contract exp / log.
 * ---------------------------------------------------------------------------------------- */
static inline uint64_t ora_bits(double x) { uint64_t u; memcpy(&u, &x, 8); return u; }
static inline double ora_from_bits(uint64_t u) { double x; memcpy(&x, &u, 8); return x; }

/* exp(x): k = round(x*log2 e) by the 1.5*2^52 shift, r = x - k ln2 in two fma steps, Taylor
 * polynomial of degree 13 in Horner form, scaling by 2^k through the exponent field.
 * x > 709 gives +inf, x < -708 gives 0 (no subnormal results), NaN propagates. */
ORA_CLONES
double ora_exp(double x) {
  if (x != x) return x;
  if (x > 709.0) return INFINITY;
  if (x < -708.0) return 0.0;
  const double shift = 6755399441055744.0; /* 1.5 * 2^52 */
  double t = fma(x, 1.4426950408889634, shift);
  double k = t - shift;
  int32_t ki = (int32_t)(uint32_t)(ora_bits(t) & 0xffffffffu);
  double r = fma(-k, 6.93147180369123816490e-01, x);
  r = fma(-k, 1.90821492927058770002e-10, r);
  double p = 1.6059043836821613e-10;          /* 1/13! */
  p = fma(p, r, 2.08767569878681e-09);        /* 1/12! */
  p = fma(p, r, 2.505210838544172e-08);       /* 1/11! */
  p = fma(p, r, 2.755731922398589e-07);       /* 1/10! */
  p = fma(p, r, 2.7557319223985893e-06);      /* 1/9!  */
  p = fma(p, r, 2.48015873015873e-05);        /* 1/8!  */
  p = fma(p, r, 0.0001984126984126984);       /* 1/7!  */
  p = fma(p, r, 0.001388888888888889);        /* 1/6!  */
  p = fma(p, r, 0.008333333333333333);        /* 1/5!  */
  p = fma(p, r, 0.041666666666666664);        /* 1/4!  */
  p = fma(p, r, 0.16666666666666666);         /* 1/3!  */
  p = fma(p, r, 0.5);
  p = fma(p, r, 1.0);
  p = fma(p, r, 1.0);
  double two_k = ora_from_bits((uint64_t)(int64_t)(ki + 1023) << 52);
#ifdef ORA_SENSITIVITY_ULP
  /* Self-sensitivity variant (SURVEY.md section 8c "Arithmetic contract"): built ONLY into
   * libstev_oracle_ulp.so by tests/test_oracle_sensitivity.py.  It moves the result by one unit in the last place,
   * up or down by a hash of the argument's bits, i.e. it is another routine that is still within 2 ulp of libm. */
  {
    uint64_t hsh = ora_bits(x) * 0x9e3779b97f4a7c15ULL;
    uint64_t rb = ora_bits(p * two_k);
    if (rb > 0x0010000000000000ULL && rb < 0x7fe0000000000000ULL) return ora_from_bits((hsh >> 63) ? rb + 1 : rb - 1);
  }
#endif
  return p * two_k;
}

/* log(x) for positive normal x: x = m 2^e with m in (sqrt(1/2), sqrt 2], f = (m-1)/(m+1),
 * log m = 2f (1 + s/3 + s^2/5 + ... + s^11/23), s = f^2.  x <= 0, NaN, inf, subnormal: as libm
 * would only in the sense of sign/NaN (these never occur on the path; see tests). */
ORA_CLONES
double ora_log(double x) {
  if (x != x || x < 0.0) return NAN;
  if (x == 0.0) return -INFINITY;
  if (x == INFINITY) return x;
  uint64_t u = ora_bits(x);
  int32_t e = (int32_t)(u >> 52) - 1023;
  double m = ora_from_bits((u & 0x000fffffffffffffULL) | 0x3ff0000000000000ULL);
  if (m > 1.4142135623730951) { m = m * 0.5; e = e + 1; }
  double f = (m - 1.0) / (m + 1.0);
  double s = f * f;
  double P = 0.043478260869565216;            /* 1/23 */
  P = fma(P, s, 0.047619047619047616);        /* 1/21 */
  P = fma(P, s, 0.05263157894736842);         /* 1/19 */
  P = fma(P, s, 0.058823529411764705);        /* 1/17 */
  P = fma(P, s, 0.06666666666666667);         /* 1/15 */
  P = fma(P, s, 0.07692307692307693);         /* 1/13 */
  P = fma(P, s, 0.09090909090909091);         /* 1/11 */
  P = fma(P, s, 0.1111111111111111);          /* 1/9  */
  P = fma(P, s, 0.14285714285714285);         /* 1/7  */
  P = fma(P, s, 0.2);                         /* 1/5  */
  P = fma(P, s, 0.3333333333333333);          /* 1/3  */
  double two_f = f + f;
  double log_m = fma(two_f, s * P, two_f);
  double ed = (double)e;
  return fma(ed, 6.93147180369123816490e-01, fma(ed, 1.90821492927058770002e-10, log_m));
}

/* ------------------------------------------------------------------------------------------
 * NASA-7 thermodynamics, PAPER.md:113-120 (Eqs 15, 16) + standard entropy (R17).
 * cp/R  = a1 + a2 T + a3 T^2 + a4 T^3 + a5 T^4                              (Eq 15)
 * h/RT  = a1 + a2 T/2 + a3 T^2/3 + a4 T^3/4 + a5 T^4/5 + a6/T               (Eq 16)
 * s/R   = a1 ln T + a2 T + a3 T^2/2 + a4 T^3/3 + a5 T^4/4 + a7              (R17)
 * Polynomials in Horner form; the divided coefficients a_k/n are formed by IEEE division.
 * ---------------------------------------------------------------------------------------- */
ORA_CLONES
void ora_nasa7(const double *a, double T, double lnT, double invT, double *cpR, double *hRT, double *sR) {
  *cpR = fma(fma(fma(fma(a[4], T, a[3]), T, a[2]), T, a[1]), T, a[0]);
  double hp = fma(fma(fma(fma(a[4] / 5.0, T, a[3] / 4.0), T, a[2] / 3.0), T, a[1] / 2.0), T, a[0]);
  *hRT = fma(a[5], invT, hp);
  double sp = fma(fma(fma(a[4] / 4.0, T, a[3] / 3.0), T, a[2] / 2.0), T, a[1]);
  *sR = fma(a[0], lnT, fma(sp, T, a[6]));
}

/* Species thermo at one temperature: range select "evaluated logically". */
void ora_thermo(const ora_mechanism *m, double T, double *cpR, double *hRT, double *sR) {
  double lnT = ora_log(T), invT = 1.0 / T;
  for (int i = 0; i < m->n_species; ++i) {
    const double *a = (T < m->t_mid[i]) ? m->nasa_lo + 7 * i : m->nasa_hi + 7 * i;
    ora_nasa7(a, T, lnT, invT, &cpR[i], &hRT[i], &sR[i]);
  }
}

/* ------------------------------------------------------------------------------------------
 * Shallow MLP property estimator, PAPER.md:120-136 (Fig 2): one hidden layer, linear output.
 * fp32 weights, fp32 fmaf accumulation in index order, activation through the contract exp in
 * fp64 then rounded to fp32 (R18).  raw[] are the fp64 inputs (T) or (T, p, Y...).
 * ---------------------------------------------------------------------------------------- */
ORA_CLONES
void ora_mlp_forward(const ora_estimator *e, const double *raw, float *hidden, float *out) {
  float x[64];
  for (int k = 0; k < e->n_in; ++k) x[k] = ((float)raw[k] - e->in_shift[k]) * e->in_scale[k];
  for (int j = 0; j < e->n_hidden; ++j) {
    float z = e->b1[j];
    for (int k = 0; k < e->n_in; ++k) z = fmaf(e->W1[j * e->n_in + k], x[k], z);
    double zd = (double)z;
    if (e->activation == 0) hidden[j] = (float)(1.0 - 2.0 / (1.0 + ora_exp(2.0 * zd))); /* tanh */
    else hidden[j] = (float)(1.0 / (1.0 + ora_exp(-zd)));                               /* sigmoid */
  }
  for (int o = 0; o < e->n_out; ++o) {
    float y = e->b2[o];
    for (int j = 0; j < e->n_hidden; ++j) y = fmaf(e->W2[o * e->n_hidden + j], hidden[j], y);
    out[o] = y;
  }
}

/* Batched forward pass for the estimator tests: X [n][n_in] float (already normalised inputs are
 * NOT assumed: X holds raw inputs as float), out [n][n_out]. */
void ora_estimator_eval(const ora_estimator *e, int64_t n, const float *X, float *out) {
  float hidden[256];
  double raw[64];
  for (int64_t c = 0; c < n; ++c) {
    for (int k = 0; k < e->n_in; ++k) raw[k] = (double)X[c * e->n_in + k];
    ora_mlp_forward(e, raw, hidden, out + c * e->n_out);
  }
}

/* ------------------------------------------------------------------------------------------
 * DFT magnitudes of the 13-sample window, PAPER.md:77-81 (Eq 9).  Direct sums in physical slot
 * order with the twiddle table of DESIGN.md section 5.6 (cos, sin of 2 pi n / 13).
 * D[0] = |sum|, D[m] = |sum_k ring[k] exp(-2 pi i m k / 13)| for m = 1..6 (bins 7..12 mirror).
 * ---------------------------------------------------------------------------------------- */
static const double ORA_COS13[13] = {
    1.0, 0.8854560256532099, 0.5680647467311559, 0.120536680255323, -0.35460488704253545,
    -0.7485107481711012, -0.970941817426052, -0.9709418174260521, -0.7485107481711013,
    -0.3546048870425359, 0.1205366802553232, 0.5680647467311548, 0.88545602565321};
static const double ORA_SIN13[13] = {
    0.0, 0.4647231720437685, 0.8229838658936564, 0.992708874098054, 0.9350162426854148,
    0.6631226582407952, 0.23931566428755768, -0.23931566428755743, -0.663122658240795,
    -0.9350162426854147, -0.992708874098054, -0.822983865893657, -0.4647231720437684};

ORA_CLONES
double ora_dft_bin(const double *ring, int m) {
  if (m == 0) {
    double s = 0.0;
    for (int k = 0; k < ORA_WINDOW; ++k) s = s + ring[k];
    return fabs(s);
  }
  double re = 0.0, im = 0.0;
  for (int k = 0; k < ORA_WINDOW; ++k) {
    int n = (m * k) % ORA_WINDOW;
    re = fma(ring[k], ORA_COS13[n], re);
    im = fma(ring[k], -ORA_SIN13[n], im);
  }
  return sqrt(fma(re, re, im * im));
}

void ora_dft_mag(const double *ring, double *D /*[7]*/) {
  for (int m = 0; m <= 6; ++m) D[m] = ora_dft_bin(ring, m);
}

/* Stoichiometric coefficient and rate-law exponent of CSR entry e (Eqs 28-29; R22). */
static inline double ora_coef(const double *coef, const int32_t *nu, int e) { return coef ? coef[e] : (double)nu[e]; }
static inline double ora_order(const double *order, const double *coef, const int32_t *nu, int e) {
  return order ? order[e] : ora_coef(coef, nu, e);
}

/* f * C^x.  x = 1, 2, 3 by repeated multiplication (contract 5.5, the mass-action case); x = 0 leaves f; any other
 * exponent (Eq 28: C^0.5, C^0.65) as exp(x log C), with C^x = 0 for C <= 0 (R22: the stabilised concentration is
 * never negative, and a vanished reactant stops the reaction). */
ORA_CLONES
static double ora_times_power(double f, double c, double x) {
  if (x == 1.0) return f * c;
  if (x == 2.0) return (f * c) * c;
  if (x == 3.0) return ((f * c) * c) * c;
  if (x == 0.0) return f;
  return f * ((c > 0.0) ? ora_exp(x * ora_log(c)) : 0.0);
}

/* ------------------------------------------------------------------------------------------
 * One evaluation of the right-hand side for one cell: steps 1-5 of DESIGN.md section 2.
 * Scratch arrays are caller-provided (length S or R).
 * ---------------------------------------------------------------------------------------- */
typedef struct {
  double *cpR, *hRT, *gRT, *conc, *q, *omega, *r; /* [S],[S],[S],[S],[R],[S],[S] */
  double rho, c_tot, dTdt;
  /* loop invariants, formed once per call by ora_rhs_alloc: ln A_j, Ea_j/R_cal, 1/W_i */
  double *ln_A, *T_a, *inv_W;
  double *rOF, *ring;                              /* [R], [R][13] */
  double *base;
} ora_rhs;

static void ora_rhs_alloc(const ora_mechanism *m, ora_rhs *w) {
  const int S = m->n_species, R = m->n_reactions;
  double *b = (double *)calloc((size_t)(7 * S + 4 * R + R * ORA_WINDOW), sizeof(double));
  w->base = b;
  w->cpR = b; w->hRT = b + S; w->gRT = b + 2 * S; w->conc = b + 3 * S; w->omega = b + 4 * S; w->r = b + 5 * S;
  w->inv_W = b + 6 * S;
  w->q = b + 7 * S; w->ln_A = w->q + R; w->T_a = w->q + 2 * R; w->rOF = w->q + 3 * R; w->ring = w->q + 4 * R;
  for (int i = 0; i < S; ++i) w->inv_W[i] = 1.0 / m->mol_weight[i];
  for (int j = 0; j < R; ++j) { w->ln_A[j] = ora_log(m->A[j]); w->T_a[j] = m->Ea[j] / ORA_RCAL; }
}

ORA_CLONES
static void ora_rhs_eval(const ora_mechanism *m, const ora_estimator *est, const ora_params *prm,
                         double T, double p, const double *Y, int64_t ldy, const double *rOF, ora_rhs *w) {
  const int S = m->n_species, R = m->n_reactions;

  /* 1. thermo.  g/RT always from NASA-7; cp, h from the MLP if attached (R18). */
  double lnT = ora_log(T), invT = 1.0 / T;
  for (int i = 0; i < S; ++i) {
    const double *a = (T < m->t_mid[i]) ? m->nasa_lo + 7 * i : m->nasa_hi + 7 * i;
    double sR;
    ora_nasa7(a, T, lnT, invT, &w->cpR[i], &w->hRT[i], &sR);
    w->gRT[i] = w->hRT[i] - sR;
  }
  if (est) {
    float hidden[256], out[512];
    double raw[64];
    raw[0] = T;
    if (est->input_map == 1) {
      raw[1] = p;
      for (int i = 0; i < S; ++i) raw[2 + i] = Y[i * ldy];
    }
    ora_mlp_forward(est, raw, hidden, out);
    for (int i = 0; i < S; ++i) {
      w->cpR[i] = (double)out[i];
      w->hRT[i] = ((double)out[S + i] * (double)est->h_ref_temperature) * invT;
    }
  }

  /* 2. mixture: 1/Wbar = sum Y_i/W_i, C_tot = p/(R_u T), rho = C_tot * Wbar;
   *    small-species stabilisation gamma(y) = y/(alpha+y), y** = gamma y (Eqs 6-7, R7). */
  double inv_wbar = 0.0;
  for (int i = 0; i < S; ++i) inv_wbar = fma(Y[i * ldy], w->inv_W[i], inv_wbar);
  double c_tot = p / (ORA_RU * T);
  double rho = c_tot / inv_wbar;
  for (int i = 0; i < S; ++i) {
    double yp = Y[i * ldy] > 0.0 ? Y[i * ldy] : 0.0;
    double c = (rho * yp) * w->inv_W[i];
    if (prm->alpha > 0.0) c = (yp / (prm->alpha + yp)) * c;
    w->conc[i] = c;
  }

  /* 3.-4. rate constants and progress rates, PAPER.md:212-218 (Eqs 28-30):
   *    k_f = A T^b exp(-Ea/(R_cal T)), K_c = (p_atm/(R_u T))^dnu exp(-dG/RT), k_r = k_f / K_c,
   *    q = k_f prod C_reac^nu' - k_r prod C_prod^nu'' ; q_eff = q * rOF (Eq 14). */
  double ln_c0 = ora_log(ORA_PATM / (ORA_RU * T));
  for (int j = 0; j < R; ++j) {
    double ln_kf = fma(-w->T_a[j], invT, fma(m->b[j], lnT, w->ln_A[j]));
    double fwd = ora_exp(ln_kf);
    for (int e = m->reac_ptr[j]; e < m->reac_ptr[j + 1]; ++e)
      fwd = ora_times_power(fwd, w->conc[m->reac_species[e]], ora_order(m->reac_order, m->reac_coef, m->reac_nu, e));
    double qj = fwd;
    if (m->reversible[j]) {
      double dg = 0.0, dnu = 0.0;
      for (int e = m->reac_ptr[j]; e < m->reac_ptr[j + 1]; ++e) {
        dg = dg - ora_coef(m->reac_coef, m->reac_nu, e) * w->gRT[m->reac_species[e]];
        dnu = dnu - ora_coef(m->reac_coef, m->reac_nu, e);
      }
      for (int e = m->prod_ptr[j]; e < m->prod_ptr[j + 1]; ++e) {
        dg = dg + ora_coef(m->prod_coef, m->prod_nu, e) * w->gRT[m->prod_species[e]];
        dnu = dnu + ora_coef(m->prod_coef, m->prod_nu, e);
      }
      double ln_kc = fma(dnu, ln_c0, -dg);
      double rev = ora_exp(ln_kf - ln_kc);
      for (int e = m->prod_ptr[j]; e < m->prod_ptr[j + 1]; ++e)
        rev = ora_times_power(rev, w->conc[m->prod_species[e]], ora_order(m->prod_order, m->prod_coef, m->prod_nu, e));
      qj = (fwd - rev) * (rOF ? rOF[j] : 1.0);
    }
    w->q[j] = qj;
  }

  /* 5. source terms: omega_i = sum_j dnu_ij q_j (reaction order, reactants then products),
   *    r_i = dY_i/dt = W_i omega_i / rho,
   *    dT/dt = -(sum_i h_i omega_i) / (rho c_p), h_i = (h/RT)_i R_u T, c_p = R_u sum_i Y_i (cp/R)_i / W_i (R15). */
  for (int i = 0; i < S; ++i) w->omega[i] = 0.0;
  for (int j = 0; j < R; ++j) {
    for (int e = m->reac_ptr[j]; e < m->reac_ptr[j + 1]; ++e)
      w->omega[m->reac_species[e]] = w->omega[m->reac_species[e]] - ora_coef(m->reac_coef, m->reac_nu, e) * w->q[j];
    for (int e = m->prod_ptr[j]; e < m->prod_ptr[j + 1]; ++e)
      w->omega[m->prod_species[e]] = w->omega[m->prod_species[e]] + ora_coef(m->prod_coef, m->prod_nu, e) * w->q[j];
  }
  double inv_rho = 1.0 / rho;
  double sum_h = 0.0, sum_cp = 0.0;
  for (int i = 0; i < S; ++i) {
    w->r[i] = (m->mol_weight[i] * w->omega[i]) * inv_rho;
    sum_h = fma(w->hRT[i], w->omega[i], sum_h);
    sum_cp = fma(Y[i * ldy] * w->inv_W[i], w->cpR[i], sum_cp);
  }
  w->dTdt = (prm->energy_mode == 0) ? -((sum_h * ORA_RU) * T) / (rho * (ORA_RU * sum_cp)) : 0.0;
  w->rho = rho;
  w->c_tot = c_tot;
}

/* Test export: right-hand side of n cells (rOF may be NULL = ones). Y is species-major [S][ld]. */
int ora_rates_eval(const ora_mechanism *m, const ora_estimator *est, const ora_params *prm, int64_t n,
                   int64_t ld, const double *T, const double *p, const double *Y, const double *rOF /*[R][ld]*/,
                   double *dYdt /*[S][ld]*/, double *dTdt /*[n]*/, double *q /*[R][ld]*/) {
  const int S = m->n_species, R = m->n_reactions;
  ora_rhs w;
  ora_rhs_alloc(m, &w);
  double *rof = w.rOF;
  for (int64_t c = 0; c < n; ++c) {
    if (rOF) for (int j = 0; j < R; ++j) rof[j] = rOF[j * ld + c];
    ora_rhs_eval(m, est, prm, T[c], p[c], Y + c, ld, rOF ? rof : NULL, &w);
    for (int i = 0; i < S; ++i) dYdt[i * ld + c] = w.r[i];
    for (int j = 0; j < R; ++j) q[j * ld + c] = w.q[j];
    dTdt[c] = w.dTdt;
  }
  free(w.base);
  return 0;
}

/* ------------------------------------------------------------------------------------------
 * The STEV loop for one cell (steps 1-9).  If `trace` is non-NULL, row n of
 * the trace receives, after step n: t, h, T, Y[0..S), rOF[0..R)  (row length 3+S+R), up to
 * trace_cap rows.  Returns the status (0 done, 1 max_steps, 2 non-finite).
 * ---------------------------------------------------------------------------------------- */
ORA_CLONES
static int ora_integrate_cell(const ora_mechanism *m, const ora_estimator *est, const ora_params *prm, double *T_io,
                              double p, double *Y, int64_t ldy, double t_f, int32_t *steps_out, double *trace,
                              int64_t trace_cap, double *rof_min_out) {
  const int S = m->n_species, R = m->n_reactions;
  ora_rhs w;
  ora_rhs_alloc(m, &w);
  double *rOF = w.rOF;
  double *ring = w.ring; /* [R][13], zero-initialised (R10) */
  for (int j = 0; j < R; ++j) rOF[j] = 1.0; /* Eq 11 */
  double T = *T_io, t = 0.0, rof_min = 1.0;
  int32_t steps = 0, slot = 0, status = 0;
  const double dt_max = t_f * prm->delta_max; /* Eq 4 */

  for (;;) {
    ora_rhs_eval(m, est, prm, T, p, Y, ldy, rOF, &w);

    /* 6. step size, PAPER.md:34-45 (Eqs 1-5) + landing on t_f (R5). */
    double t_star = INFINITY;
    for (int i = 0; i < S; ++i) {
      double r_star = (-w.r[i] > 1.0e-30) ? -w.r[i] : 1.0e-30;                 /* Eq 1 */
      double y_star = (Y[i * ldy] < 1.0e-20) ? 1.0 : 0.9 * Y[i * ldy];         /* Eq 2 (R2) */
      double lim = ((prm->y_step_max < y_star) ? prm->y_step_max : y_star) / r_star;
      if (lim < t_star) t_star = lim;                                          /* Eq 3 */
    }
    double h = (t_star < dt_max) ? t_star : dt_max;                            /* Eq 5 */
    int last = 0;
    double rem = t_f - t;
    if (rem - h < 1.0e-12 * t_f) { h = rem; last = 1; }

    /* 7. forward Euler, PAPER.md:146 (Eq 18). */
    for (int i = 0; i < S; ++i) Y[i * ldy] = fma(h, w.r[i], Y[i * ldy]);
    T = fma(h, w.dTdt, T);
    t = last ? t_f : t + h;
    steps += 1;

    /* 8. DFT stabilisation, PAPER.md:73-95 (Eqs 8-14); stored value = applied change in progress,
     *    normalised by C_tot of this step (R8, R9); high bins n..6 (R10); rOF floor (R13). */
    if (prm->dft_enable) {
      for (int j = 0; j < R; ++j) {
        if (!m->reversible[j]) continue;
        double *rg = ring + j * ORA_WINDOW;
        rg[slot] = (w.q[j] * h) * (1.0 / w.c_tot);                             /* Eq 8 */
        double d0 = ora_dft_bin(rg, 0);                                        /* Eq 9 */
        double d_hi = 0.0;
        for (int mb = prm->dft_first_high_bin; mb <= 6; ++mb) {
          double d = ora_dft_bin(rg, mb);
          if (d > d_hi) d_hi = d;
        }
        double f_ring = d0 / ((d_hi > 1.0e-300) ? d_hi : 1.0e-300);            /* Eq 10 */
        /* Eq 12.  A window without any high-frequency content (d_hi at or below the guard: a dormant reaction whose
         * stored changes are all zero) is not ringing: "rOF will not decline unless the reversible rate is both
         * ringing and at equilibrium". */
        int ringing = (d_hi > 1.0e-300) && (f_ring < prm->tol_ring) && (d0 < prm->tol_freq);
        double rof = rOF[j] * (ringing ? 1.0 / prm->r_fac : prm->r_fac);       /* Eq 13 */
        if (rof > 1.0) rof = 1.0;
        if (rof < prm->rof_min) rof = prm->rof_min;
        rOF[j] = rof;
        if (rof < rof_min) rof_min = rof;
      }
      slot = (slot + 1) % ORA_WINDOW;
    }

    if (trace && steps <= trace_cap) {
      double *row = trace + (int64_t)(steps - 1) * (3 + S + R);
      row[0] = t; row[1] = h; row[2] = T;
      for (int i = 0; i < S; ++i) row[3 + i] = Y[i * ldy];
      for (int j = 0; j < R; ++j) row[3 + S + j] = rOF[j];
    }

    /* 9. retirement, PAPER.md:105 (section 2.4) + R20. */
    int finite = (T - T == 0.0);
    for (int i = 0; i < S; ++i) finite = finite && (Y[i * ldy] - Y[i * ldy] == 0.0);
    if (!finite) { status = 2; break; }      /* checked first: a landing step that produced NaN is not "finished" */
    if (last) { status = 0; break; }
    if (steps >= prm->max_steps) { status = 1; break; }
  }
  *T_io = T;
  *steps_out = steps;
  if (rof_min_out) *rof_min_out = rof_min;
  free(w.base);
  return status;
}

/* N cells, species-major Y [S][ld], in place.  OpenMP over cells only (cells are independent,
 * PAPER.md:105).  rof_min_out / t_unused may be NULL.  Returns 0, or 1 / 2 if any cell has that status
 * (the larger wins). */
int ora_integrate(const ora_mechanism *m, const ora_estimator *est, const ora_params *prm, int64_t n, int64_t ld,
                  double *T, const double *p, double *Y, double dt_cfd, int32_t *steps_out, uint8_t *status_out,
                  double *rof_min_out, int32_t n_threads) {
  int worst = 0;
  if (n_threads < 1) n_threads = 1;
#pragma omp parallel for schedule(dynamic, 4) num_threads(n_threads) reduction(max : worst)
  for (int64_t c = 0; c < n; ++c) {
    int32_t steps = 0;
    double rmin = 1.0;
    int st = ora_integrate_cell(m, est, prm, &T[c], p[c], Y + c, ld, dt_cfd, &steps, NULL, 0, &rmin);
    steps_out[c] = steps;
    if (status_out) status_out[c] = (uint8_t)st;
    if (rof_min_out) rof_min_out[c] = rmin;
    if (st > worst) worst = st;
  }
  return worst;
}

/* One cell with a per-step trace (for the property pins P8-P10). Y is [S] contiguous. */
int ora_integrate_trace(const ora_mechanism *m, const ora_estimator *est, const ora_params *prm, double *T,
                        double p, double *Y, double dt_cfd, int32_t *steps_out, double *trace, int64_t trace_cap) {
  return ora_integrate_cell(m, est, prm, T, p, Y, 1, dt_cfd, steps_out, trace, trace_cap, NULL);
}
