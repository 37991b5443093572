/*
 * stev_oracle_f32.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * The binary32 mode of the oracle: the same algorithm as stev_oracle.c (steps 1-9), with the
 * thermochemical state, the rates, the step selection and the DFT stabilisation all in `float`, as the paper ran it:
 * "the thermochemical state was solved in 32-bit precision and cast back to 64-bit".  The caller's
 * arrays stay double: they are rounded to float on entry and widened on exit.  It is the oracle of
 * stev_params.state_precision = STEV_STATE_FP32; it shares no code with paper_1905_09395_b200/ and only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may load it.
 *
 * Arithmetic contract in binary32, the float twin of section 5: no implicit contraction
 * (-ffp-contract=off), fmaf only where written, + * / sqrtf IEEE, sums sequential in index order, and the two routines
 * below for exp and log.  Constants that the binary64 path takes as literals are the same literals rounded to float;
 * the guards that do not exist in float are replaced (reading R26): Eq 10's 1e-300 guard -> 1e-30f, the landing
 * tolerance 1e-12 t_f -> 1e-6 t_f (a few units in the last place of t, which is accumulated in float), exp saturates
 * outside [-87, 88].  Tables derived from the mechanism (ln A, Ea/R_cal, 1/W, a_k/n) are formed in double exactly as in
 * stev_oracle.c and then rounded to float once.
 *
 * Parity status: as for stev_oracle.c the paper prints no value of any solver quantity (parity with the paper
 * unpinned); this mode is pinned by the same closed forms at float tolerances and against the binary64 oracle at the
 * paper's own accuracy scale (tests/test_oracle_f32.py).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#include "stev_oracle_types.h"

#define F32_RU 0x1.3d2becp+26f    /* (float) 8.31446261815324e7 */
#define F32_PATM 0x1.eec04p+19f   /* (float) 1.01325e6 */
#define F32_WINDOW 13

double ora_log(double x); /* stev_oracle.c: the binary64 contract log, used once per reaction for ln A */

static inline uint32_t f32_bits(float x) { uint32_t u; memcpy(&u, &x, 4); return u; }
static inline float f32_from_bits(uint32_t u) { float x; memcpy(&x, &u, 4); return x; }

/* exp(x): k = round(x log2 e) by the 1.5 * 2^23 shift, r = x - k ln2 in two fmaf steps (ln2_hi has 11 trailing zero
 * bits, so k ln2_hi is exact), Taylor polynomial of degree 7 in Horner form, scaling by 2^k through the exponent
 * field.  x > 88 gives +inf, x < -87 gives 0 (no subnormal results), NaN propagates. */
float ora_expf(float x) {
  if (x != x) return x;
  if (x > 88.0f) return INFINITY;
  if (x < -87.0f) return 0.0f;
  const float shift = 12582912.0f; /* 1.5 * 2^23 */
  float t = fmaf(x, 0x1.715476p+0f, shift);
  float k = t - shift;
  int32_t ki = (int32_t)(f32_bits(t) & 0x7fffffu) - 0x400000;
  float r = fmaf(-k, 0x1.62e4p-1f, x);
  r = fmaf(-k, 0x1.7f7d1cp-20f, r);
  float p = 0x1.a01a02p-13f;          /* 1/5040 */
  p = fmaf(p, r, 0x1.6c16c2p-10f);    /* 1/720 */
  p = fmaf(p, r, 0x1.111112p-7f);     /* 1/120 */
  p = fmaf(p, r, 0x1.555556p-5f);     /* 1/24  */
  p = fmaf(p, r, 0x1.555556p-3f);     /* 1/6   */
  p = fmaf(p, r, 0.5f);
  p = fmaf(p, r, 1.0f);
  p = fmaf(p, r, 1.0f);
  return p * f32_from_bits((uint32_t)(ki + 127) << 23);
}

/* log(x) for positive normal x: x = m 2^e with m in (sqrt(1/2), sqrt 2], f = (m-1)/(m+1), s = f^2,
 * log m = 2f (1 + s/3 + s^2/5 + s^3/7 + s^4/9). */
float ora_logf(float x) {
  if (x != x || x < 0.0f) return NAN;
  if (x == 0.0f) return -INFINITY;
  if (x == INFINITY) return x;
  uint32_t u = f32_bits(x);
  int32_t e = (int32_t)(u >> 23) - 127;
  float m = f32_from_bits((u & 0x007fffffu) | 0x3f800000u);
  if (m > 0x1.6a09e6p+0f) { m = m * 0.5f; e = e + 1; }
  float f = (m - 1.0f) / (m + 1.0f);
  float s = f * f;
  float P = 0x1.c71c72p-4f;           /* 1/9 */
  P = fmaf(P, s, 0x1.24924ap-3f);     /* 1/7 */
  P = fmaf(P, s, 0x1.99999ap-3f);     /* 1/5 */
  P = fmaf(P, s, 0x1.555556p-2f);     /* 1/3 */
  float two_f = f + f;
  float log_m = fmaf(two_f, s * P, two_f);
  float ed = (float)e;
  return fmaf(ed, 0x1.62e4p-1f, fmaf(ed, 0x1.7f7d1cp-20f, log_m));
}

/* NASA-7 (Eqs 15-16; entropy R17) from float coefficient rows:
 * c[0..4] a1..a5 | c[5..8] a2/2, a3/3, a4/4, a5/5 | c[9] a6 | c[10..12] a3/2, a4/3, a5/4 | c[13] a7 */
static void f32_nasa7(const float *c, float T, float lnT, float invT, float *cpR, float *hRT, float *sR) {
  *cpR = fmaf(fmaf(fmaf(fmaf(c[4], T, c[3]), T, c[2]), T, c[1]), T, c[0]);
  float hp = fmaf(fmaf(fmaf(fmaf(c[8], T, c[7]), T, c[6]), T, c[5]), T, c[0]);
  *hRT = fmaf(c[9], invT, hp);
  float sp = fmaf(fmaf(fmaf(c[12], T, c[11]), T, c[10]), T, c[1]);
  *sR = fmaf(c[0], lnT, fmaf(sp, T, c[13]));
}

/* Shallow MLP (R18): fp32 fmaf in index order as in the binary64 mode; the activation goes through
 * the binary32 exp. */
static void f32_mlp_forward(const ora_estimator *e, const float *raw, float *hidden, float *out) {
  float x[64];
  for (int k = 0; k < e->n_in; ++k) x[k] = (raw[k] - e->in_shift[k]) * e->in_scale[k];
  for (int j = 0; j < e->n_hidden; ++j) {
    float z = e->b1[j];
    for (int k = 0; k < e->n_in; ++k) z = fmaf(e->W1[j * e->n_in + k], x[k], z);
    if (e->activation == 0) hidden[j] = 1.0f - 2.0f / (1.0f + ora_expf(2.0f * z)); /* tanh */
    else hidden[j] = 1.0f / (1.0f + ora_expf(-z));                                  /* sigmoid */
  }
  for (int o = 0; o < e->n_out; ++o) {
    float y = e->b2[o];
    for (int j = 0; j < e->n_hidden; ++j) y = fmaf(e->W2[o * e->n_hidden + j], hidden[j], y);
    out[o] = y;
  }
}

/* DFT magnitudes (Eq 9) with the twiddle table of DESIGN.md 5.6 rounded to float. */
static const double F32_COS13_D[13] = {
    1.0, 0.8854560256532099, 0.5680647467311559, 0.120536680255323, -0.35460488704253545,
    -0.7485107481711012, -0.970941817426052, -0.9709418174260521, -0.7485107481711013,
    -0.3546048870425359, 0.1205366802553232, 0.5680647467311548, 0.88545602565321};
static const double F32_SIN13_D[13] = {
    0.0, 0.4647231720437685, 0.8229838658936564, 0.992708874098054, 0.9350162426854148,
    0.6631226582407952, 0.23931566428755768, -0.23931566428755743, -0.663122658240795,
    -0.9350162426854147, -0.992708874098054, -0.822983865893657, -0.4647231720437684};

float ora_dft_bin_f32(const float *ring, int m) {
  if (m == 0) {
    float s = 0.0f;
    for (int k = 0; k < F32_WINDOW; ++k) s = s + ring[k];
    return fabsf(s);
  }
  float re = 0.0f, im = 0.0f;
  for (int k = 0; k < F32_WINDOW; ++k) {
    int n = (m * k) % F32_WINDOW;
    re = fmaf(ring[k], (float)F32_COS13_D[n], re);
    im = fmaf(ring[k], -(float)F32_SIN13_D[n], im);
  }
  return sqrtf(fmaf(re, re, im * im));
}

/* f * C^x (Eq 28; R22), as ora_times_power. */
static float f32_times_power(float f, float c, float x) {
  if (x == 1.0f) return f * c;
  if (x == 2.0f) return (f * c) * c;
  if (x == 3.0f) return ((f * c) * c) * c;
  if (x == 0.0f) return f;
  return f * ((c > 0.0f) ? ora_expf(x * ora_logf(c)) : 0.0f);
}

typedef struct {
  float *cpR, *hRT, *gRT, *conc, *q, *omega, *r;   /* [S],[S],[S],[S],[R],[S],[S] */
  float rho, c_tot, dTdt;
  float *ln_A, *b, *T_a, *inv_W, *W, *t_mid, *nasa; /* tables rounded once: [R],[R],[R],[S],[S],[S],[2][S][14] */
  float *rcoef, *pcoef, *rord, *pord;               /* per CSR entry */
  float *rOF, *ring;                                /* [R], [R][13] */
  float *base;
} f32_rhs;

static float f32_coef(const double *coef, const int32_t *nu, int e) { return coef ? (float)coef[e] : (float)nu[e]; }

static void f32_rhs_alloc(const ora_mechanism *m, f32_rhs *w) {
  const int S = m->n_species, R = m->n_reactions;
  const int nr = m->reac_ptr[R], np = m->prod_ptr[R];
  float *b = (float *)calloc((size_t)(10 * S + 28 * S + 7 * R + R * F32_WINDOW + 2 * nr + 2 * np), sizeof(float));
  w->base = b;
  w->cpR = b; w->hRT = b + S; w->gRT = b + 2 * S; w->conc = b + 3 * S; w->omega = b + 4 * S; w->r = b + 5 * S;
  w->inv_W = b + 6 * S; w->W = b + 7 * S; w->t_mid = b + 8 * S; /* b + 9 S spare */
  w->nasa = b + 10 * S;
  w->q = w->nasa + 28 * S; w->ln_A = w->q + R; w->b = w->q + 2 * R; w->T_a = w->q + 3 * R; w->rOF = w->q + 4 * R;
  w->ring = w->q + 7 * R;
  w->rcoef = w->ring + R * F32_WINDOW; w->rord = w->rcoef + nr; w->pcoef = w->rord + nr; w->pord = w->pcoef + np;
  for (int i = 0; i < S; ++i) {
    w->inv_W[i] = (float)(1.0 / m->mol_weight[i]);
    w->W[i] = (float)m->mol_weight[i];
    w->t_mid[i] = (float)m->t_mid[i];
    for (int rg = 0; rg < 2; ++rg) {
      const double *a = (rg == 0 ? m->nasa_lo : m->nasa_hi) + 7 * i;
      float *c = w->nasa + (rg * S + i) * 14;
      c[0] = (float)a[0]; c[1] = (float)a[1]; c[2] = (float)a[2]; c[3] = (float)a[3]; c[4] = (float)a[4];
      c[5] = (float)(a[1] / 2.0); c[6] = (float)(a[2] / 3.0); c[7] = (float)(a[3] / 4.0); c[8] = (float)(a[4] / 5.0);
      c[9] = (float)a[5];
      c[10] = (float)(a[2] / 2.0); c[11] = (float)(a[3] / 3.0); c[12] = (float)(a[4] / 4.0);
      c[13] = (float)a[6];
    }
  }
  for (int j = 0; j < R; ++j) {
    w->ln_A[j] = (float)ora_log(m->A[j]);
    w->b[j] = (float)m->b[j];
    w->T_a[j] = (float)(m->Ea[j] / 1.98720425864083);
  }
  for (int e = 0; e < nr; ++e) {
    w->rcoef[e] = f32_coef(m->reac_coef, m->reac_nu, e);
    w->rord[e] = m->reac_order ? (float)m->reac_order[e] : w->rcoef[e];
  }
  for (int e = 0; e < np; ++e) {
    w->pcoef[e] = f32_coef(m->prod_coef, m->prod_nu, e);
    w->pord[e] = m->prod_order ? (float)m->prod_order[e] : w->pcoef[e];
  }
}

/* Steps 1-5 of DESIGN.md section 2 for one cell, in float (line by line the float twin of ora_rhs_eval). */
static void f32_rhs_eval(const ora_mechanism *m, const ora_estimator *est, const ora_params *prm, float T, float p,
                         const float *Y, const float *rOF, f32_rhs *w) {
  const int S = m->n_species, R = m->n_reactions;
  const float alpha = (float)prm->alpha;
  /* 1. thermo */
  float lnT = ora_logf(T), invT = 1.0f / T;
  for (int i = 0; i < S; ++i) {
    const float *c = w->nasa + (((T < w->t_mid[i]) ? 0 : S) + i) * 14;
    float sR;
    f32_nasa7(c, T, lnT, invT, &w->cpR[i], &w->hRT[i], &sR);
    w->gRT[i] = w->hRT[i] - sR;
  }
  if (est) {
    float hidden[256], out[512], raw[64];
    raw[0] = T;
    if (est->input_map == 1) {
      raw[1] = p;
      for (int i = 0; i < S; ++i) raw[2 + i] = Y[i];
    }
    f32_mlp_forward(est, raw, hidden, out);
    for (int i = 0; i < S; ++i) {
      w->cpR[i] = out[i];
      w->hRT[i] = (out[S + i] * est->h_ref_temperature) * invT;
    }
  }
  /* 2. mixture and stabilised concentrations (Eqs 6-7) */
  float inv_wbar = 0.0f;
  for (int i = 0; i < S; ++i) inv_wbar = fmaf(Y[i], w->inv_W[i], inv_wbar);
  float c_tot = p / (F32_RU * T);
  float rho = c_tot / inv_wbar;
  for (int i = 0; i < S; ++i) {
    float yp = Y[i] > 0.0f ? Y[i] : 0.0f;
    float c = (rho * yp) * w->inv_W[i];
    if (alpha > 0.0f) c = (yp / (alpha + yp)) * c;
    w->conc[i] = c;
  }
  /* 3.-4. rate constants and progress rates (Eqs 28-30, Eq 14) */
  float ln_c0 = ora_logf(F32_PATM / (F32_RU * T));
  for (int j = 0; j < R; ++j) {
    float ln_kf = fmaf(-w->T_a[j], invT, fmaf(w->b[j], lnT, w->ln_A[j]));
    float fwd = ora_expf(ln_kf);
    for (int e = m->reac_ptr[j]; e < m->reac_ptr[j + 1]; ++e) fwd = f32_times_power(fwd, w->conc[m->reac_species[e]], w->rord[e]);
    float qj = fwd;
    if (m->reversible[j]) {
      float dg = 0.0f, dnu = 0.0f;
      for (int e = m->reac_ptr[j]; e < m->reac_ptr[j + 1]; ++e) {
        dg = dg - w->rcoef[e] * w->gRT[m->reac_species[e]];
        dnu = dnu - w->rcoef[e];
      }
      for (int e = m->prod_ptr[j]; e < m->prod_ptr[j + 1]; ++e) {
        dg = dg + w->pcoef[e] * w->gRT[m->prod_species[e]];
        dnu = dnu + w->pcoef[e];
      }
      float ln_kc = fmaf(dnu, ln_c0, -dg);
      float rev = ora_expf(ln_kf - ln_kc);
      for (int e = m->prod_ptr[j]; e < m->prod_ptr[j + 1]; ++e) rev = f32_times_power(rev, w->conc[m->prod_species[e]], w->pord[e]);
      qj = (fwd - rev) * (rOF ? rOF[j] : 1.0f);
    }
    w->q[j] = qj;
  }
  /* 5. source terms and the temperature equation (R15) */
  for (int i = 0; i < S; ++i) w->omega[i] = 0.0f;
  for (int j = 0; j < R; ++j) {
    for (int e = m->reac_ptr[j]; e < m->reac_ptr[j + 1]; ++e)
      w->omega[m->reac_species[e]] = w->omega[m->reac_species[e]] - w->rcoef[e] * w->q[j];
    for (int e = m->prod_ptr[j]; e < m->prod_ptr[j + 1]; ++e)
      w->omega[m->prod_species[e]] = w->omega[m->prod_species[e]] + w->pcoef[e] * w->q[j];
  }
  float inv_rho = 1.0f / rho;
  float sum_h = 0.0f, sum_cp = 0.0f;
  for (int i = 0; i < S; ++i) {
    w->r[i] = (w->W[i] * w->omega[i]) * inv_rho;
    sum_h = fmaf(w->hRT[i], w->omega[i], sum_h);
    sum_cp = fmaf(Y[i] * w->inv_W[i], w->cpR[i], sum_cp);
  }
  w->dTdt = (prm->energy_mode == 0) ? -((sum_h * F32_RU) * T) / (rho * (F32_RU * sum_cp)) : 0.0f;
  w->rho = rho;
  w->c_tot = c_tot;
}

int ora_rates_eval_f32(const ora_mechanism *m, const ora_estimator *est, const ora_params *prm, int64_t n, int64_t ld,
                       const double *T, const double *p, const double *Y, const double *rOF, double *dYdt, double *dTdt,
                       double *q) {
  const int S = m->n_species, R = m->n_reactions;
  f32_rhs w;
  f32_rhs_alloc(m, &w);
  float *Yc = (float *)malloc(sizeof(float) * (size_t)S);
  for (int64_t c = 0; c < n; ++c) {
    for (int i = 0; i < S; ++i) Yc[i] = (float)Y[i * ld + c];
    if (rOF) for (int j = 0; j < R; ++j) w.rOF[j] = (float)rOF[j * ld + c];
    f32_rhs_eval(m, est, prm, (float)T[c], (float)p[c], Yc, rOF ? w.rOF : NULL, &w);
    for (int i = 0; i < S; ++i) dYdt[i * ld + c] = (double)w.r[i];
    for (int j = 0; j < R; ++j) q[j * ld + c] = (double)w.q[j];
    dTdt[c] = (double)w.dTdt;
  }
  free(Yc);
  free(w.base);
  return 0;
}

/* The STEV loop for one cell in float (the float twin of ora_integrate_cell; trace rows are widened to double). */
static int f32_integrate_cell(const ora_mechanism *m, const ora_estimator *est, const ora_params *prm, double *T_io, double p_in,
                              double *Y_io, int64_t ldy, double t_f_in, int32_t *steps_out, double *trace, int64_t trace_cap,
                              double *rof_min_out) {
  const int S = m->n_species, R = m->n_reactions;
  f32_rhs w;
  f32_rhs_alloc(m, &w);
  float *Y = (float *)malloc(sizeof(float) * (size_t)S);
  for (int i = 0; i < S; ++i) Y[i] = (float)Y_io[i * ldy];
  float *rOF = w.rOF, *ring = w.ring;
  for (int j = 0; j < R; ++j) rOF[j] = 1.0f;                          /* Eq 11 */
  float T = (float)*T_io, p = (float)p_in, t = 0.0f, rof_min = 1.0f;
  const float t_f = (float)t_f_in;
  const float y_step_max = (float)prm->y_step_max, tol_ring = (float)prm->tol_ring, tol_freq = (float)prm->tol_freq;
  const float r_fac = (float)prm->r_fac, inv_r_fac = 1.0f / (float)prm->r_fac, rof_floor = (float)prm->rof_min;
  const float dt_max = t_f * (float)prm->delta_max;                   /* Eq 4 */
  const float t_tol = 1.0e-6f * t_f;                                  /* R5 in float (R26) */
  int32_t steps = 0, slot = 0, status = 0;

  for (;;) {
    f32_rhs_eval(m, est, prm, T, p, Y, rOF, &w);
    /* 6. step size (Eqs 1-5) and landing on t_f */
    float t_star = INFINITY;
    for (int i = 0; i < S; ++i) {
      float r_star = (-w.r[i] > 1.0e-30f) ? -w.r[i] : 1.0e-30f;       /* Eq 1 */
      float y_star = (Y[i] < 1.0e-20f) ? 1.0f : 0.9f * Y[i];          /* Eq 2 */
      float lim = ((y_step_max < y_star) ? y_step_max : y_star) / r_star;
      if (lim < t_star) t_star = lim;                                 /* Eq 3 */
    }
    float h = (t_star < dt_max) ? t_star : dt_max;                    /* Eq 5 */
    int last = 0;
    float rem = t_f - t;
    if (rem - h < t_tol) { h = rem; last = 1; }
    /* 7. forward Euler (Eq 18) */
    for (int i = 0; i < S; ++i) Y[i] = fmaf(h, w.r[i], Y[i]);
    T = fmaf(h, w.dTdt, T);
    t = last ? t_f : t + h;
    steps += 1;
    /* 8. DFT stabilisation (Eqs 8-14; R8, R9, R10, R13) */
    if (prm->dft_enable) {
      for (int j = 0; j < R; ++j) {
        if (!m->reversible[j]) continue;
        float *rg = ring + j * F32_WINDOW;
        rg[slot] = (w.q[j] * h) * (1.0f / w.c_tot);                   /* Eq 8 */
        float d0 = ora_dft_bin_f32(rg, 0);                            /* Eq 9 */
        float d_hi = 0.0f;
        for (int mb = prm->dft_first_high_bin; mb <= 6; ++mb) {
          float d = ora_dft_bin_f32(rg, mb);
          if (d > d_hi) d_hi = d;
        }
        float f_ring = d0 / ((d_hi > 1.0e-30f) ? d_hi : 1.0e-30f);    /* Eq 10 (guard: R26) */
        int ringing = (d_hi > 1.0e-30f) && (f_ring < tol_ring) && (d0 < tol_freq);   /* Eq 12 */
        float rof = rOF[j] * (ringing ? inv_r_fac : r_fac);           /* Eq 13 */
        if (rof > 1.0f) rof = 1.0f;
        if (rof < rof_floor) rof = rof_floor;
        rOF[j] = rof;
        if (rof < rof_min) rof_min = rof;
      }
      slot = (slot + 1) % F32_WINDOW;
    }
    if (trace && steps <= trace_cap) {
      double *row = trace + (int64_t)(steps - 1) * (3 + S + R);
      row[0] = (double)t; row[1] = (double)h; row[2] = (double)T;
      for (int i = 0; i < S; ++i) row[3 + i] = (double)Y[i];
      for (int j = 0; j < R; ++j) row[3 + S + j] = (double)rOF[j];
    }
    /* 9. retirement */
    int finite = (T - T == 0.0f);
    for (int i = 0; i < S; ++i) finite = finite && (Y[i] - Y[i] == 0.0f);
    if (!finite) { status = 2; break; }
    if (last) { status = 0; break; }
    if (steps >= prm->max_steps) { status = 1; break; }
  }
  *T_io = (double)T;
  for (int i = 0; i < S; ++i) Y_io[i * ldy] = (double)Y[i];
  *steps_out = steps;
  if (rof_min_out) *rof_min_out = (double)rof_min;
  free(Y);
  free(w.base);
  return status;
}

int ora_integrate_f32(const ora_mechanism *m, const ora_estimator *est, const ora_params *prm, int64_t n, int64_t ld,
                      double *T, const double *p, double *Y, double dt_cfd, int32_t *steps_out, uint8_t *status_out,
                      double *rof_min_out, int32_t n_threads) {
  int worst = 0;
  if (n_threads < 1) n_threads = 1;
#pragma omp parallel for schedule(dynamic, 4) num_threads(n_threads) reduction(max : worst)
  for (int64_t c = 0; c < n; ++c) {
    int32_t steps = 0;
    double rmin = 1.0;
    int st = f32_integrate_cell(m, est, prm, &T[c], p[c], Y + c, ld, dt_cfd, &steps, NULL, 0, &rmin);
    steps_out[c] = steps;
    if (status_out) status_out[c] = (uint8_t)st;
    if (rof_min_out) rof_min_out[c] = rmin;
    if (st > worst) worst = st;
  }
  return worst;
}

int ora_integrate_trace_f32(const ora_mechanism *m, const ora_estimator *est, const ora_params *prm, double *T, double p,
                            double *Y, double dt_cfd, int32_t *steps_out, double *trace, int64_t trace_cap) {
  return f32_integrate_cell(m, est, prm, T, p, Y, 1, dt_cfd, steps_out, trace, trace_cap, NULL);
}
