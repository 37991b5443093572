// stev_api.cu -- the C ABI of include/stev.h: handles, validation, table images, launch configuration,
// the pass loop of stev_integrate (integrate -> compact active list -> integrate ...).
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <new>

#include "stev_host.h"

namespace stev {

static thread_local std::string g_error;
static thread_local stev_stats g_stats{};

void set_error(const std::string &msg) { g_error = msg; }
int cuda_fail(cudaError_t e, const char *what) {
  g_error = std::string("CUDA error in ") + what + ": " + cudaGetErrorString(e);
  return STEV_ECUDA;
}

int device_sm_count() {
  static int n = 0;
  if (n == 0) {
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return 148;
    if (cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) n = 148;
  }
  return n;
}

// ---------------------------------------------------------------------------------------------------------
static int align_up(int x, int a) { return (x + a - 1) / a * a; }

void build_table_image(const HostMechanism &m, const HostEstimator *e, std::vector<unsigned char> &image, DevTables &tb, bool f32) {
  const int es = f32 ? 4 : 8;   // bytes per real: the binary32 image holds every real table rounded to float once
  const int S = m.S, R = m.R;
  tb = DevTables{};
  tb.S = S;
  tb.R = R;
  tb.Rrev = m.Rrev;
  // gather lists: for species i, every (reaction, signed coefficient) in the caller's reaction order, reactant
  // entries before product entries -- the order in which the plain definition omega_i = sum_j nu_ij q_j is summed.
  std::vector<std::vector<unsigned>> gl(S);
  std::vector<std::vector<double>> glc(S);   // the same entries' signed real coefficients
  for (int j = 0; j < R; ++j) {
    for (int en = m.reac_ptr[j]; en < m.reac_ptr[j + 1]; ++en) {
      gl[m.reac_sp[en]].push_back((unsigned)m.internal_of[j] | ((unsigned)(uint8_t)(int8_t)(-m.reac_nu[en]) << 16));
      glc[m.reac_sp[en]].push_back(-m.reac_coef[en]);
    }
    for (int en = m.prod_ptr[j]; en < m.prod_ptr[j + 1]; ++en) {
      gl[m.prod_sp[en]].push_back((unsigned)m.internal_of[j] | ((unsigned)(uint8_t)(int8_t)(m.prod_nu[en]) << 16));
      glc[m.prod_sp[en]].push_back(m.prod_coef[en]);
    }
  }
  int n_gather = 0;
  for (auto &v : gl) n_gather += (int)v.size();
  tb.n_gather = n_gather;

  int off = 0;
  auto take = [&](int bytes) {
    int o = off;
    off = align_up(off + bytes, 16);
    return o;
  };
  tb.o_invW = take(es * S);
  tb.o_W = take(es * S);
  tb.o_tmid = take(es * S);
  tb.o_nasa = take(es * 2 * kNasaRows * S);
  tb.o_lnA = take(es * R);
  tb.o_b = take(es * R);
  tb.o_Ta = take(es * R);
  tb.o_dnu = take(es * R);
  tb.o_part = take(8 * R);
  tb.o_orig = take(2 * R);
  tb.o_gptr = take(2 * (S + 1));
  tb.o_gent = take(4 * n_gather);
  tb.has_real = m.has_real ? 1 : 0;
  if (m.has_real) {
    tb.o_rcoef = take(es * 4 * R);
    tb.o_rord = take(es * 4 * R);
    tb.o_gcoef = take(es * n_gather);
  }
  if (e) {
    tb.has_est = 1;
    tb.H = e->H;
    tb.n_in = e->n_in;
    tb.n_out = e->n_out;
    tb.act = e->act;
    tb.input_map = e->input_map;
    tb.h_ref_T = e->h_ref_T;
    tb.o_eshift = take(4 * e->n_in);
    tb.o_escale = take(4 * e->n_in);
    tb.o_W1T = take(4 * e->n_in * e->H);
    tb.o_b1 = take(4 * e->H);
    tb.o_W2T = take(4 * e->H * e->n_out);
    tb.o_b2 = take(4 * e->n_out);
  }
  tb.bytes = align_up(off, 128);
  image.assign(tb.bytes, 0);
  unsigned char *base = image.data();
  // every real table entry is formed in double (the same operations as the oracle's table set-up) and stored as double or,
  // for the binary32 image, rounded to float
  auto put = [&](int off0, int idx, double v) {
    if (f32) ((float *)(base + off0))[idx] = (float)v;
    else ((double *)(base + off0))[idx] = v;
  };
  for (int i = 0; i < S; ++i) {
    put(tb.o_invW, i, 1.0 / m.W[i]);
    put(tb.o_W, i, m.W[i]);
    put(tb.o_tmid, i, m.t_mid[i]);
    for (int rg = 0; rg < 2; ++rg) {
      const double *a = (rg == 0 ? m.nasa_lo.data() : m.nasa_hi.data()) + 7 * i;
      const int r0 = rg * kNasaRows * S + i;
      put(tb.o_nasa, r0 + 0 * S, a[0]); put(tb.o_nasa, r0 + 1 * S, a[1]); put(tb.o_nasa, r0 + 2 * S, a[2]);
      put(tb.o_nasa, r0 + 3 * S, a[3]); put(tb.o_nasa, r0 + 4 * S, a[4]);
      put(tb.o_nasa, r0 + 5 * S, a[1] / 2.0); put(tb.o_nasa, r0 + 6 * S, a[2] / 3.0); put(tb.o_nasa, r0 + 7 * S, a[3] / 4.0);
      put(tb.o_nasa, r0 + 8 * S, a[4] / 5.0);
      put(tb.o_nasa, r0 + 9 * S, a[5]);
      put(tb.o_nasa, r0 + 10 * S, a[2] / 2.0); put(tb.o_nasa, r0 + 11 * S, a[3] / 3.0); put(tb.o_nasa, r0 + 12 * S, a[4] / 4.0);
      put(tb.o_nasa, r0 + 13 * S, a[6]);
    }
  }
  unsigned long long *part = (unsigned long long *)(base + tb.o_part);
  unsigned short *orig = (unsigned short *)(base + tb.o_orig);
  for (int k = 0; k < R; ++k) {
    const int j = m.orig_of[k];
    put(tb.o_lnA, k, clog(m.A[j]));
    put(tb.o_b, k, m.b[j]);
    put(tb.o_Ta, k, m.Ea[j] / kRcal);
    orig[k] = (unsigned short)j;
    unsigned long long pk = 0;
    double d = 0.0;
    float d32 = 0.0f;   // Delta-nu summed in the precision of the image, in entry order (as the oracle sums it)
    int slot = 0;
    for (int en = m.reac_ptr[j]; en < m.reac_ptr[j + 1]; ++en, ++slot) {
      pk |= (unsigned long long)(m.reac_sp[en] & 0xff) << (16 * slot);
      pk |= (unsigned long long)(m.reac_nu[en] & 0xff) << (16 * slot + 8);
      d = d - m.reac_coef[en];
      d32 = d32 - (float)m.reac_coef[en];
      if (m.has_real) {
        put(tb.o_rcoef, 4 * k + slot, m.reac_coef[en]);
        put(tb.o_rord, 4 * k + slot, m.reac_order[en]);
      }
    }
    slot = 0;
    for (int en = m.prod_ptr[j]; en < m.prod_ptr[j + 1]; ++en, ++slot) {
      pk |= (unsigned long long)(m.prod_sp[en] & 0xff) << (32 + 16 * slot);
      pk |= (unsigned long long)(m.prod_nu[en] & 0xff) << (32 + 16 * slot + 8);
      d = d + m.prod_coef[en];
      d32 = d32 + (float)m.prod_coef[en];
      if (m.has_real) {
        put(tb.o_rcoef, 4 * k + 2 + slot, m.prod_coef[en]);
        put(tb.o_rord, 4 * k + 2 + slot, m.prod_order[en]);
      }
    }
    part[k] = pk;
    put(tb.o_dnu, k, f32 ? (double)d32 : d);
  }
  unsigned short *gptr = (unsigned short *)(base + tb.o_gptr);
  unsigned *gent = (unsigned *)(base + tb.o_gent);
  int pos = 0;
  for (int i = 0; i < S; ++i) {
    gptr[i] = (unsigned short)pos;
    for (size_t q = 0; q < gl[i].size(); ++q) {
      if (m.has_real) put(tb.o_gcoef, pos, glc[i][q]);
      gent[pos++] = gl[i][q];
    }
  }
  gptr[S] = (unsigned short)pos;
  if (e) {
    float *sh = (float *)(base + tb.o_eshift), *sc = (float *)(base + tb.o_escale), *W1T = (float *)(base + tb.o_W1T);
    float *b1 = (float *)(base + tb.o_b1), *W2T = (float *)(base + tb.o_W2T), *b2 = (float *)(base + tb.o_b2);
    for (int k = 0; k < e->n_in; ++k) {
      sh[k] = e->in_shift[k];
      sc[k] = e->in_scale[k];
      for (int j = 0; j < e->H; ++j) W1T[k * e->H + j] = e->W1[j * e->n_in + k];
    }
    for (int j = 0; j < e->H; ++j) {
      b1[j] = e->b1[j];
      for (int o = 0; o < e->n_out; ++o) W2T[j * e->n_out + o] = e->W2[o * e->H + j];
    }
    for (int o = 0; o < e->n_out; ++o) b2[o] = e->b2[o];
  }
}

// ---------------------------------------------------------------------------------------------------------
static constexpr size_t kSmemMax = 227 * 1024;   // opt-in dynamic shared memory per block on sm_100
static constexpr size_t kSmemPerSM = 228 * 1024;

static void make_layout(const DevTables &tb, int G, CellLayout &cl, int es) {
  const int S = tb.S, R = tb.R, Rrev = tb.Rrev;
  int o = 0;
  auto take = [&](int n) {
    int r = o;
    o += (n + 1) & ~1;
    return r;
  };
  cl.oY = take(S);
  cl.oConc = take(S);
  cl.oG = take(S);
  cl.oCp = take(S);
  cl.oH = take(S);
  cl.oQ = take(R);
  cl.oRof = take(Rrev);
  cl.rrev_pad = Rrev;
  cl.oRing = take(kWindow * Rrev);
  cl.oHid = take(tb.has_est ? (es == 8 ? (tb.H + 1) / 2 : tb.H) : 0);   // H floats
  // pad the stride so that the groups of a half-warp (one 128-byte shared-memory phase) start in distinct banks
  int stride = o;
  if (G < 16) {
    while (stride % (2 * G) != G) ++stride;
  }
  cl.stride = stride;
}

bool choose_config(const DevTables &tb, int request, LaunchConfig &cfg, int es) {
  auto fits = [&](int G, LaunchConfig &c) -> bool {
    make_layout(tb, G, c.cl, es);
    const size_t cell_bytes = (size_t)c.cl.stride * es;
    const size_t avail = kSmemMax - tb.bytes - 64;
    const int cells_sm = (int)std::min<size_t>(avail / cell_bytes, 2048 / G);
    const int per_warp = 32 / G;
    if (cells_sm < per_warp) return false;
    c.G = G;
    if (cells_sm * G <= 512) {
      // one block per SM holding every cell that fits
      c.cells_per_block = cells_sm / per_warp * per_warp;
      c.threads = c.cells_per_block * G;
      c.blocks_per_sm = 1;
    } else {
      c.threads = 256;
      c.cells_per_block = 256 / G;
      size_t blk = tb.bytes + (size_t)c.cells_per_block * cell_bytes + 1024;
      c.blocks_per_sm = (int)std::min<size_t>(kSmemPerSM / blk, 2048 / 256);
      if (c.blocks_per_sm < 1) return false;
    }
    c.smem = tb.bytes + (size_t)c.cells_per_block * cell_bytes;
    return c.smem <= kSmemMax;
  };
  if (request > 0) {
    if (request > 32 || (request & (request - 1))) return false;
    return fits(request, cfg);
  }
  // heuristic: about ten reactions per lane, then widen until an SM holds at least 12 warps (or G = 32)
  int G = 1;
  while (G < 32 && tb.R > 10 * G) G *= 2;
  LaunchConfig best;
  bool have = false;
  for (; G <= 32; G *= 2) {
    LaunchConfig c;
    if (!fits(G, c)) continue;
    best = c;
    have = true;
    const int warps_sm = c.threads * c.blocks_per_sm / 32;
    if (warps_sm >= 12) break;
  }
  if (have) cfg = best;
  return have;
}

}  // namespace stev

using namespace stev;

// =========================================================================================================
//                                               C ABI
// =========================================================================================================
extern "C" {

const char *stev_last_error(void) { return g_error.c_str(); }
const char *stev_version(void) { return "stev-b200 0.1 (sm_100a)"; }

void stev_params_default(stev_params *p) {
  if (!p) return;
  p->y_step_max = 1.0e-2;
  p->delta_max = 1.0e-2;
  p->alpha = 1.0e-5;
  p->tol_ring = 0.5;
  p->tol_freq = 0.1;
  p->r_fac = 2.0;
  p->rof_min = 7.888609052210118e-31;  // 2^-100
  p->dft_window = STEV_DFT_WINDOW;
  p->dft_first_high_bin = 4;
  p->dft_enable = 1;
  p->max_steps = 200000;
  p->energy_mode = STEV_ENERGY_ADIABATIC;
  p->estimator_precision = STEV_PREC_FP32;
  p->state_precision = STEV_STATE_FP64;
  p->nonblocking = 0;
  p->chunk_steps = 0;
  p->lanes_per_cell = 0;
  p->order_cells = 1;
}

void stev_last_stats(stev_stats *out) {
  if (out) *out = g_stats;
}

int stev_mechanism_create(const stev_mechanism_desc *d, stev_mechanism **out) {
  if (!d || !out) { set_error("stev_mechanism_create: null argument"); return STEV_EINVAL; }
  *out = nullptr;
  const int S = d->n_species, R = d->n_reactions, E = d->n_elements;
  if (S < 1 || S > STEV_MAX_SPECIES || R < 1 || R > STEV_MAX_REACTIONS) {
    set_error("stev_mechanism_create: n_species must be 1..64 and n_reactions 1..512");
    return STEV_EINVAL;
  }
  if (!d->mol_weight || !d->nasa_lo || !d->nasa_hi || !d->t_mid || !d->A || !d->b || !d->Ea || !d->reversible ||
      !d->reac_ptr || !d->reac_species || !d->reac_nu || !d->prod_ptr || !d->prod_species || !d->prod_nu) {
    set_error("stev_mechanism_create: null array in descriptor");
    return STEV_EINVAL;
  }
  stev_mechanism *m = new (std::nothrow) stev_mechanism;
  if (!m) { set_error("out of host memory"); return STEV_EINVAL; }
  HostMechanism &h = m->host;
  h.S = S;
  h.R = R;
  h.W.assign(d->mol_weight, d->mol_weight + S);
  h.nasa_lo.assign(d->nasa_lo, d->nasa_lo + 7 * S);
  h.nasa_hi.assign(d->nasa_hi, d->nasa_hi + 7 * S);
  h.t_mid.assign(d->t_mid, d->t_mid + S);
  h.A.assign(d->A, d->A + R);
  h.b.assign(d->b, d->b + R);
  h.Ea.assign(d->Ea, d->Ea + R);
  h.reversible.assign(d->reversible, d->reversible + R);
  h.reac_ptr.assign(d->reac_ptr, d->reac_ptr + R + 1);
  h.prod_ptr.assign(d->prod_ptr, d->prod_ptr + R + 1);
  auto bad = [&](const char *msg) {
    set_error(std::string("stev_mechanism_create: ") + msg);
    delete m;
    return STEV_EINVAL;
  };
  for (int i = 0; i < S; ++i)
    if (!(h.W[i] > 0.0) || !std::isfinite(h.W[i])) return bad("mol_weight must be positive");
  if (h.reac_ptr[0] != 0 || h.prod_ptr[0] != 0) return bad("CSR pointers must start at 0");
  for (int j = 0; j < R; ++j) {
    const int nr = h.reac_ptr[j + 1] - h.reac_ptr[j], np = h.prod_ptr[j + 1] - h.prod_ptr[j];
    if (nr < 1 || nr > 2 || np < 1 || np > 2) return bad("each reaction needs 1..2 reactant and 1..2 product entries");
    if (!(h.A[j] > 0.0) || !std::isfinite(h.A[j])) return bad("A must be positive and finite");
  }
  h.reac_sp.assign(d->reac_species, d->reac_species + h.reac_ptr[R]);
  h.reac_nu.assign(d->reac_nu, d->reac_nu + h.reac_ptr[R]);
  h.prod_sp.assign(d->prod_species, d->prod_species + h.prod_ptr[R]);
  h.prod_nu.assign(d->prod_nu, d->prod_nu + h.prod_ptr[R]);
  h.has_real = d->reac_coef || d->prod_coef || d->reac_order || d->prod_order;
  h.reac_coef.resize(h.reac_sp.size());
  h.reac_order.resize(h.reac_sp.size());
  h.prod_coef.resize(h.prod_sp.size());
  h.prod_order.resize(h.prod_sp.size());
  for (size_t en = 0; en < h.reac_sp.size(); ++en) {
    h.reac_coef[en] = d->reac_coef ? d->reac_coef[en] : (double)h.reac_nu[en];
    h.reac_order[en] = d->reac_order ? d->reac_order[en] : h.reac_coef[en];
  }
  for (size_t en = 0; en < h.prod_sp.size(); ++en) {
    h.prod_coef[en] = d->prod_coef ? d->prod_coef[en] : (double)h.prod_nu[en];
    h.prod_order[en] = d->prod_order ? d->prod_order[en] : h.prod_coef[en];
  }
  for (size_t en = 0; en < h.reac_sp.size(); ++en)
    if (!(h.reac_coef[en] > 0.0) || !(h.reac_order[en] >= 0.0) || !std::isfinite(h.reac_coef[en]) || !std::isfinite(h.reac_order[en]))
      return bad("reac_coef must be positive and reac_order non-negative");
  for (size_t en = 0; en < h.prod_sp.size(); ++en)
    if (!(h.prod_coef[en] > 0.0) || !(h.prod_order[en] >= 0.0) || !std::isfinite(h.prod_coef[en]) || !std::isfinite(h.prod_order[en]))
      return bad("prod_coef must be positive and prod_order non-negative");
  for (int j = 0; j < R; ++j) {
    int seen[4], ns = 0;
    for (int side = 0; side < 2; ++side) {
      const std::vector<int> &ptr = side ? h.prod_ptr : h.reac_ptr, &sp = side ? h.prod_sp : h.reac_sp,
                             &nu = side ? h.prod_nu : h.reac_nu;
      for (int en = ptr[j]; en < ptr[j + 1]; ++en) {
        if (sp[en] < 0 || sp[en] >= S) return bad("species index out of range");
        if (nu[en] < 1 || nu[en] > 3) return bad("stoichiometric coefficients must be 1..3");
        for (int q = 0; q < ns; ++q)
          if (seen[q] == sp[en]) return bad("a species may appear only once per reaction");
        seen[ns++] = sp[en];
      }
    }
    if (d->elem_comp && E > 0) {
      for (int el = 0; el < E; ++el) {
        double bal = 0.0;
        for (int en = h.reac_ptr[j]; en < h.reac_ptr[j + 1]; ++en) bal -= h.reac_coef[en] * d->elem_comp[h.reac_sp[en] * E + el];
        for (int en = h.prod_ptr[j]; en < h.prod_ptr[j + 1]; ++en) bal += h.prod_coef[en] * d->elem_comp[h.prod_sp[en] * E + el];
        if (std::fabs(bal) > 1e-9) return bad("reaction does not conserve elements");
      }
    }
  }
  h.internal_of.assign(R, 0);
  h.orig_of.clear();
  for (int j = 0; j < R; ++j)
    if (h.reversible[j]) h.orig_of.push_back(j);
  h.Rrev = (int)h.orig_of.size();
  for (int j = 0; j < R; ++j)
    if (!h.reversible[j]) h.orig_of.push_back(j);
  for (int k = 0; k < R; ++k) h.internal_of[h.orig_of[k]] = k;

  std::vector<unsigned char> image;
  build_table_image(h, nullptr, image, m->tb);
  cudaError_t e = cudaMalloc(&m->d_table, image.size());
  if (e == cudaSuccess) e = cudaMemcpy(m->d_table, image.data(), image.size(), cudaMemcpyHostToDevice);
  if (e == cudaSuccess) {
    build_table_image(h, nullptr, image, m->tb32, true);
    e = cudaMalloc(&m->d_table32, image.size());
    if (e == cudaSuccess) e = cudaMemcpy(m->d_table32, image.data(), image.size(), cudaMemcpyHostToDevice);
  }
  if (e == cudaSuccess) {
    std::vector<unsigned char> ls;
    m->ls_ok = build_ls_image(h, nullptr, ls, m->ls_tb);
    if (m->ls_ok) {
      e = cudaMalloc(&m->d_ls_table, ls.size());
      if (e == cudaSuccess) e = cudaMemcpy(m->d_ls_table, ls.data(), ls.size(), cudaMemcpyHostToDevice);
    }
    m->ls32_ok = e == cudaSuccess && build_ls_image(h, nullptr, ls, m->ls_tb32, true);
    if (m->ls32_ok) {
      e = cudaMalloc(&m->d_ls_table32, ls.size());
      if (e == cudaSuccess) e = cudaMemcpy(m->d_ls_table32, ls.data(), ls.size(), cudaMemcpyHostToDevice);
    }
  }
  if (e != cudaSuccess) {
    stev_mechanism_destroy(m);
    return cuda_fail(e, "mechanism table upload");
  }
  *out = m;
  return STEV_OK;
}

void stev_mechanism_destroy(stev_mechanism *m) {
  if (!m) return;
  if (m->d_table) cudaFree(m->d_table);
  if (m->d_table32) cudaFree(m->d_table32);
  if (m->d_ls_table) cudaFree(m->d_ls_table);
  if (m->d_ls_table32) cudaFree(m->d_ls_table32);
  delete m;
}

int stev_mechanism_sizes(const stev_mechanism *m, int32_t *S, int32_t *R, int32_t *Rrev) {
  if (!m) { set_error("null mechanism"); return STEV_EINVAL; }
  if (S) *S = m->host.S;
  if (R) *R = m->host.R;
  if (Rrev) *Rrev = m->host.Rrev;
  return STEV_OK;
}

int stev_estimator_load(const stev_mechanism *m, const stev_estimator_desc *d, stev_estimator **out) {
  if (!d || !out) { set_error("stev_estimator_load: null argument"); return STEV_EINVAL; }
  *out = nullptr;
  if (d->n_in < 1 || d->n_in > 64 || d->n_hidden < 8 || d->n_hidden > 128 || d->n_hidden % 8 || d->n_out < 1 || d->n_out > 256) {
    set_error("stev_estimator_load: need 1 <= n_in <= 64, 8 <= n_hidden <= 128 (multiple of 8), 1 <= n_out <= 256");
    return STEV_EINVAL;
  }
  if (d->activation != STEV_ACT_TANH && d->activation != STEV_ACT_SIGMOID) { set_error("unknown activation"); return STEV_EINVAL; }
  if (d->input_map != STEV_IN_T && d->input_map != STEV_IN_T_P_Y) { set_error("unknown input_map"); return STEV_EINVAL; }
  if (!d->in_shift || !d->in_scale || !d->W1 || !d->b1 || !d->W2 || !d->b2) { set_error("null weight array"); return STEV_EINVAL; }
  if (m) {
    const int S = m->host.S;
    if (d->n_out != 2 * S) { set_error("an estimator attached to a mechanism must have n_out = 2 * n_species"); return STEV_EINVAL; }
    if ((d->input_map == STEV_IN_T && d->n_in != 1) || (d->input_map == STEV_IN_T_P_Y && d->n_in != 2 + S)) {
      set_error("n_in does not match input_map");
      return STEV_EINVAL;
    }
  }
  stev_estimator *e = new (std::nothrow) stev_estimator;
  if (!e) { set_error("out of host memory"); return STEV_EINVAL; }
  HostEstimator &h = e->host;
  h.n_in = d->n_in; h.H = d->n_hidden; h.n_out = d->n_out; h.act = d->activation; h.input_map = d->input_map;
  h.h_ref_T = d->h_ref_temperature;
  h.in_shift.assign(d->in_shift, d->in_shift + h.n_in);
  h.in_scale.assign(d->in_scale, d->in_scale + h.n_in);
  h.W1.assign(d->W1, d->W1 + (size_t)h.H * h.n_in);
  h.b1.assign(d->b1, d->b1 + h.H);
  h.W2.assign(d->W2, d->W2 + (size_t)h.n_out * h.H);
  h.b2.assign(d->b2, d->b2 + h.n_out);
  e->mech = m;
  cudaError_t ce = cudaSuccess;
  if (m) {
    std::vector<unsigned char> image;
    build_table_image(m->host, &h, image, e->tb);
    ce = cudaMalloc(&e->d_table, image.size());
    if (ce == cudaSuccess) ce = cudaMemcpy(e->d_table, image.data(), image.size(), cudaMemcpyHostToDevice);
    if (ce == cudaSuccess) {
      build_table_image(m->host, &h, image, e->tb32, true);
      ce = cudaMalloc(&e->d_table32, image.size());
      if (ce == cudaSuccess) ce = cudaMemcpy(e->d_table32, image.data(), image.size(), cudaMemcpyHostToDevice);
    }
  }
  if (ce == cudaSuccess && m) {
    std::vector<unsigned char> ls;
    e->ls_ok = build_ls_image(m->host, &h, ls, e->ls_tb);
    if (e->ls_ok) {
      ce = cudaMalloc(&e->d_ls_table, ls.size());
      if (ce == cudaSuccess) ce = cudaMemcpy(e->d_ls_table, ls.data(), ls.size(), cudaMemcpyHostToDevice);
    }
    e->ls32_ok = ce == cudaSuccess && build_ls_image(m->host, &h, ls, e->ls_tb32, true);
    if (e->ls32_ok) {
      ce = cudaMalloc(&e->d_ls_table32, ls.size());
      if (ce == cudaSuccess) ce = cudaMemcpy(e->d_ls_table32, ls.data(), ls.size(), cudaMemcpyHostToDevice);
    }
  }
  if (ce == cudaSuccess) {
    // standalone parameter block: in_shift, in_scale, W1T [n_in][H], b1, W2T [H][n_out], b2
    std::vector<float> pb;
    pb.insert(pb.end(), h.in_shift.begin(), h.in_shift.end());
    pb.insert(pb.end(), h.in_scale.begin(), h.in_scale.end());
    for (int k = 0; k < h.n_in; ++k)
      for (int j = 0; j < h.H; ++j) pb.push_back(h.W1[(size_t)j * h.n_in + k]);
    pb.insert(pb.end(), h.b1.begin(), h.b1.end());
    for (int j = 0; j < h.H; ++j)
      for (int o = 0; o < h.n_out; ++o) pb.push_back(h.W2[(size_t)o * h.H + j]);
    pb.insert(pb.end(), h.b2.begin(), h.b2.end());
    e->params_floats = pb.size();
    ce = cudaMalloc(&e->d_params, pb.size() * sizeof(float));
    if (ce == cudaSuccess) ce = cudaMemcpy(e->d_params, pb.data(), pb.size() * sizeof(float), cudaMemcpyHostToDevice);
  }
  if (ce == cudaSuccess && estimator_tensor_prepare(e) != STEV_OK) {
    stev_estimator_destroy(e);
    return STEV_ECUDA;
  }
  if (ce != cudaSuccess) {
    stev_estimator_destroy(e);
    return cuda_fail(ce, "estimator upload");
  }
  *out = e;
  return STEV_OK;
}

void stev_estimator_destroy(stev_estimator *e) {
  if (!e) return;
  if (e->d_table) cudaFree(e->d_table);
  if (e->d_table32) cudaFree(e->d_table32);
  if (e->d_ls_table) cudaFree(e->d_ls_table);
  if (e->d_ls_table32) cudaFree(e->d_ls_table32);
  if (e->d_params) cudaFree(e->d_params);
  for (int k = 0; k < 2; ++k)
    if (e->d_tc_image[k]) cudaFree(e->d_tc_image[k]);
  delete e;
}

}  // extern "C"

// ---------------------------------------------------------------------------------------------------------
// Workspace carving
// ---------------------------------------------------------------------------------------------------------
namespace {
struct Workspace {
  int *counters;            // [0] queue head, [1] worst status, [2] active count
  int *list[2];
  int *order;               // launch order (hottest cells first), order_hist: its counting-sort scratch
  int *order_hist;
  unsigned char *flags;
  int *block_counts;
  double *spill;
  long long spill_stride;
  size_t bytes;
};
size_t rnd256(size_t x) { return (x + 255) & ~(size_t)255; }

Workspace carve(void *base, const DevTables &tb, const stev_params *p, int64_t n) {
  Workspace w{};
  size_t off = 0;
  auto take = [&](size_t bytes) {
    size_t o = off;
    off += rnd256(bytes);
    return base ? (unsigned char *)base + o : (unsigned char *)nullptr;
  };
  w.counters = (int *)take(256);
  if (p->order_cells) {
    w.order = (int *)take(4 * (size_t)n);
    w.order_hist = (int *)take(4 * (size_t)(kOrderBuckets + 1));
  }
  if (p->chunk_steps > 0) {
    w.list[0] = (int *)take(4 * (size_t)n);
    w.list[1] = (int *)take(4 * (size_t)n);
    w.flags = take((size_t)n);
    w.block_counts = (int *)take(4 * ((size_t)n / 1024 + 2));
    w.spill_stride = 3 + (long long)tb.Rrev * (1 + kWindow);
    w.spill = (double *)take(8 * (size_t)n * (size_t)w.spill_stride);
  }
  w.bytes = off;
  return w;
}

int check_params(const stev_params *p) {
  if (!p) { set_error("null params"); return STEV_EINVAL; }
  if (!(p->y_step_max > 0) || !(p->delta_max > 0 && p->delta_max <= 1) || !(p->alpha >= 0) || !(p->r_fac > 1) ||
      !(p->rof_min > 0 && p->rof_min <= 1) || p->dft_first_high_bin < 1 || p->dft_first_high_bin > 6 || p->max_steps < 1 ||
      (p->energy_mode != 0 && p->energy_mode != 1) || p->chunk_steps < 0) {
    set_error("stev_params out of range");
    return STEV_EINVAL;
  }
  if (p->dft_window != STEV_DFT_WINDOW) {
    set_error("stev_params.dft_window: only 13 is implemented (PAPER.md:77, 'the thirteen most recent changes')");
    return STEV_EINVAL;
  }
  if (p->estimator_precision != STEV_PREC_FP32) {
    set_error("stev_params.estimator_precision: inside stev_integrate the estimator runs on the fp32 CUDA-core path only "
              "(STEV_PREC_FP32); the TF32 / BF16 tensor-core paths are reached through stev_estimator_eval");
    return STEV_EINVAL;
  }
  if (p->state_precision != STEV_STATE_FP64 && p->state_precision != STEV_STATE_FP32) {
    set_error("stev_params.state_precision must be STEV_STATE_FP64 or STEV_STATE_FP32");
    return STEV_EINVAL;
  }
  return STEV_OK;
}

SolverConsts make_consts(const stev_params *p) {
  SolverConsts sc;
  sc.y_step_max = p->y_step_max;
  sc.delta_max = p->delta_max;
  sc.alpha = p->alpha;
  sc.tol_ring = p->tol_ring;
  sc.tol_freq = p->tol_freq;
  sc.r_fac = p->r_fac;
  sc.inv_r_fac = 1.0 / p->r_fac;
  sc.rof_min = p->rof_min;
  sc.tol_ring2 = p->tol_ring * p->tol_ring;
  sc.ring_lo = 1.0 - 1.0e-14;
  sc.ring_hi = 1.0 + 1.0e-14;
  sc.ring_filter_ok = (p->tol_ring > 1.0e-9 && p->tol_ring < 1.0e9) ? 1 : 0;
  sc.nhf = p->dft_first_high_bin;
  sc.dft_enable = p->dft_enable;
  sc.max_steps = p->max_steps;
  sc.energy_mode = p->energy_mode;
  return sc;
}

int pick_tables(const stev_mechanism *m, const stev_estimator *e, const DevTables **tb, const unsigned char **table,
                bool f32 = false) {
  if (!m) { set_error("null mechanism"); return STEV_EINVAL; }
  if (e) {
    if (e->mech != m || !e->d_table) { set_error("estimator was not loaded against this mechanism"); return STEV_EINVAL; }
    *tb = f32 ? &e->tb32 : &e->tb;
    *table = f32 ? e->d_table32 : e->d_table;
  } else {
    *tb = f32 ? &m->tb32 : &m->tb;
    *table = f32 ? m->d_table32 : m->d_table;
  }
  return STEV_OK;
}

template <typename Args>
using KernelPtr = void (*)(const Args);

template <int G> void *integrate_fn(bool f32) { return f32 ? (void *)stev_integrate_kernel<G, float> : (void *)stev_integrate_kernel<G, double>; }
template <int G> void *rates_fn(bool f32) { return f32 ? (void *)stev_rates_kernel<G, float> : (void *)stev_rates_kernel<G, double>; }

void *integrate_kernel_for(int G, bool f32) {
  switch (G) {
    case 1: return integrate_fn<1>(f32);
    case 2: return integrate_fn<2>(f32);
    case 4: return integrate_fn<4>(f32);
    case 8: return integrate_fn<8>(f32);
    case 16: return integrate_fn<16>(f32);
    default: return integrate_fn<32>(f32);
  }
}
void *rates_kernel_for(int G, bool f32) {
  switch (G) {
    case 1: return rates_fn<1>(f32);
    case 2: return rates_fn<2>(f32);
    case 4: return rates_fn<4>(f32);
    case 8: return rates_fn<8>(f32);
    case 16: return rates_fn<16>(f32);
    default: return rates_fn<32>(f32);
  }
}
}  // namespace

// compaction kernels live in stev_compact.cu
namespace stev {
int compact_launch(const unsigned char *flags, const int *list_in, int n, int *list_out, int *count_out, int *block_counts,
                   cudaStream_t s);
}

namespace {
std::mutex g_scratch_mutex;
void *g_scratch = nullptr;
size_t g_scratch_bytes = 0;
cudaStream_t g_host_stream = nullptr;
}  // namespace

// Reads back the worst per-cell status (one int) after the stream has drained and turns it into the return code.
static int finish_integrate(const int *counters, cudaStream_t s) {
  int worst = 0;
  STEV_CUDA(cudaMemcpyAsync(&worst, counters + 1, 4, cudaMemcpyDeviceToHost, s));
  STEV_CUDA(cudaStreamSynchronize(s));
  STEV_CUDA(cudaGetLastError());
  if (worst == 2) { set_error("some cells produced non-finite values (status 2)"); return STEV_WNONFINITE; }
  if (worst == 1) { set_error("some cells stopped at max_steps (status 1)"); return STEV_WMAXSTEPS; }
  return STEV_OK;
}

extern "C" {

size_t stev_workspace_bytes(const stev_mechanism *m, const stev_estimator *e, const stev_params *p, int64_t n_cells) {
  const DevTables *tb;
  const unsigned char *table;
  if (!p || n_cells < 0 || pick_tables(m, e, &tb, &table) != STEV_OK) return 0;
  return carve(nullptr, *tb, p, n_cells).bytes;
}

int stev_integrate(const stev_mechanism *m, const stev_estimator *est, const stev_params *p, int64_t n, int64_t ld,
                   double *T, const double *pressure, double *Y, double dt_cfd, int32_t *steps_out, uint8_t *status_out,
                   void *workspace, size_t workspace_bytes, void *cuda_stream) {
  const DevTables *tb;
  const unsigned char *table;
  int rc = check_params(p);
  if (rc) return rc;
  const bool f32 = p->state_precision == STEV_STATE_FP32;
  if ((rc = pick_tables(m, est, &tb, &table, f32))) return rc;
  if (n < 0 || n > 0x7fffffff || ld < n || !(dt_cfd > 0.0) || !std::isfinite(dt_cfd)) {
    set_error("stev_integrate: need 0 <= n_cells <= 2^31-1, ld >= n_cells, dt_cfd > 0");
    return STEV_EINVAL;
  }
  g_stats = stev_stats{};
  g_stats.total_steps = -1;
  if (n == 0) return STEV_OK;
  if (!T || !pressure || !Y || !steps_out) { set_error("stev_integrate: null state pointer"); return STEV_EINVAL; }
  Workspace need = carve(nullptr, *tb, p, n);
  if (!workspace || workspace_bytes < need.bytes || ((uintptr_t)workspace & 255)) {
    set_error("stev_integrate: workspace missing, misaligned or smaller than stev_workspace_bytes()");
    return STEV_EWORKSPACE;
  }
  cudaStream_t s = (cudaStream_t)cuda_stream;
  Workspace w = carve(workspace, *tb, p, n);

  // The lock-step kernel keeps the DFT history in tensor memory and the whole working set of its cells on chip
  // (stev_ls_kernel.cuh); it needs chunk_steps = 0, at most two concentration factors per reaction side and integer
  // coefficients.  lanes_per_cell = 0: that kernel wherever the mechanism fits it; 512: the same, refusing if it does not
  // fit; 513: the same with the dimensions read at run time even if the shape list has the mechanism; 1..32: the
  // shared-memory-history kernel below.
  const int g_request = (p->lanes_per_cell >= 1 && p->lanes_per_cell <= 32) ? p->lanes_per_cell : 0;
  {
    const bool ls_ok = (f32 ? (est ? est->ls32_ok : m->ls32_ok) : (est ? est->ls_ok : m->ls_ok)) && p->chunk_steps == 0;
    const bool want_ls = p->lanes_per_cell == 512 || p->lanes_per_cell == 513;
    if (p->lanes_per_cell != 0 && !want_ls && g_request == 0) {
      set_error("stev_integrate: lanes_per_cell must be 0, 1, 2, 4, 8, 16, 32, 512 or 513");
      return STEV_EINVAL;
    }
    if (want_ls && !ls_ok) {
      set_error("stev_integrate: lanes_per_cell = 512 / 513 (lock-step kernel, DFT history in tensor memory) needs chunk_steps = 0, "
                "at most two factors per reaction side, integer coefficients, at most 64 species");
      return STEV_EINVAL;
    }
    if (ls_ok && (want_ls || p->lanes_per_cell == 0)) {
      STEV_CUDA(cudaMemsetAsync(w.counters, 0, 256, s));
      const int *order = nullptr;
      if (p->order_cells && n > 1) {
        rc = order_cells_launch(T, n, order_group(p->order_cells, n, tb->S), w.order, w.order_hist, s);
        if (rc) return rc;
        order = w.order;
      }
      int blocks = 0;
      size_t smem = 0;
      const stev::LsTables &ltb = f32 ? (est ? est->ls_tb32 : m->ls_tb32) : (est ? est->ls_tb : m->ls_tb);
      const unsigned char *ltable = f32 ? (est ? est->d_ls_table32 : m->d_ls_table32) : (est ? est->d_ls_table : m->d_ls_table);
      bool is_static = false;
      rc = integrate_ls_launch(ltb, ltable, make_consts(p), dt_cfd, n, ld, T, pressure, Y, steps_out, status_out, w.counters, s,
                               &blocks, &smem, order, p->lanes_per_cell != 513, &is_static);
      if (rc) return rc;
      g_stats.passes = 1;
      g_stats.specialised = is_static ? 1 : 0;
      g_stats.kernel_launches = 1 + (order ? 3 : 0);   // integrator + histogram, scan, scatter of the launch order
      g_stats.blocks = blocks;
      g_stats.lanes_per_cell = p->lanes_per_cell == 513 ? 513 : 512;
      g_stats.threads_per_block = kLsThreads;
      g_stats.cells_per_block = ltb.d.C;
      g_stats.smem_bytes = (int64_t)smem;
      if (p->nonblocking) return STEV_OK;
      return finish_integrate(w.counters, s);
    }
  }

  const int es = f32 ? 4 : 8;
  LaunchConfig cfg;
  if (!choose_config(*tb, g_request, cfg, es) && !(p->lanes_per_cell == 0 && choose_config(*tb, 0, cfg, es))) {
    set_error("stev_integrate: no launch configuration fits shared memory for this mechanism / lanes_per_cell");
    return STEV_EINVAL;
  }
  void *fn = integrate_kernel_for(cfg.G, f32);
  STEV_CUDA(cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)cfg.smem));

  IntegrateArgs a{};
  a.tb = *tb;
  a.table = table;
  a.cl = cfg.cl;
  a.sc = make_consts(p);
  a.t_f = dt_cfd;
  a.ld = ld;
  a.T = T;
  a.p = pressure;
  a.Y = Y;
  a.steps = steps_out;
  a.status = status_out;
  a.queue_head = w.counters;
  a.worst_status = w.counters + 1;
  a.chunk_steps = p->chunk_steps;
  a.flags = w.flags;
  a.spill = w.spill;
  a.spill_stride = w.spill_stride;

  const int sms = device_sm_count();
  long long n_active = n;
  int cur = 0;
  STEV_CUDA(cudaMemsetAsync(w.counters, 0, 256, s));
  const int *order = nullptr;
  if (p->order_cells && n > 1) {
    rc = order_cells_launch(T, n, order_group(p->order_cells, n, tb->S), w.order, w.order_hist, s);
    if (rc) return rc;
    order = w.order;
  }
  if (order) g_stats.kernel_launches += 3;
  for (int pass = 0; n_active > 0; ++pass) {
    a.n_active = n_active;
    a.list = (pass == 0) ? order : w.list[cur];
    a.restore = (pass > 0);
    long long blocks = std::min<long long>((long long)sms * cfg.blocks_per_sm, (n_active + cfg.cells_per_block - 1) / cfg.cells_per_block);
    if (pass > 0) STEV_CUDA(cudaMemsetAsync(w.counters, 0, 4, s));
    void *args[] = {&a};
    STEV_CUDA(cudaLaunchKernel(fn, dim3((unsigned)blocks), dim3(cfg.threads), args, cfg.smem, s));
    g_stats.passes += 1;
    g_stats.kernel_launches += 1;
    g_stats.blocks = (int)blocks;
    if (p->chunk_steps <= 0) break;
    int rcc = compact_launch(w.flags, a.list, (int)n_active, w.list[cur ^ 1], w.counters + 2, w.block_counts, s);
    if (rcc) return rcc;
    g_stats.kernel_launches += 3;
    int count = 0;
    STEV_CUDA(cudaMemcpyAsync(&count, w.counters + 2, 4, cudaMemcpyDeviceToHost, s));
    STEV_CUDA(cudaStreamSynchronize(s));
    n_active = count;
    cur ^= 1;
  }
  g_stats.lanes_per_cell = cfg.G;
  g_stats.threads_per_block = cfg.threads;
  g_stats.cells_per_block = cfg.cells_per_block;
  g_stats.smem_bytes = (int64_t)cfg.smem;
  if (p->nonblocking && p->chunk_steps <= 0) return STEV_OK;
  return finish_integrate(w.counters, s);
}

int stev_integrate_finish(void *workspace, void *cuda_stream) {
  if (!workspace) { set_error("stev_integrate_finish: null workspace"); return STEV_EINVAL; }
  return finish_integrate((const int *)workspace, (cudaStream_t)cuda_stream);   // the counters are the first 256 bytes
}

// ---------------------------------------------------------------------------------------------------------
// Host-buffer entry point: grow-only device scratch owned by the library.
// ---------------------------------------------------------------------------------------------------------
int stev_integrate_host(const stev_mechanism *m, const stev_estimator *est, const stev_params *p, int64_t n, int64_t ld,
                        double *T, const double *pressure, double *Y, double dt_cfd, int32_t *steps_out, uint8_t *status_out) {
  if (!m) { set_error("null mechanism"); return STEV_EINVAL; }
  if (n == 0) return STEV_OK;
  if (n < 0 || ld < n || !T || !pressure || !Y || !steps_out) { set_error("stev_integrate_host: bad argument"); return STEV_EINVAL; }
  std::lock_guard<std::mutex> lock(g_scratch_mutex);
  const int S = m->host.S;
  const size_t ws = stev_workspace_bytes(m, est, p, n);
  if (p == nullptr) { set_error("null params"); return STEV_EINVAL; }
  size_t off = 0;
  auto take = [&](size_t b) { size_t o = off; off += rnd256(b); return o; };
  const size_t oT = take(8 * (size_t)n), oP = take(8 * (size_t)n), oY = take(8 * (size_t)n * S), oS = take(4 * (size_t)n),
               oSt = take((size_t)n), oW = take(ws);
  if (off > g_scratch_bytes) {
    if (g_scratch) cudaFree(g_scratch);
    g_scratch = nullptr;
    g_scratch_bytes = 0;
    STEV_CUDA(cudaMalloc(&g_scratch, off));
    g_scratch_bytes = off;
  }
  if (!g_host_stream) STEV_CUDA(cudaStreamCreateWithFlags(&g_host_stream, cudaStreamNonBlocking));
  unsigned char *b = (unsigned char *)g_scratch;
  cudaStream_t s = g_host_stream;
  STEV_CUDA(cudaMemcpyAsync(b + oT, T, 8 * (size_t)n, cudaMemcpyHostToDevice, s));
  STEV_CUDA(cudaMemcpyAsync(b + oP, pressure, 8 * (size_t)n, cudaMemcpyHostToDevice, s));
  if (ld == n) {
    STEV_CUDA(cudaMemcpyAsync(b + oY, Y, 8 * (size_t)n * S, cudaMemcpyHostToDevice, s));
  } else {
    STEV_CUDA(cudaMemcpy2DAsync(b + oY, 8 * (size_t)n, Y, 8 * (size_t)ld, 8 * (size_t)n, S, cudaMemcpyHostToDevice, s));
  }
  stev_params pb = *p;
  pb.nonblocking = 0;
  p = &pb;
  int rc = stev_integrate(m, est, p, n, n, (double *)(b + oT), (const double *)(b + oP), (double *)(b + oY), dt_cfd,
                          (int32_t *)(b + oS), (uint8_t *)(b + oSt), b + oW, ws, s);
  if (rc < 0) return rc;
  stev_stats keep = g_stats;
  STEV_CUDA(cudaMemcpyAsync(T, b + oT, 8 * (size_t)n, cudaMemcpyDeviceToHost, s));
  if (ld == n) {
    STEV_CUDA(cudaMemcpyAsync(Y, b + oY, 8 * (size_t)n * S, cudaMemcpyDeviceToHost, s));
  } else {
    STEV_CUDA(cudaMemcpy2DAsync(Y, 8 * (size_t)ld, b + oY, 8 * (size_t)n, 8 * (size_t)n, S, cudaMemcpyDeviceToHost, s));
  }
  STEV_CUDA(cudaMemcpyAsync(steps_out, b + oS, 4 * (size_t)n, cudaMemcpyDeviceToHost, s));
  if (status_out) STEV_CUDA(cudaMemcpyAsync(status_out, b + oSt, (size_t)n, cudaMemcpyDeviceToHost, s));
  STEV_CUDA(cudaStreamSynchronize(s));
  long long tot = 0;
  for (int64_t c = 0; c < n; ++c) tot += steps_out[c];
  keep.total_steps = tot;
  g_stats = keep;
  return rc;
}

int stev_rates_eval(const stev_mechanism *m, const stev_estimator *est, const stev_params *p, int64_t n, int64_t ld,
                    const double *T, const double *pressure, const double *Y, const double *rOF, double *dYdt, double *dTdt,
                    double *q, void *cuda_stream) {
  const DevTables *tb;
  const unsigned char *table;
  int rc = check_params(p);
  if (rc) return rc;
  const bool f32 = p->state_precision == STEV_STATE_FP32;
  if ((rc = pick_tables(m, est, &tb, &table, f32))) return rc;
  if (n < 0 || ld < n) { set_error("stev_rates_eval: bad sizes"); return STEV_EINVAL; }
  if (n == 0) return STEV_OK;
  if (!T || !pressure || !Y || !dYdt || !dTdt || !q) { set_error("stev_rates_eval: null pointer"); return STEV_EINVAL; }
  LaunchConfig cfg;
  // lanes_per_cell values above 32 name the tensor-memory kernels of stev_integrate: here they mean "choose"
  if (!choose_config(*tb, p->lanes_per_cell > 32 ? 0 : p->lanes_per_cell, cfg, f32 ? 4 : 8)) { set_error("no launch configuration fits"); return STEV_EINVAL; }
  void *fn = rates_kernel_for(cfg.G, f32);
  STEV_CUDA(cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)cfg.smem));
  RatesArgs a{};
  a.tb = *tb;
  a.table = table;
  a.cl = cfg.cl;
  a.sc = make_consts(p);
  a.n = n;
  a.ld = ld;
  a.T = T;
  a.p = pressure;
  a.Y = Y;
  a.rOF = rOF;
  a.dYdt = dYdt;
  a.dTdt = dTdt;
  a.q = q;
  long long blocks = std::min<long long>((long long)device_sm_count() * cfg.blocks_per_sm, (n + cfg.cells_per_block - 1) / cfg.cells_per_block);
  void *args[] = {&a};
  STEV_CUDA(cudaLaunchKernel(fn, dim3((unsigned)blocks), dim3(cfg.threads), args, cfg.smem, (cudaStream_t)cuda_stream));
  STEV_CUDA(cudaGetLastError());
  return STEV_OK;
}

}  // extern "C"

// ---------------------------------------------------------------------------------------------------------
// stev_integrate_static: the lock-step integrator for callers that cannot allocate (code under CUDA graph capture,
// serving loops, harnesses that forbid cudaMalloc).  Its scratch -- the queue head / worst-status counters, the launch
// order of the cells and the counting sort's histogram -- lives in ONE file-scope device array of fixed size that every
// GPU loading this library holds until the process exits.  In host code the array's name is a host-side stand-in, not a
// device address: its address is taken once per device with cudaGetSymbolAddress (that device current) and that
// pointer is what the kernels get.
// ---------------------------------------------------------------------------------------------------------
namespace {
constexpr size_t kStaticCountersBytes = 256;
constexpr size_t kStaticOrderBytes = 4 * (size_t)STEV_STATIC_MAX_CELLS;
constexpr size_t kStaticHistBytes = (4 * (size_t)(stev::kOrderBuckets + 1) + 255) & ~(size_t)255;
constexpr size_t kStaticScratchBytes = kStaticCountersBytes + kStaticOrderBytes + kStaticHistBytes;   // 1 MiB + 16.25 KiB
static __device__ __align__(256) unsigned char g_static_scratch[kStaticScratchBytes];

constexpr int kStaticMaxDevices = 64;
std::mutex g_static_mutex;
unsigned char *g_static_ptr[kStaticMaxDevices] = {};

// device address of g_static_scratch on the current device (looked up once per device)
int static_scratch(unsigned char **out) {
  int dev = -1;
  STEV_CUDA(cudaGetDevice(&dev));
  if (dev < 0 || dev >= kStaticMaxDevices) { stev::set_error("stev_integrate_static: device ordinal beyond 63"); return STEV_EINVAL; }
  std::lock_guard<std::mutex> lock(g_static_mutex);
  if (!g_static_ptr[dev]) {
    void *ptr = nullptr;
    STEV_CUDA(cudaGetSymbolAddress(&ptr, g_static_scratch));
    if (!ptr) { stev::set_error("stev_integrate_static: cudaGetSymbolAddress returned a null address"); return STEV_ECUDA; }
    g_static_ptr[dev] = (unsigned char *)ptr;
  }
  *out = g_static_ptr[dev];
  return STEV_OK;
}
}  // namespace

extern "C" {

int stev_integrate_static(const stev_mechanism *m, const stev_estimator *est, const stev_params *p, int64_t n, int64_t ld,
                          double *T, const double *pressure, double *Y, double dt_cfd, int32_t *steps_out, uint8_t *status_out,
                          void *cuda_stream) {
  const DevTables *tb;
  const unsigned char *table;
  int rc = check_params(p);
  if (rc) return rc;
  const bool f32 = p->state_precision == STEV_STATE_FP32;
  if ((rc = pick_tables(m, est, &tb, &table, f32))) return rc;
  if (n < 0 || ld < n || !(dt_cfd > 0.0) || !std::isfinite(dt_cfd)) {
    set_error("stev_integrate_static: need n_cells >= 0, ld >= n_cells, dt_cfd > 0");
    return STEV_EINVAL;
  }
  if (n > STEV_STATIC_MAX_CELLS) {
    set_error("stev_integrate_static: n_cells = " + std::to_string((long long)n) + " is beyond STEV_STATIC_MAX_CELLS = " +
              std::to_string((long long)STEV_STATIC_MAX_CELLS) + " (the fixed scratch array holds one launch-order entry per cell); "
              "split the field or use stev_integrate with a caller-owned workspace");
    return STEV_EINVAL;
  }
  const bool ls_ok = (f32 ? (est ? est->ls32_ok : m->ls32_ok) : (est ? est->ls_ok : m->ls_ok)) && p->chunk_steps == 0;
  if (!ls_ok || !(p->lanes_per_cell == 0 || p->lanes_per_cell == 512 || p->lanes_per_cell == 513)) {
    set_error("stev_integrate_static runs the lock-step kernel only: chunk_steps = 0, lanes_per_cell 0 / 512 / 513, at most two "
              "factors per reaction side, integer coefficients, at most 64 species");
    return STEV_EINVAL;
  }
  g_stats = stev_stats{};
  g_stats.total_steps = -1;
  if (n == 0) return STEV_OK;
  if (!T || !pressure || !Y || !steps_out) { set_error("stev_integrate_static: null state pointer"); return STEV_EINVAL; }
  unsigned char *scratch = nullptr;
  if ((rc = static_scratch(&scratch))) return rc;
  int *counters = (int *)scratch;
  int *order_list = (int *)(scratch + kStaticCountersBytes);
  int *order_hist = (int *)(scratch + kStaticCountersBytes + kStaticOrderBytes);
  cudaStream_t s = (cudaStream_t)cuda_stream;
  // the array keeps the previous call's contents: the counters must start at zero; the launch order and its histogram
  // are rewritten in full by order_cells_launch before they are read
  STEV_CUDA(cudaMemsetAsync(counters, 0, kStaticCountersBytes, s));
  const int *order = nullptr;
  if (p->order_cells && n > 1) {
    rc = order_cells_launch(T, n, order_group(p->order_cells, n, tb->S), order_list, order_hist, s);
    if (rc) return rc;
    order = order_list;
  }
  int blocks = 0;
  size_t smem = 0;
  const stev::LsTables &ltb = f32 ? (est ? est->ls_tb32 : m->ls_tb32) : (est ? est->ls_tb : m->ls_tb);
  const unsigned char *ltable = f32 ? (est ? est->d_ls_table32 : m->d_ls_table32) : (est ? est->d_ls_table : m->d_ls_table);
  bool is_static = false;
  rc = integrate_ls_launch(ltb, ltable, make_consts(p), dt_cfd, n, ld, T, pressure, Y, steps_out, status_out, counters, s, &blocks,
                           &smem, order, p->lanes_per_cell != 513, &is_static);
  if (rc) return rc;
  g_stats.passes = 1;
  g_stats.specialised = is_static ? 1 : 0;
  g_stats.kernel_launches = 1 + (order ? 3 : 0);
  g_stats.blocks = blocks;
  g_stats.lanes_per_cell = p->lanes_per_cell == 513 ? 513 : 512;
  g_stats.threads_per_block = kLsThreads;
  g_stats.cells_per_block = ltb.d.C;
  g_stats.smem_bytes = (int64_t)smem;
  if (p->nonblocking) return STEV_OK;
  return finish_integrate(counters, s);
}

}  // extern "C"
