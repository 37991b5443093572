// stev_ab.cu -- host side of the warp-specialised integrator (stev_ab.cuh): table image, per-cell layout, launch.
#include <algorithm>
#include <cstring>
#include <numeric>

#include "stev_ab_kernel.cuh"
#include "stev_host.h"

namespace stev {

static int align_up(int x, int a) { return (x + a - 1) / a * a; }
static constexpr size_t kSmemMax = 227 * 1024;

// The AB kernel's rate loop keeps at most two concentration factors per reaction side (total nu per side <= 2, so
// nu*g is exact for the equilibrium sum) and 8 reversible reactions per lane (Rrev <= 256).
static bool ab_mechanism_ok(const HostMechanism &m) {
  if (m.Rrev < 1 || m.Rrev > 32 * kAbMaxIt) return false;
  for (int j = 0; j < m.R; ++j) {
    int nr = 0, np = 0;
    for (int e = m.reac_ptr[j]; e < m.reac_ptr[j + 1]; ++e) nr += m.reac_nu[e];
    for (int e = m.prod_ptr[j]; e < m.prod_ptr[j + 1]; ++e) np += m.prod_nu[e];
    if (nr > 2 || np > 2) return false;
  }
  return true;
}

static void ab_layout(const AbTables &tb, AbCell &cl) {
  int o = 0;
  auto take = [&](int bytes) {
    int r = o;
    o = align_up(o + bytes, 16);
    return r;
  };
  cl.oYp = take(16 * tb.S);
  cl.oYwCp = take(16 * tb.S);
  cl.oHOm = take(16 * tb.S);
  cl.oConc = take(8 * (1 + tb.S));
  cl.oG = take(8 * (1 + 2 * tb.S));
  cl.oQ = take(8 * tb.n_var * tb.Rp);
  cl.oQraw = take(8 * tb.R);
  cl.oRof = take(8 * tb.Rrev);
  cl.oHid = take(4 * (tb.has_est ? tb.H : 0));
  cl.oCtrl = take((int)sizeof(AbCtrl));
  // an odd multiple of 16 bytes keeps the cells of different warps on different bank groups for the broadcast loads
  cl.stride = align_up(o, 16);
  if ((cl.stride / 16) % 2 == 0) cl.stride += 16;
}

bool build_ab_image(const HostMechanism &m, const HostEstimator *e, std::vector<unsigned char> &image, AbTables &tb, AbCell &cl) {
  if (!ab_mechanism_ok(m)) return false;
  const int S = m.S, R = m.R, Rrev = m.Rrev;
  tb = AbTables{};
  tb.S = S;
  tb.R = R;
  tb.Rrev = Rrev;
  tb.n_it = (Rrev + 31) / 32;
  tb.Rp = (R + 1) & ~1;
  if (e) {
    tb.has_est = 1;
    tb.H = e->H;
    tb.Hpad = e->H + 4;
    tb.n_in = e->n_in;
    tb.n_out = e->n_out;
    tb.act = e->act;
    tb.input_map = e->input_map;
    tb.h_ref_T = e->h_ref_T;
  }
  // per-species entry lists in the caller's reaction order, reactant entries before product entries: the order in
  // which the plain definition omega_i = sum_j nu_ij q_j adds them (same as the oracle's scatter, per species)
  struct Ent { int k, coef; };
  std::vector<std::vector<Ent>> gl(S);
  // stored multiples of q, fixed order: +1, -1 (always), +2, -2 (if any coefficient is +-2)
  const int variants[4] = {1, -1, 2, -2};
  bool has2 = false;
  auto variant_of = [&](int coef) {
    for (int v = 0; v < 4; ++v)
      if (variants[v] == coef) return v;
    return -1;
  };
  for (int j = 0; j < R; ++j) {
    for (int en = m.reac_ptr[j]; en < m.reac_ptr[j + 1]; ++en) gl[m.reac_sp[en]].push_back({m.internal_of[j], -m.reac_nu[en]});
    for (int en = m.prod_ptr[j]; en < m.prod_ptr[j + 1]; ++en) gl[m.prod_sp[en]].push_back({m.internal_of[j], m.prod_nu[en]});
  }
  for (auto &v : gl)
    for (auto &en : v) {
      if (variant_of(en.coef) < 0) return false;
      has2 = has2 || en.coef == 2 || en.coef == -2;
    }
  tb.n_var = has2 ? 4 : 2;
  ab_layout(tb, cl);

  // species -> (round, lane): the 32 longest lists in round 0, the rest in round 1 (each round is as long as its
  // longest list; shorter lists are padded with the 0.0 slot)
  std::vector<int> order(S);
  std::iota(order.begin(), order.end(), 0);
  std::stable_sort(order.begin(), order.end(), [&](int x, int y) { return gl[x].size() > gl[y].size(); });
  if (S > 64) return false;
  unsigned char gsp[64];
  std::memset(gsp, 255, sizeof(gsp));
  tb.g_len[0] = tb.g_len[1] = 0;
  for (int n = 0; n < S; ++n) {
    const int round = n / 32, lane = n % 32;
    gsp[32 * round + lane] = (unsigned char)order[n];
    tb.g_len[round] = std::max(tb.g_len[round], (int)gl[order[n]].size());
  }
  const int g_total = tb.g_len[0] + tb.g_len[1];

  int off = 0;
  auto take = [&](int bytes) {
    int o = off;
    off = align_up(off + bytes, 16);
    return o;
  };
  tb.o_tmid = take(8 * S);
  tb.o_W = take(8 * S);
  tb.o_invW = take(8 * S);
  tb.o_nasa = take(8 * 2 * kNasaRows * S);
  tb.o_rkA = take(16 * R);
  tb.o_rkB = take(16 * R);
  tb.o_rfac = take(16 * R);
  tb.o_rdg = take(16 * Rrev);
  tb.o_gsp = take(64);
  tb.o_gent = take(2 * 32 * std::max(g_total, 1));
  if (e) {
    tb.o_eshift = take(4 * e->n_in);
    tb.o_escale = take(4 * e->n_in);
    tb.o_W1T = take(4 * e->n_in * e->H);
    tb.o_b1 = take(4 * e->H);
    tb.o_W2p = take(4 * e->n_out * tb.Hpad);
    tb.o_b2 = take(4 * e->n_out);
  }
  tb.bytes = align_up(off, 128);
  if ((size_t)tb.bytes + (size_t)cl.stride + 256 > kSmemMax) return false;
  if (cl.oQ + 8 * tb.n_var * tb.Rp > 65535 || cl.oG > 65535) return false;   // 16-bit entry offsets

  image.assign(tb.bytes, 0);
  unsigned char *base = image.data();
  double *tmid = (double *)(base + tb.o_tmid), *W = (double *)(base + tb.o_W), *invW = (double *)(base + tb.o_invW);
  double *nasa = (double *)(base + tb.o_nasa);
  for (int i = 0; i < S; ++i) {
    tmid[i] = m.t_mid[i];
    W[i] = m.W[i];
    invW[i] = 1.0 / m.W[i];
    for (int rg = 0; rg < 2; ++rg) {
      const double *c = (rg == 0 ? m.nasa_lo.data() : m.nasa_hi.data()) + 7 * i;
      double *row = nasa + rg * kNasaRows * S + i;
      row[0 * S] = c[0]; row[1 * S] = c[1]; row[2 * S] = c[2]; row[3 * S] = c[3]; row[4 * S] = c[4];
      row[5 * S] = c[1] / 2.0; row[6 * S] = c[2] / 3.0; row[7 * S] = c[3] / 4.0; row[8 * S] = c[4] / 5.0;
      row[9 * S] = c[5];
      row[10 * S] = c[2] / 2.0; row[11 * S] = c[3] / 3.0; row[12 * S] = c[4] / 4.0;
      row[13 * S] = c[6];
    }
  }
  double *rkA = (double *)(base + tb.o_rkA), *rkB = (double *)(base + tb.o_rkB);
  unsigned *rfac = (unsigned *)(base + tb.o_rfac), *rdg = (unsigned *)(base + tb.o_rdg);
  const unsigned one_slot = (unsigned)cl.oConc, zero_slot = (unsigned)cl.oG;
  for (int k = 0; k < R; ++k) {
    const int j = m.orig_of[k];
    rkA[2 * k] = clog(m.A[j]);
    rkA[2 * k + 1] = m.b[j];
    rkB[2 * k] = m.Ea[j] / kRcal;
    double dnu = 0.0;
    unsigned fac[4] = {one_slot, one_slot, one_slot, one_slot};
    unsigned dgo[4] = {zero_slot, zero_slot, zero_slot, zero_slot};
    int nf = 0, ne = 0;
    for (int en = m.reac_ptr[j]; en < m.reac_ptr[j + 1]; ++en, ++ne) {
      for (int n = 0; n < m.reac_nu[en]; ++n) fac[nf++] = (unsigned)(cl.oConc + 8 * (1 + m.reac_sp[en]));
      dgo[ne] = (unsigned)(cl.oG + 8 * (1 + (m.reac_nu[en] == 2 ? S : 0) + m.reac_sp[en]));
      dnu = dnu - (double)m.reac_nu[en];
    }
    nf = 2;
    ne = 2;
    for (int en = m.prod_ptr[j]; en < m.prod_ptr[j + 1]; ++en, ++ne) {
      for (int n = 0; n < m.prod_nu[en]; ++n) fac[nf++] = (unsigned)(cl.oConc + 8 * (1 + m.prod_sp[en]));
      dgo[ne] = (unsigned)(cl.oG + 8 * (1 + (m.prod_nu[en] == 2 ? S : 0) + m.prod_sp[en]));
      dnu = dnu + (double)m.prod_nu[en];
    }
    rkB[2 * k + 1] = dnu;
    std::memcpy(rfac + 4 * k, fac, 16);
    if (k < Rrev) std::memcpy(rdg + 4 * k, dgo, 16);
  }
  std::memcpy(base + tb.o_gsp, gsp, 64);
  unsigned short *gent = (unsigned short *)(base + tb.o_gent);
  for (int round = 0, row0 = 0; round < 2; ++round) {
    for (int lane = 0; lane < 32; ++lane) {
      const int i = gsp[32 * round + lane];
      for (int en = 0; en < tb.g_len[round]; ++en) {
        unsigned o = zero_slot;
        if (i != 255 && en < (int)gl[i].size()) o = (unsigned)(cl.oQ + 8 * (variant_of(gl[i][en].coef) * tb.Rp + gl[i][en].k));
        gent[(row0 + en) * 32 + lane] = (unsigned short)o;
      }
    }
    row0 += tb.g_len[round];
  }
  if (e) {
    float *sh = (float *)(base + tb.o_eshift), *sc = (float *)(base + tb.o_escale), *W1T = (float *)(base + tb.o_W1T);
    float *b1 = (float *)(base + tb.o_b1), *W2p = (float *)(base + tb.o_W2p), *b2 = (float *)(base + tb.o_b2);
    for (int k = 0; k < e->n_in; ++k) {
      sh[k] = e->in_shift[k];
      sc[k] = e->in_scale[k];
      for (int jh = 0; jh < e->H; ++jh) W1T[k * e->H + jh] = e->W1[(size_t)jh * e->n_in + k];
    }
    for (int jh = 0; jh < e->H; ++jh) b1[jh] = e->b1[jh];
    for (int o = 0; o < e->n_out; ++o) {
      b2[o] = e->b2[o];
      for (int jh = 0; jh < e->H; ++jh) W2p[(size_t)o * tb.Hpad + jh] = e->W2[(size_t)o * e->H + jh];
    }
  }
  return true;
}

int ab_cells_per_block(const AbTables &tb, const AbCell &cl) {
  const size_t avail = kSmemMax - (size_t)tb.bytes - 256;
  return (int)std::min<size_t>(kAbMaxCells, avail / (size_t)cl.stride);
}

int integrate_ab_launch(const AbTables &tb, const AbCell &cl, const unsigned char *d_table, const SolverConsts &sc, double t_f,
                        long long n, long long ld, double *T, const double *p, double *Y, int *steps, unsigned char *status,
                        int *counters, cudaStream_t s, int *blocks_out, int *cells_per_block_out, size_t *smem_out) {
  AbArgs a{};
  a.tb = tb;
  a.table = d_table;
  a.cl = cl;
  a.sc = sc;
  a.t_f = t_f;
  a.n_active = n;
  a.list = nullptr;
  a.ld = ld;
  a.T = T;
  a.p = p;
  a.Y = Y;
  a.steps = steps;
  a.status = status;
  a.queue_head = counters;
  a.worst_status = counters + 1;
  a.cells_per_block = ab_cells_per_block(tb, cl);
  if (a.cells_per_block < 1) { set_error("AB kernel: shared memory too small"); return STEV_EINVAL; }
  const size_t smem = (size_t)tb.bytes + (size_t)a.cells_per_block * cl.stride;
  STEV_CUDA(cudaFuncSetAttribute(stev_ab_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  const long long blocks = std::min<long long>(device_sm_count(), (n + a.cells_per_block - 1) / a.cells_per_block);
  void *args[] = {&a};
  STEV_CUDA(cudaLaunchKernel((void *)stev_ab_kernel, dim3((unsigned)blocks), dim3(kAbThreads), args, smem, s));
  *blocks_out = (int)blocks;
  *cells_per_block_out = a.cells_per_block;
  *smem_out = smem;
  return STEV_OK;
}

}  // namespace stev
