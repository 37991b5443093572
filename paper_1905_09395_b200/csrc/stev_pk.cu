// stev_pk.cu -- host side of the warp-pair integrator (stev_pk.cuh): table image, per-cell layout, launch.
#include <algorithm>
#include <cmath>
#include <cstring>
#include <numeric>

#include "stev_host.h"
#include "stev_pk_kernel.cuh"

namespace stev {

static int align_up(int x, int a) { return (x + a - 1) / a * a; }
static constexpr size_t kSmemMax = 227 * 1024;

// The pair kernel keeps at most two concentration factors per reaction side (total nu per side <= 2, so nu*g is exact
// for the equilibrium sum), 8 reversible reactions per TMEM lane (Rrev <= 256) and one species per lane (S <= 64).
static bool pk_mechanism_ok(const HostMechanism &m, int nw) {
  const int nw2 = std::min(nw, 2);   // species and gather lists live in at most two warps, histories in 256 TMEM columns
  if (m.has_real || m.S > 32 * nw2 || m.Rrev < 1 || m.Rrev > 16 * nw2 * kPkMaxIt) return false;
  for (int j = 0; j < m.R; ++j) {
    int nr = 0, np = 0;
    for (int e = m.reac_ptr[j]; e < m.reac_ptr[j + 1]; ++e) nr += m.reac_nu[e];
    for (int e = m.prod_ptr[j]; e < m.prod_ptr[j + 1]; ++e) np += m.prod_nu[e];
    if (nr > 2 || np > 2) return false;
  }
  return true;
}

static void pk_layout(const PkTables &tb, PkCell &cl) {
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
  cl.oRof = take(8 * tb.Rrev);
  cl.oHid = take(4 * (tb.has_est ? tb.H + align_up(tb.n_in, 4) : 0));   // hidden activations, then the normalised inputs
  cl.oSc = take((int)sizeof(PkScal));
  // an odd multiple of 16 bytes keeps the cells of different pairs on different bank groups for the broadcast loads
  cl.stride = align_up(o, 16);
  if ((cl.stride / 16) % 2 == 0) cl.stride += 16;
}

bool build_pk_image(const HostMechanism &m, const HostEstimator *e, int nw, std::vector<unsigned char> &image, PkTables &tb,
                    PkCell &cl) {
  if (nw < 1 || nw > 2 || !pk_mechanism_ok(m, nw)) return false;
  const int S = m.S, R = m.R, Rrev = m.Rrev;
  tb = PkTables{};
  tb.S = S;
  tb.R = R;
  tb.Rrev = Rrev;
  tb.n_it = (Rrev + 31) / 32;
  tb.Rp = (R + 1) & ~1;
  // DFT blocks: each warp keeps at most four blocks (128 TMEM columns); warp 0 takes the smaller half because it also
  // walks the two sequential sums of the temperature equation
  tb.nw = nw;
  tb.it_split[0] = 0;
  for (int h = 0; h < kPkMaxNw; ++h) {
    int cnt = 0;
    if (nw == 1) cnt = (h == 0) ? tb.n_it : 0;
    else cnt = (h == 0) ? tb.n_it / 2 : tb.n_it - tb.n_it / 2;
    tb.it_split[h + 1] = tb.it_split[h] + cnt;
  }
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
  // which the plain definition omega_i = sum_j nu_ij q_j adds them (same as the oracle's scatter, per species).
  // Entries name the caller's reaction index here; the internal index follows from the ordering chosen below.
  struct Ent { int j, coef; };
  std::vector<std::vector<Ent>> gl(S);
  const int variants[4] = {1, -1, 2, -2};   // stored multiples of q, fixed order
  bool has2 = false;
  auto variant_of = [&](int coef) {
    for (int v = 0; v < 4; ++v)
      if (variants[v] == coef) return v;
    return -1;
  };
  for (int j = 0; j < R; ++j) {
    for (int en = m.reac_ptr[j]; en < m.reac_ptr[j + 1]; ++en) gl[m.reac_sp[en]].push_back({j, -m.reac_nu[en]});
    for (int en = m.prod_ptr[j]; en < m.prod_ptr[j + 1]; ++en) gl[m.prod_sp[en]].push_back({j, m.prod_nu[en]});
  }
  for (auto &v : gl) {
    if (v.size() > 65535) return false;
    for (auto &en : v) {
      if (variant_of(en.coef) < 0) return false;
      has2 = has2 || en.coef == 2 || en.coef == -2;
    }
  }
  tb.n_var = has2 ? 4 : 2;
  pk_layout(tb, cl);

  // species -> (warp of the pair, lane): sorted by decreasing list length and dealt in groups of 16 lanes (one
  // shared-memory wavefront serves a half-warp), so that whole half-warps finish together and stop loading.  Warp 1
  // takes the two longest groups: warp 0 has the sequential sums of the temperature equation on top.
  std::vector<int> order(S);
  std::iota(order.begin(), order.end(), 0);
  std::stable_sort(order.begin(), order.end(), [&](int x, int y) { return gl[x].size() > gl[y].size(); });
  unsigned char gsp[32 * kPkMaxNw];
  unsigned short glen[32 * kPkMaxNw];
  std::memset(gsp, 255, sizeof(gsp));
  std::memset(glen, 0, sizeof(glen));
  int g_len[kPkMaxNw] = {0, 0};
  const int g_short = 0, g_long = 1;
  for (int n = 0; n < S; ++n) {
    const int group = n / 16;
    const int half = (nw >= 2) ? (group < 2 ? g_long : g_short) : 0, lane = (nw >= 2) ? (group & 1) * 16 + n % 16 : n;
    gsp[32 * half + lane] = (unsigned char)order[n];
    glen[32 * half + lane] = (unsigned short)gl[order[n]].size();
    g_len[half] = std::max(g_len[half], (int)gl[order[n]].size());
  }
  // rows of four entries, an even number per warp (the kernel walks two rows per trip) plus two spare rows that the
  // kernel prefetches past the end
  int g_rows = 0;
  for (int h = 0; h < kPkMaxNw; ++h) {
    tb.g_len4[h] = (g_len[h] + 7) / 8 * 2;
    tb.g_row0[h] = g_rows;
    g_rows += tb.g_len4[h];
  }
  g_rows += 2;

  // Internal reaction order: reversible reactions first (lanes never diverge on reversibility); within each group the
  // order is free, because every table is indexed through it.  It decides which shared-memory banks the lanes of a
  // half-warp hit in the rate loop (concentrations and g of the participants) and in the source-term gather (stored
  // multiples of q), so it is chosen by a short annealing run that minimises the modelled wavefront count.
  const unsigned one_slot = (unsigned)cl.oConc, zero_slot = (unsigned)cl.oG;
  std::vector<unsigned> fac_of(4 * (size_t)R), dg_of(4 * (size_t)R);
  std::vector<double> dnu_of(R);
  for (int j = 0; j < R; ++j) {
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
    dnu_of[j] = dnu;
    std::memcpy(&fac_of[4 * (size_t)j], fac, 16);
    std::memcpy(&dg_of[4 * (size_t)j], dgo, 16);
  }
  std::vector<int> orig_of(m.orig_of), internal_of(R);   // start: caller order within each group
  // modelled wavefronts of one 8-byte load by 16 lanes: the largest number of distinct addresses in one bank pair
  auto half_warp = [](const unsigned *addr, int n) {
    int cnt[16] = {0};
    unsigned seen[16][16];
    int worst = 0;
    for (int l = 0; l < n; ++l) {
      const unsigned a = addr[l], b = (a >> 3) & 15u;
      bool dup = false;
      for (int q = 0; q < cnt[b]; ++q) dup = dup || seen[b][q] == a;
      if (!dup) {
        seen[b][cnt[b]++] = a;
        worst = std::max(worst, cnt[b]);
      }
    }
    return worst;
  };
  auto modelled_wavefronts = [&]() {
    for (int k = 0; k < R; ++k) internal_of[orig_of[k]] = k;
    long long total = 0;
    unsigned addr[16];
    for (int half = 0; half < kPkMaxNw; ++half)     // gather: step e of the lists of one half-warp
      for (int hw = 0; hw < 2; ++hw)
        for (int e = 0;; ++e) {
          int n = 0;
          for (int l = 0; l < 16; ++l) {
            const int slot = 32 * half + 16 * hw + l, i = gsp[slot];
            if (i != 255 && e < (int)gl[i].size())
              addr[n++] = (unsigned)(cl.oQ + 8 * (variant_of(gl[i][e].coef) * tb.Rp + internal_of[gl[i][e].j]));
          }
          if (n == 0) break;
          total += half_warp(addr, n);
        }
    for (int k0 = 0; k0 < R; k0 += 16) {              // rate loop: participant loads of 16 consecutive reactions
      const int n = std::min(16, (k0 < Rrev ? Rrev : R) - k0);
      if (n <= 0) continue;
      for (int q = 0; q < 4; ++q) {
        if (k0 >= Rrev && q >= 2) break;              // irreversible: two reactant factors only
        for (int l = 0; l < n; ++l) addr[l] = fac_of[4 * (size_t)orig_of[k0 + l] + q];
        total += half_warp(addr, n);
        if (k0 < Rrev) {
          for (int l = 0; l < n; ++l) addr[l] = dg_of[4 * (size_t)orig_of[k0 + l] + q];
          total += half_warp(addr, n);
        }
      }
    }
    return total;
  };
  if (m.pk_order.size() == (size_t)R) {
    orig_of = m.pk_order;   // chosen once per mechanism (the estimator image reuses it)
  } else if (R >= 64) {
    unsigned long long rng = 0x9e3779b97f4a7c15ull;
    auto next = [&]() {
      rng ^= rng << 13;
      rng ^= rng >> 7;
      rng ^= rng << 17;
      return rng;
    };
    long long cur = modelled_wavefronts(), best = cur;
    std::vector<int> best_order = orig_of;
    double temp = 2.0;
    const int iters = 12000;
    for (int it = 0; it < iters; ++it, temp = std::max(0.05, temp * 0.9995)) {
      const bool in_rev = (Rrev >= 2) && (R - Rrev < 2 || next() % 4 != 0);
      const int lo = in_rev ? 0 : Rrev, cnt = in_rev ? Rrev : R - Rrev;
      if (cnt < 2) continue;
      const int x = lo + (int)(next() % (unsigned)cnt), y = lo + (int)(next() % (unsigned)cnt);
      if (x == y) continue;
      std::swap(orig_of[x], orig_of[y]);
      const long long c = modelled_wavefronts();
      const double u = (double)(next() >> 11) * (1.0 / 9007199254740992.0);
      if (c <= cur || u < std::exp(-(double)(c - cur) / temp)) {
        cur = c;
        if (c < best) {
          best = c;
          best_order = orig_of;
        }
      } else {
        std::swap(orig_of[x], orig_of[y]);
      }
    }
    orig_of = best_order;
  }
  m.pk_order = orig_of;
  for (int k = 0; k < R; ++k) internal_of[orig_of[k]] = k;

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
  tb.o_gsp = take(sizeof(gsp));
  tb.o_glen = take(sizeof(glen));
  tb.o_gent = take(16 * 32 * std::max(g_rows, 1));
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
  for (int k = 0; k < R; ++k) {
    const int j = orig_of[k];
    rkA[2 * k] = clog(m.A[j]);
    rkA[2 * k + 1] = m.b[j];
    rkB[2 * k] = m.Ea[j] / kRcal;
    rkB[2 * k + 1] = dnu_of[j];
    std::memcpy(rfac + 4 * k, &fac_of[4 * (size_t)j], 16);
    if (k < Rrev) std::memcpy(rdg + 4 * k, &dg_of[4 * (size_t)j], 16);
  }
  std::memcpy(base + tb.o_gsp, gsp, sizeof(gsp));
  std::memcpy(base + tb.o_glen, glen, sizeof(glen));
  unsigned *gent = (unsigned *)(base + tb.o_gent);   // [row][lane][4]
  for (int n = 0; n < 4 * 32 * g_rows; ++n) gent[n] = zero_slot;
  for (int half = 0, row0 = 0; half < kPkMaxNw; ++half) {
    for (int lane = 0; lane < 32; ++lane) {
      const int i = gsp[32 * half + lane];
      for (int en = 0; en < 4 * tb.g_len4[half]; ++en) {
        unsigned o = zero_slot;
        if (i != 255 && en < (int)gl[i].size()) o = (unsigned)(cl.oQ + 8 * (variant_of(gl[i][en].coef) * tb.Rp + internal_of[gl[i][en].j]));
        gent[((row0 + en / 4) * 32 + lane) * 4 + (en & 3)] = o;
      }
    }
    row0 += tb.g_len4[half];
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

// dense (one warp per cell only): 32 cells per block at 64 registers; needs at most two 32-blocks of reversible reactions
bool pk_dense_ok(const PkTables &tb) { return tb.nw == 1 && tb.n_it <= 2; }

int pk_cells_per_block(const PkTables &tb, const PkCell &cl, bool dense) {
  const size_t avail = kSmemMax - (size_t)tb.bytes - 256;
  const int cap = dense ? 4 * kPkMaxCells : (tb.nw == 1 ? 2 * kPkMaxCells : kPkMaxCells);
  return (int)std::min<size_t>(cap, avail / (size_t)cl.stride);
}

int integrate_pk_launch(const PkTables &tb, const PkCell &cl, const unsigned char *d_table, const SolverConsts &sc, double t_f,
                        long long n, long long ld, double *T, const double *p, double *Y, int *steps, unsigned char *status,
                        int *counters, cudaStream_t s, int *blocks_out, int *cells_per_block_out, size_t *smem_out, bool dense, const int *list) {
  if (dense && !pk_dense_ok(tb)) { set_error("dense tensor-memory kernel: more than 64 reversible reactions"); return STEV_EINVAL; }
  PkArgs a{};
  a.tb = tb;
  a.table = d_table;
  a.cl = cl;
  a.sc = sc;
  a.t_f = t_f;
  a.n_active = n;
  a.list = list;
  a.ld = ld;
  a.T = T;
  a.p = p;
  a.Y = Y;
  a.steps = steps;
  a.status = status;
  a.queue_head = counters;
  a.worst_status = counters + 1;
  a.cells_per_block = pk_cells_per_block(tb, cl, dense);
  if (a.cells_per_block < 1) { set_error("pair kernel: shared memory too small"); return STEV_EINVAL; }
  const size_t smem = (size_t)tb.bytes + (size_t)a.cells_per_block * cl.stride;
  void *fn = dense ? (void *)stev_pk_kernel<1, true> : (tb.nw == 2) ? (void *)stev_pk_kernel<2> : (void *)stev_pk_kernel<1>;
  const int threads = dense ? kPkThreads4 : kPkThreads;
  STEV_CUDA(cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  const long long blocks = std::min<long long>(device_sm_count(), (n + a.cells_per_block - 1) / a.cells_per_block);
  void *args[] = {&a};
  STEV_CUDA(cudaLaunchKernel(fn, dim3((unsigned)blocks), dim3(threads), args, smem, s));
  *blocks_out = (int)blocks;
  *cells_per_block_out = a.cells_per_block;
  *smem_out = smem;
  return STEV_OK;
}

}  // namespace stev
