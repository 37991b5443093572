// stev_ls.cu -- host side of the lock-step integrator (stev_ls.cuh): table image, per-cell layout, launch.
#include <algorithm>
#include <cmath>
#include <cstring>
#include <numeric>

#include "stev_host.h"
#include "stev_ls_kernel.cuh"

namespace stev {

static int align_up(int x, int a) { return (x + a - 1) / a * a; }
static constexpr size_t kSmemMax = 227 * 1024;

static unsigned magic(int d) { return d <= 1 ? 0u : (unsigned)(((1ull << 32) + (unsigned)d - 1) / (unsigned)d); }

// At most two concentration factors per reaction side (total nu per side <= 2, so nu*g is exact for the equilibrium sum
// and the stored multiples +-q, +-2q cover every coefficient) and one byte per species index.
static bool ls_mechanism_ok(const HostMechanism &m) {
  if (m.has_real || m.S > 64 || m.R > STEV_MAX_REACTIONS) return false;
  for (int j = 0; j < m.R; ++j) {
    int nr = 0, np = 0;
    for (int e = m.reac_ptr[j]; e < m.reac_ptr[j + 1]; ++e) nr += m.reac_nu[e];
    for (int e = m.prod_ptr[j]; e < m.prod_ptr[j + 1]; ++e) np += m.prod_nu[e];
    if (nr > 2 || np > 2) return false;
  }
  return true;
}

bool build_ls_image(const HostMechanism &m, const HostEstimator *e, std::vector<unsigned char> &image, LsTables &tb, bool f32) {
  if (!ls_mechanism_ok(m)) return false;
  const int es = f32 ? 4 : 8;
  const int S = m.S, R = m.R, Rrev = m.Rrev;
  tb = LsTables{};
  LsDims &d = tb.d;
  d.S = S;
  d.R = R;
  d.Rrev = Rrev;
  d.es = es;
  if (e) {
    d.has_est = 1;
    d.H = e->H;
    d.n_in = e->n_in;
    d.n_out = e->n_out;
    tb.act = e->act;
    tb.input_map = e->input_map;
    tb.h_ref_T = e->h_ref_T;
  }
  // per-species entry lists in the caller's reaction order, reactant entries before product entries: the order in
  // which the plain definition omega_i = sum_j nu_ij q_j adds them (same as the oracle's scatter, per species)
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
  for (auto &v : gl)
    for (auto &en : v) {
      if (variant_of(en.coef) < 0) return false;
      has2 = has2 || en.coef == 2 || en.coef == -2;
    }
  d.n_var = has2 ? 4 : 2;
  d.C = 1;
  LsLayout L = ls_layout_of(d);   // table offsets do not depend on C

  // internal reaction order: reversible first; within each group the caller's order, re-paired below once C is known
  std::vector<int> orig_of = m.orig_of, internal_of(R);

  // species sorted by decreasing list length: a warp of phase 3 holds a few neighbouring ranks (times all cells), so its
  // lanes walk lists of nearly equal length
  std::vector<int> rank(S);
  std::iota(rank.begin(), rank.end(), 0);
  std::stable_sort(rank.begin(), rank.end(), [&](int x, int y) { return gl[x].size() > gl[y].size(); });
  int g_rows = 0;
  std::vector<int> row0(S), rows(S);
  for (int r = 0; r < S; ++r) {
    row0[r] = g_rows;
    rows[r] = ((int)gl[rank[r]].size() + 3) / 4;
    g_rows += rows[r];
  }
  if (g_rows + 1 > 65535) return false;
  tb.g_zero_row = g_rows;

  tb.bytes = align_up(L.o_gent + 16 * (g_rows + 1), 128);

  // cell slots per block: one lane of the scalar warp each, 2048 DFT windows in tensor memory, shared memory
  const size_t avail = kSmemMax > (size_t)tb.bytes + 1024 ? kSmemMax - (size_t)tb.bytes - 1024 : 0;
  int C = kLsMaxCells;
  if (Rrev > 0) C = std::min(C, (32 * ls_max_passes(es)) / Rrev);
  for (; C >= 1; --C) {
    d.C = C;
    L = ls_layout_of(d);
    if ((size_t)L.cell_bytes <= avail) break;
  }
  if (C < 1) return false;
  // When C divides 32 a lane holds the same cell in every pass and the kernel loads that cell's scalars once per step
  // (+5 % on config 3); worth up to an eighth of the cell slots (17 -> 16, 9 -> 8).
  for (int dv = 16; dv >= 2; dv >>= 1)
    if (C > dv && C < 2 * dv && (C - dv) * 8 <= C) {
      C = dv;
      d.C = C;
      L = ls_layout_of(d);
    }
  // When a row of the working set (C reals of one species) is 64 bytes -- 8 cells in binary64, 16 in binary32 -- the
  // lanes that issue one shared-memory access together hold TWO consecutive reactions, and their two rows are served in
  // one wavefront only if they lie in different halves of the 128-byte bank line, i.e. if the row indices differ by an
  // odd number.  Consecutive internal indices (2m, 2m + 1) are therefore chosen so that as many as possible of the
  // eight rows a rate pass reads (two + two concentration factors, two + two nu g terms) have opposite parity.  Any
  // internal order is valid: every table is indexed through it and the source terms are summed in the caller's order.
  if (es * C == 64) {
    auto rows_of = [&](int j, int (&row)[8]) {
      for (int n = 0; n < 8; ++n) row[n] = 0;   // the 1.0 slot / the 0.0 slot
      int nf = 0, ne = 4;
      for (int en = m.reac_ptr[j]; en < m.reac_ptr[j + 1]; ++en, ++ne) {
        for (int n = 0; n < m.reac_nu[en]; ++n) row[nf++] = 1 + m.reac_sp[en];
        row[ne] = 1 + (m.reac_nu[en] == 2 ? S : 0) + m.reac_sp[en];
      }
      nf = 2;
      ne = 6;
      for (int en = m.prod_ptr[j]; en < m.prod_ptr[j + 1]; ++en, ++ne) {
        for (int n = 0; n < m.prod_nu[en]; ++n) row[nf++] = 1 + m.prod_sp[en];
        row[ne] = 1 + (m.prod_nu[en] == 2 ? S : 0) + m.prod_sp[en];
      }
    };
    auto pair_up = [&](int lo, int hi, int n_slots) {   // greedy matching inside orig_of[lo, hi)
      std::vector<int> in(orig_of.begin() + lo, orig_of.begin() + hi), out;
      std::vector<char> used(in.size(), 0);
      for (size_t x = 0; x < in.size(); ++x) {
        if (used[x]) continue;
        used[x] = 1;
        out.push_back(in[x]);
        int ra[8], rb[8], best = -1, best_cost = 1 << 30;
        rows_of(in[x], ra);
        for (size_t y = x + 1; y < in.size(); ++y) {
          if (used[y]) continue;
          rows_of(in[y], rb);
          int cost = 0;
          for (int n = 0; n < n_slots; ++n) cost += ((ra[n] - rb[n]) & 1) ? 0 : 1;
          if (cost < best_cost) {
            best_cost = cost;
            best = (int)y;
          }
        }
        if (best >= 0) {
          used[best] = 1;
          out.push_back(in[best]);
        }
      }
      std::copy(out.begin(), out.end(), orig_of.begin() + lo);
    };
    pair_up(0, Rrev, 8);
    pair_up(Rrev, R, 2);   // an irreversible pass reads only its two reactant factors
  }
  for (int k = 0; k < R; ++k) internal_of[orig_of[k]] = k;
  {
    // irreversible passes dealt by rate work: a reversible pass (two exponentials, the equilibrium sum, evaluated two
    // passes side by side) counts three, an irreversible one (one exponential, one at a time) two; each pass goes to
    // the warp with the least work so far, then every warp takes a contiguous range
    const int n_rev_pass = L.n_rev_pass, n_irr_pass = L.n_irr_pass, PW = kLsPassWarps, NW = kLsWarps;
    if (n_irr_pass > 255) return false;
    int load[16] = {}, cnt[16] = {};
    for (int r = 0; r < PW; ++r) load[r] = 3 * ((n_rev_pass - r + PW - 1) / PW);
    for (int p = 0; p < n_irr_pass; ++p) {
      int best = NW - 1;   // ties go to the scalar warp first, then to the highest ranks (the warps with one reversible pass less)
      for (int r = NW - 2; r >= 0; --r)
        if (load[r] < load[best]) best = r;
      load[best] += 2;
      cnt[best] += 1;
    }
    int start = 0;
    for (int r = 0; r < NW; ++r) {
      tb.irr_start[r] = (unsigned char)start;
      tb.irr_count[r] = (unsigned char)cnt[r];
      start += cnt[r];
    }
  }

  image.assign(tb.bytes, 0);
  unsigned char *base = image.data();
  // every real table entry is formed in double and stored as double or, for the binary32 image, rounded to float once
  auto put = [&](int off0, int idx, double v) {
    if (f32) ((float *)(base + off0))[idx] = (float)v;
    else ((double *)(base + off0))[idx] = v;
  };
  for (int i = 0; i < S; ++i) {
    put(L.o_tmid, i, m.t_mid[i]);
    put(L.o_W, i, m.W[i]);
    put(L.o_invW, i, 1.0 / m.W[i]);
    for (int rg = 0; rg < 2; ++rg) {
      const double *c = (rg == 0 ? m.nasa_lo.data() : m.nasa_hi.data()) + 7 * i;
      const int r0 = rg * kNasaRows * S + i;
      put(L.o_nasa, r0 + 0 * S, c[0]); put(L.o_nasa, r0 + 1 * S, c[1]); put(L.o_nasa, r0 + 2 * S, c[2]);
      put(L.o_nasa, r0 + 3 * S, c[3]); put(L.o_nasa, r0 + 4 * S, c[4]);
      put(L.o_nasa, r0 + 5 * S, c[1] / 2.0); put(L.o_nasa, r0 + 6 * S, c[2] / 3.0); put(L.o_nasa, r0 + 7 * S, c[3] / 4.0);
      put(L.o_nasa, r0 + 8 * S, c[4] / 5.0);
      put(L.o_nasa, r0 + 9 * S, c[5]);
      put(L.o_nasa, r0 + 10 * S, c[2] / 2.0); put(L.o_nasa, r0 + 11 * S, c[3] / 3.0); put(L.o_nasa, r0 + 12 * S, c[4] / 4.0);
      put(L.o_nasa, r0 + 13 * S, c[6]);
    }
  }
  const unsigned one_slot = (unsigned)L.oConc, zero_slot = (unsigned)L.oG;
  unsigned *rfac = (unsigned *)(base + L.o_rfac), *rdg = (unsigned *)(base + L.o_rdg);
  for (int k = 0; k < R; ++k) {
    const int j = orig_of[k];
    double dnu = 0.0;
    float dnu32 = 0.0f;   // Delta-nu summed in the precision of the image, in entry order (as the oracle sums it)
    unsigned fac[4] = {one_slot, one_slot, one_slot, one_slot};
    unsigned dgo[4] = {zero_slot, zero_slot, zero_slot, zero_slot};
    int nf = 0, ne = 0;
    for (int en = m.reac_ptr[j]; en < m.reac_ptr[j + 1]; ++en, ++ne) {
      for (int n = 0; n < m.reac_nu[en]; ++n) fac[nf++] = (unsigned)(L.oConc + es * C * (1 + m.reac_sp[en]));
      dgo[ne] = (unsigned)(L.oG + es * C * (1 + (m.reac_nu[en] == 2 ? S : 0) + m.reac_sp[en]));
      dnu = dnu - (double)m.reac_nu[en];
      dnu32 = dnu32 - (float)m.reac_nu[en];
    }
    nf = 2;
    ne = 2;
    for (int en = m.prod_ptr[j]; en < m.prod_ptr[j + 1]; ++en, ++ne) {
      for (int n = 0; n < m.prod_nu[en]; ++n) fac[nf++] = (unsigned)(L.oConc + es * C * (1 + m.prod_sp[en]));
      dgo[ne] = (unsigned)(L.oG + es * C * (1 + (m.prod_nu[en] == 2 ? S : 0) + m.prod_sp[en]));
      dnu = dnu + (double)m.prod_nu[en];
      dnu32 = dnu32 + (float)m.prod_nu[en];
    }
    put(L.o_rkA, 2 * k, clog(m.A[j]));
    put(L.o_rkA, 2 * k + 1, m.b[j]);
    put(L.o_rkB, 2 * k, m.Ea[j] / kRcal);
    put(L.o_rkB, 2 * k + 1, f32 ? (double)dnu32 : dnu);
    // top bit of the fourth offset: some species has a coefficient of 2 in this reaction, i.e. the doubled multiples
    // +2q, -2q are read by a gather list (the rate passes store them only then)
    bool uses2 = false;
    for (int en = m.reac_ptr[j]; en < m.reac_ptr[j + 1]; ++en) uses2 = uses2 || m.reac_nu[en] == 2;
    for (int en = m.prod_ptr[j]; en < m.prod_ptr[j + 1]; ++en) uses2 = uses2 || m.prod_nu[en] == 2;
    if (uses2) fac[3] |= 0x80000000u;
    std::memcpy(rfac + 4 * k, fac, 16);
    if (k < Rrev) std::memcpy(rdg + 4 * k, dgo, 16);
  }
  unsigned char *gsp = base + L.o_gsp;
  unsigned short *grow = (unsigned short *)(base + L.o_grow), *glen = (unsigned short *)(base + L.o_glen);
  unsigned *gent = (unsigned *)(base + L.o_gent);
  for (int n = 0; n < 4 * (g_rows + 1); ++n) gent[n] = zero_slot;
  for (int r = 0; r < S; ++r) {
    const int i = rank[r];
    gsp[r] = (unsigned char)i;
    grow[r] = (unsigned short)row0[r];
    glen[r] = (unsigned short)rows[r];
    for (int en = 0; en < (int)gl[i].size(); ++en)
      gent[4 * row0[r] + en] = (unsigned)(L.oQ + es * C * (variant_of(gl[i][en].coef) * L.Rp + internal_of[gl[i][en].j]));
  }
  if (e) {
    float *sh = (float *)(base + L.o_eshift), *scl = (float *)(base + L.o_escale), *W1T = (float *)(base + L.o_W1T);
    float *b1 = (float *)(base + L.o_b1), *W2p = (float *)(base + L.o_W2p), *b2 = (float *)(base + L.o_b2);
    for (int k = 0; k < e->n_in; ++k) {
      sh[k] = e->in_shift[k];
      scl[k] = e->in_scale[k];
      for (int jh = 0; jh < e->H; ++jh) W1T[k * e->H + jh] = e->W1[(size_t)jh * e->n_in + k];
    }
    for (int jh = 0; jh < e->H; ++jh) b1[jh] = e->b1[jh];
    for (int o = 0; o < e->n_out; ++o) {
      b2[o] = e->b2[o];
      for (int jh = 0; jh < e->H; ++jh) W2p[(size_t)o * L.Hpad + jh] = e->W2[(size_t)o * e->H + jh];
    }
  }
  return true;
}

// ---------------------------------------------------------------------------------------------------------
// Shape list: mechanisms whose dimensions match an entry run the instantiation with compile-time dimensions, every
// other mechanism runs the same kernel with the dimensions read at run time.  The entries are the shapes of the five
// benchmark configurations of BASELINE.json (S, R, R_rev, stored multiples, estimator, H, n_in, n_out, C).
// ---------------------------------------------------------------------------------------------------------
using LsShape0 = LsFix<3, 2, 1, 2, 0, 0, 0, 0, 32>;
using LsShape1 = LsFix<9, 19, 11, 4, 0, 0, 0, 0, 32>;
using LsShape2 = LsFix<20, 60, 42, 4, 0, 0, 0, 0, 32>;
using LsShape3 = LsFix<53, 325, 225, 4, 1, 32, 1, 106, 8>;
using LsShape4 = LsFix<20, 60, 42, 4, 1, 64, 22, 40, 32>;
using LsShape3f = LsFix<53, 325, 225, 4, 1, 32, 1, 106, 16, 4>;   // config 3 with the binary32 state: 16 cells per block (17 fit)
using LsShape4f = LsFix<20, 60, 42, 4, 1, 64, 22, 40, 32, 4>;

static bool same_dims(const LsDims &x, const LsDims &y) {
  return x.S == y.S && x.R == y.R && x.Rrev == y.Rrev && x.n_var == y.n_var && x.has_est == y.has_est && x.H == y.H &&
         x.n_in == y.n_in && x.n_out == y.n_out && x.C == y.C && x.es == y.es;
}

static void *ls_kernel_for(const LsDims &d, bool allow_static, bool *is_static) {
  *is_static = true;
  if (allow_static) {
    if (same_dims(d, LsShape0::D)) return (void *)stev_ls_kernel<LsShape0, false, double>;
    if (same_dims(d, LsShape1::D)) return (void *)stev_ls_kernel<LsShape1, false, double>;
    if (same_dims(d, LsShape2::D)) return (void *)stev_ls_kernel<LsShape2, false, double>;
    if (same_dims(d, LsShape3::D)) return (void *)stev_ls_kernel<LsShape3, true, double>;
    if (same_dims(d, LsShape4::D)) return (void *)stev_ls_kernel<LsShape4, true, double>;
    if (same_dims(d, LsShape3f::D)) return (void *)stev_ls_kernel<LsShape3f, true, float>;
    if (same_dims(d, LsShape4f::D)) return (void *)stev_ls_kernel<LsShape4f, true, float>;
  }
  *is_static = false;
  if (d.es == 4) return d.has_est ? (void *)stev_ls_kernel<LsDyn, true, float> : (void *)stev_ls_kernel<LsDyn, false, float>;
  return d.has_est ? (void *)stev_ls_kernel<LsDyn, true, double> : (void *)stev_ls_kernel<LsDyn, false, double>;
}

int integrate_ls_launch(const LsTables &tb, const unsigned char *d_table, const SolverConsts &sc, double t_f, long long n,
                        long long ld, double *T, const double *p, double *Y, int *steps, unsigned char *status, int *counters,
                        cudaStream_t s, int *blocks_out, size_t *smem_out, const int *list, bool allow_static, bool *is_static) {
  LsArgs a{};
  a.tb = tb;
  a.lay = ls_layout_of(tb.d);
  a.mC = magic(tb.d.C);
  a.table = d_table;
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
  const size_t smem = (size_t)tb.bytes + (size_t)a.lay.cell_bytes;
  void *fn = ls_kernel_for(tb.d, allow_static, is_static);
  STEV_CUDA(cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  const long long blocks = std::min<long long>(device_sm_count(), (n + tb.d.C - 1) / tb.d.C);
  void *args[] = {&a};
  STEV_CUDA(cudaLaunchKernel(fn, dim3((unsigned)blocks), dim3(kLsThreads), args, smem, s));
  *blocks_out = (int)blocks;
  *smem_out = smem;
  return STEV_OK;
}

}  // namespace stev
