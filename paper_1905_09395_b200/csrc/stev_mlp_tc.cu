// stev_mlp_tc.cu -- tensor-core path of the standalone estimator forward pass (row a7 of DESIGN.md section 1;
// PAPER.md:120-136, Fig 2: one hidden layer, linear output; PAPER.md:136 projects the tensor-core speed-up).
//
//   hidden = act(Xn W1^T + b1),  out = hidden W2^T + b2,   Xn = (X - shift) * scale        (include/stev.h)
//
// Both contractions run on the 5th-generation tensor cores: tcgen05.mma (kind::tf32, or kind::f16 with BF16
// operands), M = 128 cells per instruction, fp32 accumulators in tensor memory.  One CTA of 128 threads owns a tile of
// 128 cells: thread t is cell row t and TMEM lane t.  Per tile
//   1. the raw input tile arrives by one TMA bulk copy (cp.async.bulk on an mbarrier, issued one tile ahead), is
//      normalised in fp32, rounded to the operand type and written to shared memory in the canonical K-major
//      core-matrix layout (8 rows x 16 bytes per core matrix, no swizzle);
//   2. one elected thread issues the layer-1 MMAs (accumulator D1: 128 x Hp in TMEM) and commits to an mbarrier;
//   3. every thread reads its row of D1 with tcgen05.ld, adds the bias in fp32, applies the activation (MUFU
//      tanh / ex2) and writes the hidden activations back to shared memory as the A operand of layer 2;
//   4. layer-2 MMAs (D2: 128 x Np), then the epilogue adds b2 in fp32, stages the rows in shared memory and one TMA
//      bulk store writes the tile (a ragged last tile is read and written row by row).
// BF16 keeps only 8 mantissa bits, which alone would put the result at the edge of the 1e-2 tolerance, so on that
// path both contractions are compensated: a = a_hi + a_lo and w = w_hi + w_lo (all BF16) and the K axis carries the
// three products a_hi w_hi + a_lo w_hi + a_hi w_lo side by side (the tensor cores have an order of magnitude of slack).
// The weights are rounded once on the host (TF32: round-to-nearest of the 10-bit mantissa; BF16: round-to-nearest-
// even), laid out in the same canonical layout and copied to shared memory once per CTA.  Several CTAs per SM overlap
// each other's load, MMA and epilogue phases; the op is HBM-bound (config 4: 88 B in + 160 B out per cell).
#include <algorithm>
#include <cstring>
#include <vector>

#include "stev_host.h"

namespace stev {

namespace {

constexpr int kTcRows = 128;     // cells per tile = UMMA M
constexpr int kTcThreads = 128;

struct TcImage {                 // offsets (bytes) into the device/shared weight image
  int o_w1, o_w2, o_b1, o_b2, o_shift, o_scale, bytes;
};

struct TcArgs {
  const unsigned char *image;
  TcImage im;
  int n_in, K1, K2, H, Hp, n_out, Np, act;   // K1, K2: padded contraction lengths of the two layers
  int esize;                     // operand element size: 4 (TF32) or 2 (BF16)
  int kstep_elems;               // K elements per MMA: 8 (TF32) or 16 (BF16) = 32 bytes
  int lbo_a1, lbo_a2, lbo_w1, lbo_w2;   // byte distance between K-adjacent core matrices
  int o_a1, o_a2;                // shared-memory offsets of the two A operands
  int o_xs, o_os;                // staging of one raw input tile (TMA bulk load) and one output tile (TMA bulk store;
                                 // aliases A2 when it fits: A2 is dead once the layer-2 MMAs have completed)
  uint32_t idesc1, idesc2;
  int tmem_cols;
  const float *X;
  float *out;
  long long n;
};

__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

// Shared-memory matrix descriptor (no swizzle, K-major): start address, LBO (K direction), SBO (M/N direction, 8 rows
// = 128 bytes), version 1 (sm_100).
__device__ __forceinline__ uint64_t make_desc(uint32_t saddr, uint32_t lbo_bytes, uint32_t sbo_bytes) {
  uint64_t d = 0;
  d |= (uint64_t)((saddr & 0x3ffffu) >> 4);
  d |= (uint64_t)((lbo_bytes >> 4) & 0x3fffu) << 16;
  d |= (uint64_t)((sbo_bytes >> 4) & 0x3fffu) << 32;
  d |= (uint64_t)1 << 46;
  return d;
}

template <bool BF16>
__device__ __forceinline__ void mma_ss(uint32_t d_tmem, uint64_t a_desc, uint64_t b_desc, uint32_t idesc, uint32_t accumulate) {
  if (BF16) {
    asm volatile(
        "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t}"
        ::"r"(d_tmem), "l"(a_desc), "l"(b_desc), "r"(idesc), "r"(accumulate)
        : "memory");
  } else {
    asm volatile(
        "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::1.kind::tf32 [%0], %1, %2, %3, p;\n\t}"
        ::"r"(d_tmem), "l"(a_desc), "l"(b_desc), "r"(idesc), "r"(accumulate)
        : "memory");
  }
}

__device__ __forceinline__ void mma_commit(unsigned long long *mbar) {
  asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(mbar)) : "memory");
}

__device__ __forceinline__ void mbar_wait(unsigned long long *mbar, uint32_t parity) {
  const uint32_t a = smem_u32(mbar);
  uint32_t done = 0;
  while (!done) {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(done)
        : "r"(a), "r"(parity)
        : "memory");
  }
}

__device__ __forceinline__ void tmem_ld16(uint32_t taddr, uint32_t (&r)[16]) {
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
      : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]), "=r"(r[9]),
        "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
      : "r"(taddr)
      : "memory");
  asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
}

__device__ __forceinline__ uint32_t to_tf32(float x) {
  uint32_t r;
  asm("cvt.rna.tf32.f32 %0, %1;" : "=r"(r) : "f"(x));
  return r;
}
__device__ __forceinline__ uint32_t pack_bf16(float lo, float hi) {
  uint32_t r;
  asm("cvt.rn.bf16x2.f32 %0, %1, %2;" : "=r"(r) : "f"(hi), "f"(lo));
  return r;
}
__device__ __forceinline__ unsigned short to_bf16(float x) { return (unsigned short)(pack_bf16(x, 0.f) & 0xffffu); }

__device__ __forceinline__ float activation(float z, int act) {
  float a;
  if (act == STEV_ACT_TANH) {
    asm("tanh.approx.f32 %0, %1;" : "=f"(a) : "f"(z));
  } else {
    float e;
    asm("ex2.approx.f32 %0, %1;" : "=f"(e) : "f"(-1.4426950408889634f * z));
    asm("rcp.approx.f32 %0, %1;" : "=f"(a) : "f"(1.0f + e));
  }
  return a;
}

// Byte offset of element (row r, column c) of a K-major operand in the canonical no-swizzle layout used here:
// core matrix = 8 rows x 16 bytes, rows of one 16-byte K chunk are contiguous (SBO = 128), K chunks `lbo` apart.
__device__ __forceinline__ int canon_off(int r, int c, int esize, int lbo) {
  const int per = 16 / esize;
  return (c / per) * lbo + r * 16 + (c % per) * esize;
}

template <bool BF16>
__global__ void __launch_bounds__(kTcThreads) estimator_tc_kernel(const __grid_constant__ TcArgs a) {
  extern __shared__ __align__(128) unsigned char smem[];
  __shared__ unsigned long long mbar, mbar_x;
  __shared__ uint32_t tmem_base_s;
  const int t = threadIdx.x, warp = t >> 5;

  // weights, biases, normalisation constants: one copy per CTA
  for (int i = t * 16; i < a.im.bytes; i += kTcThreads * 16) *(uint4 *)(smem + i) = *(const uint4 *)(a.image + i);
  // zero both A operands once: the K padding columns are never written afterwards
  for (int i = a.o_a1 + t * 16; i < a.o_a2 + a.lbo_a2 * (a.K2 * a.esize / 16); i += kTcThreads * 16) *(uint4 *)(smem + i) = make_uint4(0, 0, 0, 0);
  if (t == 0) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(smem_u32(&mbar)));
    asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(smem_u32(&mbar_x)));
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (warp == 0) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(&tmem_base_s)), "r"(a.tmem_cols) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  __syncthreads();
  asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
  const uint32_t tmem_base = tmem_base_s;
  const uint32_t d1 = tmem_base, d2 = tmem_base + (uint32_t)a.Hp;
  const uint32_t my_lane = (uint32_t)(warp * 32) << 16;

  const float *shift = (const float *)(smem + a.im.o_shift), *scale = (const float *)(smem + a.im.o_scale);
  const float *b1 = (const float *)(smem + a.im.o_b1), *b2 = (const float *)(smem + a.im.o_b2);
  unsigned char *A1 = smem + a.o_a1, *A2 = smem + a.o_a2;
  const uint32_t sA1 = smem_u32(A1), sA2 = smem_u32(A2), sW1 = smem_u32(smem + a.im.o_w1), sW2 = smem_u32(smem + a.im.o_w2);
  const int n_in = a.n_in;
  uint32_t parity = 0, parity_x = 0;
  float *Xs = (float *)(smem + a.o_xs), *Os = (float *)(smem + a.o_os);
  const int tile_in_bytes = kTcRows * n_in * 4, tile_out_bytes = kTcRows * a.n_out * 4;
  const int r_first = t / n_in, c_first = t - r_first * n_in, r_step = kTcThreads / n_in, c_step = kTcThreads - r_step * n_in;

  const long long n_tiles = (a.n + kTcRows - 1) / kTcRows;
  // raw input tiles arrive by TMA bulk copy (one instruction per tile, signalled on mbar_x), one tile ahead
  auto prefetch = [&](long long tile) {
    if (tile < n_tiles && (tile + 1) * kTcRows <= a.n) {
      const uint32_t mb = smem_u32(&mbar_x);
      asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(mb), "r"(tile_in_bytes) : "memory");
      asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(Xs)),
                   "l"(a.X + tile * kTcRows * n_in), "r"(tile_in_bytes), "r"(mb)
                   : "memory");
    }
  };
  if (t == 0) prefetch(blockIdx.x);
  for (long long tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
    const long long row0 = tile * kTcRows;
    const int rows = (int)((a.n - row0 < kTcRows) ? (a.n - row0) : kTcRows);
    const bool full = rows == kTcRows;
    // ---- 1. inputs: fp32 normalisation, operand rounding, canonical layout (a ragged last tile is read directly)
    const float *Xt = a.X + row0 * n_in;
    if (full) {
      mbar_wait(&mbar_x, parity_x);
      parity_x ^= 1;
      Xt = Xs;
    }
    for (int e = t, r = r_first, c = c_first; e < kTcRows * n_in; e += kTcThreads) {
      const float x = (r < rows) ? (Xt[e] - shift[c]) * scale[c] : 0.f;
      if (BF16) {
        const unsigned short hi = to_bf16(x);
        const unsigned short lo = to_bf16(x - __uint_as_float((uint32_t)hi << 16));
        *(unsigned short *)(A1 + canon_off(r, c, 2, a.lbo_a1)) = hi;
        *(unsigned short *)(A1 + canon_off(r, n_in + c, 2, a.lbo_a1)) = lo;
        *(unsigned short *)(A1 + canon_off(r, 2 * n_in + c, 2, a.lbo_a1)) = hi;
      } else {
        *(uint32_t *)(A1 + canon_off(r, c, 4, a.lbo_a1)) = to_tf32(x);
      }
      r += r_step;
      c += c_step;
      if (c >= n_in) {
        c -= n_in;
        r += 1;
      }
    }
    // the previous tile's bulk store must have finished reading the output staging (it may alias A2)
    if (t == 0) asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // generic-proxy writes -> visible to the tensor core
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    // ---- 2. layer 1: D1[128 x Hp] = A1[128 x K1] * W1^T
    if (t == 0) {
      prefetch(tile + gridDim.x);   // the staging buffer is free: every thread has converted its part
      asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
      const int ksteps = a.K1 / a.kstep_elems;
      for (int ks = 0; ks < ksteps; ++ks) {
        const uint64_t da = make_desc(sA1 + ks * 2 * a.lbo_a1, a.lbo_a1, 128);
        const uint64_t db = make_desc(sW1 + ks * 2 * a.lbo_w1, a.lbo_w1, 128);
        mma_ss<BF16>(d1, da, db, a.idesc1, ks > 0);
      }
      mma_commit(&mbar);
    }
    mbar_wait(&mbar, parity);
    parity ^= 1;
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    // ---- 3. epilogue 1: bias + activation in fp32, hidden activations become the A operand of layer 2
    for (int c0 = 0; c0 < a.Hp; c0 += 16) {
      uint32_t v[16];
      tmem_ld16(d1 + my_lane + c0, v);
      float h[16];
#pragma unroll
      for (int i = 0; i < 16; ++i) h[i] = activation(__uint_as_float(v[i]) + b1[c0 + i], a.act);
      if (BF16) {
#pragma unroll
        for (int g = 0; g < 2; ++g) {
          uint32_t hi[4], lo[4];
#pragma unroll
          for (int q = 0; q < 4; ++q) {
            const float x0 = h[8 * g + 2 * q], x1 = h[8 * g + 2 * q + 1];
            hi[q] = pack_bf16(x0, x1);
            lo[q] = pack_bf16(x0 - __uint_as_float(hi[q] << 16), x1 - __uint_as_float(hi[q] & 0xffff0000u));
          }
          const uint4 whi = make_uint4(hi[0], hi[1], hi[2], hi[3]), wlo = make_uint4(lo[0], lo[1], lo[2], lo[3]);
          const int kc = (c0 + 8 * g) / 8, blk = a.Hp / 8;
          *(uint4 *)(A2 + kc * a.lbo_a2 + t * 16) = whi;
          *(uint4 *)(A2 + (blk + kc) * a.lbo_a2 + t * 16) = wlo;
          *(uint4 *)(A2 + (2 * blk + kc) * a.lbo_a2 + t * 16) = whi;
        }
      } else {
#pragma unroll
        for (int g = 0; g < 4; ++g) {
          uint4 w;
          w.x = to_tf32(h[4 * g + 0]);
          w.y = to_tf32(h[4 * g + 1]);
          w.z = to_tf32(h[4 * g + 2]);
          w.w = to_tf32(h[4 * g + 3]);
          *(uint4 *)(A2 + ((c0 + 4 * g) / 4) * a.lbo_a2 + t * 16) = w;
        }
      }
    }
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    // ---- 4. layer 2: D2[128 x Np] = A2[128 x Hp] * W2^T
    if (t == 0) {
      asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
      const int ksteps = a.K2 / a.kstep_elems;
      for (int ks = 0; ks < ksteps; ++ks) {
        const uint64_t da = make_desc(sA2 + ks * 2 * a.lbo_a2, a.lbo_a2, 128);
        const uint64_t db = make_desc(sW2 + ks * 2 * a.lbo_w2, a.lbo_w2, 128);
        mma_ss<BF16>(d2, da, db, a.idesc2, ks > 0);
      }
      mma_commit(&mbar);
    }
    mbar_wait(&mbar, parity);
    parity ^= 1;
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    // ---- epilogue 2: bias in fp32; a full tile is staged in shared memory and leaves by one TMA bulk store, a ragged
    //      last tile is written row by row
    float *orow = full ? (Os + t * a.n_out) : (a.out + (row0 + t) * a.n_out);
    const bool vec = (a.n_out % 4) == 0;
    for (int c0 = 0; c0 < a.Np; c0 += 16) {
      uint32_t v[16];
      tmem_ld16(d2 + my_lane + c0, v);
      if (t < rows) {
        if (vec) {
#pragma unroll
          for (int g = 0; g < 4; ++g) {
            const int c = c0 + 4 * g;
            if (c < a.n_out) {
              float4 o;
              o.x = __uint_as_float(v[4 * g + 0]) + b2[c + 0];
              o.y = __uint_as_float(v[4 * g + 1]) + b2[c + 1];
              o.z = __uint_as_float(v[4 * g + 2]) + b2[c + 2];
              o.w = __uint_as_float(v[4 * g + 3]) + b2[c + 3];
              *(float4 *)(orow + c) = o;
            }
          }
        } else {
#pragma unroll
          for (int i = 0; i < 16; ++i)
            if (c0 + i < a.n_out) orow[c0 + i] = __uint_as_float(v[i]) + b2[c0 + i];
        }
      }
    }
    if (full) asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();   // D1, D2, A1 are free again; the output tile is complete in shared memory
    if (full && t == 0) {
      asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(a.out + row0 * a.n_out), "r"(smem_u32(Os)),
                   "r"(tile_out_bytes)
                   : "memory");
      asm volatile("cp.async.bulk.commit_group;" ::: "memory");
    }
  }
  if (t == 0) asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  __syncthreads();
  if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "r"(a.tmem_cols) : "memory");
}

// ---- host side ------------------------------------------------------------------------------------------
int round_up(int x, int m) { return (x + m - 1) / m * m; }

uint32_t host_tf32(float x) {   // cvt.rna.tf32.f32: round to nearest, ties away, 10 explicit mantissa bits
  uint32_t u;
  std::memcpy(&u, &x, 4);
  if ((u & 0x7f800000u) == 0x7f800000u) return u;
  return (u + 0x1000u) & 0xffffe000u;
}
unsigned short host_bf16(float x) {   // round to nearest even
  uint32_t u;
  std::memcpy(&u, &x, 4);
  if ((u & 0x7f800000u) == 0x7f800000u) return (unsigned short)(u >> 16);
  return (unsigned short)((u + 0x7fffu + ((u >> 16) & 1u)) >> 16);
}

uint32_t make_idesc(bool bf16, int M, int N) {
  const uint32_t fmt = bf16 ? 1u : 2u;   // F16F32Format: BF16 = 1, TF32 = 2
  uint32_t d = 0;
  d |= 1u << 4;               // accumulator format F32
  d |= fmt << 7;              // A format
  d |= fmt << 10;             // B format
  // bits 13-16: no negation, A and B K-major
  d |= (uint32_t)(N >> 3) << 17;
  d |= (uint32_t)(M >> 4) << 24;
  return d;
}

struct TcPlan {
  TcArgs args{};
  size_t smem = 0;
  std::vector<unsigned char> image;
};

// Lays out weights (rounded to the operand type) and constants; returns false if the network does not fit.
bool make_plan(const HostEstimator &h, bool bf16, TcPlan &p) {
  TcArgs &a = p.args;
  a.esize = bf16 ? 2 : 4;
  a.kstep_elems = bf16 ? 16 : 8;
  a.n_in = h.n_in;
  a.H = h.H;
  a.n_out = h.n_out;
  a.act = h.act;
  a.Hp = round_up(h.H, 16);
  a.K1 = round_up((bf16 ? 3 : 1) * h.n_in, a.kstep_elems);
  a.K2 = (bf16 ? 3 : 1) * a.Hp;
  a.Np = round_up(h.n_out, 16);
  if (a.Hp > 256 || a.Np > 256) return false;
  // +16 bytes on the K-chunk stride of the A operands staggers the banks of the column-wise input writes
  a.lbo_a1 = kTcRows * 16 + 16;
  a.lbo_a2 = kTcRows * 16;
  a.lbo_w1 = a.Hp * 16;
  a.lbo_w2 = a.Np * 16;
  const int per = 16 / a.esize;
  int off = 0;
  auto take = [&](int bytes) {
    int o = off;
    off = round_up(off + bytes, 128);
    return o;
  };
  a.im.o_w1 = take(a.lbo_w1 * (a.K1 / per));
  a.im.o_w2 = take(a.lbo_w2 * (a.K2 / per));
  a.im.o_b1 = take(4 * a.Hp);
  a.im.o_b2 = take(4 * a.Np);
  a.im.o_shift = take(4 * h.n_in);
  a.im.o_scale = take(4 * h.n_in);
  a.im.bytes = off;
  a.o_a1 = take(a.lbo_a1 * (a.K1 / per));
  const int a2_bytes = a.lbo_a2 * (a.K2 / per);
  a.o_a2 = take(a2_bytes);
  a.o_xs = take(kTcRows * h.n_in * 4);
  a.o_os = (kTcRows * h.n_out * 4 <= a2_bytes) ? a.o_a2 : take(kTcRows * h.n_out * 4);
  p.smem = (size_t)off;
  if (p.smem > 200 * 1024) return false;
  a.idesc1 = make_idesc(bf16, kTcRows, a.Hp);
  a.idesc2 = make_idesc(bf16, kTcRows, a.Np);
  int cols = 32;
  while (cols < a.Hp + a.Np) cols *= 2;
  if (cols > 512) return false;
  a.tmem_cols = cols;

  p.image.assign(a.im.bytes, 0);
  unsigned char *base = p.image.data();
  auto put = [&](unsigned char *dst, float v) {
    if (bf16) { unsigned short b = host_bf16(v); std::memcpy(dst, &b, 2); }
    else { uint32_t b = host_tf32(v); std::memcpy(dst, &b, 4); }
  };
  auto canon = [&](int r, int c, int lbo) { return (c / per) * lbo + r * 16 + (c % per) * a.esize; };
  auto bf16_value = [&](float v) {
    const uint32_t u = (uint32_t)host_bf16(v) << 16;
    float f;
    std::memcpy(&f, &u, 4);
    return f;
  };
  // TF32: one column per input.  BF16: column blocks [a_hi w_hi | a_lo w_hi | a_hi w_lo] (w_lo = bf16(w - w_hi)).
  auto put_w = [&](int o_w, int lbo, int row, int col, int block, float w) {
    if (!bf16) { put(base + o_w + canon(row, col, lbo), w); return; }
    const float w_hi = bf16_value(w);
    put(base + o_w + canon(row, col, lbo), w_hi);
    put(base + o_w + canon(row, block + col, lbo), w_hi);
    put(base + o_w + canon(row, 2 * block + col, lbo), w - w_hi);
  };
  for (int j = 0; j < h.H; ++j)
    for (int k = 0; k < h.n_in; ++k) put_w(a.im.o_w1, a.lbo_w1, j, k, h.n_in, h.W1[(size_t)j * h.n_in + k]);
  for (int o = 0; o < h.n_out; ++o)
    for (int j = 0; j < h.H; ++j) put_w(a.im.o_w2, a.lbo_w2, o, j, a.Hp, h.W2[(size_t)o * h.H + j]);
  std::memcpy(base + a.im.o_b1, h.b1.data(), 4 * h.H);
  std::memcpy(base + a.im.o_b2, h.b2.data(), 4 * h.n_out);
  std::memcpy(base + a.im.o_shift, h.in_shift.data(), 4 * h.n_in);
  std::memcpy(base + a.im.o_scale, h.in_scale.data(), 4 * h.n_in);
  return true;
}

}  // namespace

// Builds (once per estimator and precision) the device weight image; called from stev_estimator_load.
int estimator_tensor_prepare(stev_estimator *e) {
  for (int prec = 0; prec < 2; ++prec) {
    TcPlan plan;
    e->tc_ok[prec] = make_plan(e->host, prec == 1, plan);
    if (!e->tc_ok[prec]) continue;
    STEV_CUDA(cudaMalloc(&e->d_tc_image[prec], plan.image.size()));
    STEV_CUDA(cudaMemcpy(e->d_tc_image[prec], plan.image.data(), plan.image.size(), cudaMemcpyHostToDevice));
  }
  return STEV_OK;
}

int estimator_eval_tensor(const stev_estimator *e, long long n, const float *X, float *out, int precision, cudaStream_t s) {
  const bool bf16 = precision == STEV_PREC_BF16;
  const int prec = bf16 ? 1 : 0;
  if (!e->tc_ok[prec] || !e->d_tc_image[prec]) {
    set_error("stev_estimator_eval: network too large for the tensor-core path (hidden and output widths <= 256, shared memory <= 200 KB)");
    return STEV_EINVAL;
  }
  TcPlan plan;
  make_plan(e->host, bf16, plan);   // host-side arithmetic only (offsets); the image itself is already on the device
  TcArgs a = plan.args;
  a.image = e->d_tc_image[prec];
  a.X = X;
  a.out = out;
  a.n = n;
  const void *fn = bf16 ? (const void *)estimator_tc_kernel<true> : (const void *)estimator_tc_kernel<false>;
  STEV_CUDA(cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)plan.smem));
  // CTAs per SM: bounded by shared memory, tensor-memory columns (512 per SM) and 2048 threads
  int per_sm = (int)std::min<size_t>((227 * 1024) / (plan.smem + 1024), (size_t)(512 / a.tmem_cols));
  per_sm = std::max(1, std::min(per_sm, 8));
  const long long tiles = (n + kTcRows - 1) / kTcRows;
  const long long blocks = std::min<long long>(tiles, (long long)device_sm_count() * per_sm);
  void *args[] = {&a};
  STEV_CUDA(cudaLaunchKernel(fn, dim3((unsigned)blocks), dim3(kTcThreads), args, plan.smem, s));
  STEV_CUDA(cudaGetLastError());
  return STEV_OK;
}

}  // namespace stev
