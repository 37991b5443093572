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
//      tanh / ex2) and writes the hidden activations back to TENSOR MEMORY with tcgen05.st (TF32: in place over D1),
//      where they are the A operand of layer 2 (tcgen05.mma with A from TMEM: no shared-memory round trip);
//   4. layer-2 MMAs (D2: 128 x Np), then the epilogue adds b2 in fp32, stages the rows in shared memory and one TMA
//      bulk store writes the tile (a ragged last tile is read and written row by row).
// BF16 keeps only 8 mantissa bits, which alone would put the result at the edge of the 1e-2 tolerance, so on that
// path both contractions are compensated: a = a_hi + a_lo and w = w_hi + w_lo (all BF16) and the K axis carries the
// three products a_hi w_hi + a_lo w_hi + a_hi w_lo side by side (the tensor cores have an order of magnitude of slack).
// The weights are rounded once on the host (TF32: round-to-nearest of the 10-bit mantissa; BF16: round-to-nearest-
// even), laid out in the same canonical layout and copied to shared memory once per CTA.  The tiles of a CTA are
// software-pipelined (layer-2 MMAs of a tile against the input conversion of the next, layer-1 MMAs of the next tile
// against the output staging of this one) and several CTAs share an SM; the op is HBM-bound (config 4: 88 B in +
// 160 B out per cell).
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
  int lbo_a1, lbo_w1, lbo_w2;    // byte distance between K-adjacent core matrices
  int o_a1;                      // shared-memory offset of the layer-1 A operand
  int o_xs, o_os;                // staging of one raw input tile (TMA bulk load) and one output tile (TMA bulk store)
  int blk1;                      // BF16: columns per block of the layer-1 K axis (n_in rounded up to 8); TF32: unused
  int a2col;                     // TMEM column of the layer-2 A operand (hidden activations): 0 = in place over D1
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

// Round-to-nearest (ties away) to TF32 for finite values: add half an ulp of the 10-bit mantissa; the tensor core
// ignores the 13 low bits.  (cvt.rna.tf32.f32 is a three-instruction sequence in SASS; this is one integer add.)
__device__ __forceinline__ uint32_t to_tf32(float x) { return __float_as_uint(x) + 0x1000u; }
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

__device__ __forceinline__ void tmem_st16(uint32_t taddr, const uint32_t (&r)[16]) {
  asm volatile(
      "tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16};" ::"r"(taddr),
      "r"(r[0]), "r"(r[1]), "r"(r[2]), "r"(r[3]), "r"(r[4]), "r"(r[5]), "r"(r[6]), "r"(r[7]), "r"(r[8]), "r"(r[9]), "r"(r[10]),
      "r"(r[11]), "r"(r[12]), "r"(r[13]), "r"(r[14]), "r"(r[15])
      : "memory");
}
__device__ __forceinline__ void tmem_st8(uint32_t taddr, const uint32_t (&r)[8]) {
  asm volatile("tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};" ::"r"(taddr), "r"(r[0]), "r"(r[1]),
               "r"(r[2]), "r"(r[3]), "r"(r[4]), "r"(r[5]), "r"(r[6]), "r"(r[7])
               : "memory");
}

// A operand from tensor memory (row = TMEM lane, K along the columns: one TF32 or two BF16 per column)
template <bool BF16>
__device__ __forceinline__ void mma_ts(uint32_t d_tmem, uint32_t a_tmem, uint64_t b_desc, uint32_t idesc, uint32_t accumulate) {
  if (BF16) {
    asm volatile(
        "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::1.kind::f16 [%0], [%1], %2, %3, p;\n\t}"
        ::"r"(d_tmem), "r"(a_tmem), "l"(b_desc), "r"(idesc), "r"(accumulate)
        : "memory");
  } else {
    asm volatile(
        "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::1.kind::tf32 [%0], [%1], %2, %3, p;\n\t}"
        ::"r"(d_tmem), "r"(a_tmem), "l"(b_desc), "r"(idesc), "r"(accumulate)
        : "memory");
  }
}

template <bool BF16>
__global__ void __launch_bounds__(kTcThreads) estimator_tc_kernel(const __grid_constant__ TcArgs a) {
  extern __shared__ __align__(128) unsigned char smem[];
  __shared__ unsigned long long mbar1, mbar2, mbar_x;
  __shared__ uint32_t tmem_base_s;
  const int t = threadIdx.x, warp = t >> 5;

  // weights, biases, normalisation constants: one copy per CTA
  for (int i = t * 16; i < a.im.bytes; i += kTcThreads * 16) *(uint4 *)(smem + i) = *(const uint4 *)(a.image + i);
  // zero the layer-1 A operand once: its K padding columns are never written afterwards
  for (int i = a.o_a1 + t * 16; i < a.o_xs; i += kTcThreads * 16) *(uint4 *)(smem + i) = make_uint4(0, 0, 0, 0);
  if (t == 0) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(smem_u32(&mbar1)));
    asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(smem_u32(&mbar2)));
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
  // D1 [128 x Hp] at column 0, D2 [128 x Np] at column Hp, hidden A operand at a2col (TF32: in place over D1)
  const uint32_t d1 = tmem_base, d2 = tmem_base + (uint32_t)a.Hp, ta2 = tmem_base + (uint32_t)a.a2col;
  const uint32_t my_lane = (uint32_t)(warp * 32) << 16;

  const float *shift = (const float *)(smem + a.im.o_shift), *scale = (const float *)(smem + a.im.o_scale);
  const float *b1 = (const float *)(smem + a.im.o_b1), *b2 = (const float *)(smem + a.im.o_b2);
  unsigned char *A1 = smem + a.o_a1;
  const uint32_t sA1 = smem_u32(A1), sW1 = smem_u32(smem + a.im.o_w1), sW2 = smem_u32(smem + a.im.o_w2);
  const int n_in = a.n_in;
  uint32_t parity1 = 0, parity2 = 0, parity_x = 0;
  float *Xs = (float *)(smem + a.o_xs), *Os = (float *)(smem + a.o_os);
  const int tile_in_bytes = kTcRows * n_in * 4, tile_out_bytes = kTcRows * a.n_out * 4;
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
  // 1. inputs of a tile: thread t owns row t.  fp32 normalisation, operand rounding, one 16-byte core-matrix row per
  //    store (conflict-free: consecutive rows are contiguous).  A ragged last tile is first copied into the staging.
  auto convert = [&](long long tile) {
    const long long row0 = tile * kTcRows;
    const int rows = (int)((a.n - row0 < kTcRows) ? (a.n - row0) : kTcRows);
    if (rows == kTcRows) {
      mbar_wait(&mbar_x, parity_x);
      parity_x ^= 1;
    } else {
      const float *Xt = a.X + row0 * n_in;
      for (int e = t; e < kTcRows * n_in; e += kTcThreads) Xs[e] = (e < rows * n_in) ? Xt[e] : 0.f;
      __syncthreads();
    }
    const float *xrow = Xs + t * n_in;
    unsigned char *arow = A1 + t * 16;
    if (BF16) {
      const int nb = a.blk1 / 8;   // 16-byte chunks per column block [a_hi | a_lo | a_hi]
      for (int kc = 0; kc < nb; ++kc) {
        uint32_t hi[4], lo[4];
#pragma unroll
        for (int q = 0; q < 4; ++q) {
          const int c = 8 * kc + 2 * q;
          const float x0 = (c < n_in) ? (xrow[c] - shift[c]) * scale[c] : 0.f;
          const float x1 = (c + 1 < n_in) ? (xrow[c + 1] - shift[c + 1]) * scale[c + 1] : 0.f;
          hi[q] = pack_bf16(x0, x1);
          lo[q] = pack_bf16(x0 - __uint_as_float(hi[q] << 16), x1 - __uint_as_float(hi[q] & 0xffff0000u));
        }
        const uint4 whi = make_uint4(hi[0], hi[1], hi[2], hi[3]), wlo = make_uint4(lo[0], lo[1], lo[2], lo[3]);
        *(uint4 *)(arow + kc * a.lbo_a1) = whi;
        *(uint4 *)(arow + (nb + kc) * a.lbo_a1) = wlo;
        *(uint4 *)(arow + (2 * nb + kc) * a.lbo_a1) = whi;
      }
    } else {
      for (int kc = 0; kc < a.K1 / 4; ++kc) {
        uint32_t w[4];
#pragma unroll
        for (int q = 0; q < 4; ++q) {
          const int c = 4 * kc + q;
          w[q] = (c < n_in) ? to_tf32((xrow[c] - shift[c]) * scale[c]) : 0u;
        }
        *(uint4 *)(arow + kc * a.lbo_a1) = make_uint4(w[0], w[1], w[2], w[3]);
      }
    }
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // generic-proxy writes -> visible to the tensor core
  };
  // 2. layer 1: D1[128 x Hp] = A1[128 x K1] * W1^T (one elected thread)
  auto issue_mma1 = [&]() {
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    const int ksteps = a.K1 / a.kstep_elems;
    for (int ks = 0; ks < ksteps; ++ks) {
      const uint64_t da = make_desc(sA1 + ks * 2 * a.lbo_a1, a.lbo_a1, 128);
      const uint64_t db = make_desc(sW1 + ks * 2 * a.lbo_w1, a.lbo_w1, 128);
      mma_ss<BF16>(d1, da, db, a.idesc1, ks > 0);
    }
    mma_commit(&mbar1);
  };
  // 4. layer 2: D2[128 x Np] = hidden[128 x K2] * W2^T, A operand from tensor memory
  auto issue_mma2 = [&]() {
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    const int ksteps = a.K2 / a.kstep_elems;
    for (int ks = 0; ks < ksteps; ++ks) {
      const uint64_t db = make_desc(sW2 + ks * 2 * a.lbo_w2, a.lbo_w2, 128);
      mma_ts<BF16>(d2, ta2 + ks * 8, db, a.idesc2, ks > 0);   // 32 bytes of K = 8 columns per instruction
    }
    mma_commit(&mbar2);
  };

  // Software pipeline over the tiles of this CTA: the layer-2 MMAs of a tile run while the inputs of the next tile are
  // converted, the layer-1 MMAs of the next tile run while the outputs of this tile are staged.
  long long tile = blockIdx.x;
  if (tile < n_tiles) {
    if (t == 0) prefetch(tile);
    convert(tile);
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    if (t == 0) {
      prefetch(tile + gridDim.x);
      issue_mma1();
    }
  }
  for (; tile < n_tiles; tile += gridDim.x) {
    const long long row0 = tile * kTcRows, next = tile + gridDim.x;
    const int rows = (int)((a.n - row0 < kTcRows) ? (a.n - row0) : kTcRows);
    const bool full = rows == kTcRows, has_next = next < n_tiles;
    // ---- 3. epilogue 1: bias + activation in fp32; the hidden activations go back to tensor memory as the A operand
    mbar_wait(&mbar1, parity1);
    parity1 ^= 1;
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    for (int c0 = 0; c0 < a.Hp; c0 += 16) {
      uint32_t v[16];
      tmem_ld16(d1 + my_lane + c0, v);
      float h[16];
#pragma unroll
      for (int g = 0; g < 4; ++g) {
        const float4 bv = *(const float4 *)(b1 + c0 + 4 * g);
        h[4 * g + 0] = activation(__uint_as_float(v[4 * g + 0]) + bv.x, a.act);
        h[4 * g + 1] = activation(__uint_as_float(v[4 * g + 1]) + bv.y, a.act);
        h[4 * g + 2] = activation(__uint_as_float(v[4 * g + 2]) + bv.z, a.act);
        h[4 * g + 3] = activation(__uint_as_float(v[4 * g + 3]) + bv.w, a.act);
      }
      if (BF16) {
        uint32_t hi[8], lo[8];
#pragma unroll
        for (int q = 0; q < 8; ++q) {
          hi[q] = pack_bf16(h[2 * q], h[2 * q + 1]);
          lo[q] = pack_bf16(h[2 * q] - __uint_as_float(hi[q] << 16), h[2 * q + 1] - __uint_as_float(hi[q] & 0xffff0000u));
        }
        const uint32_t col = ta2 + my_lane + c0 / 2, blk = a.Hp / 2;   // column blocks [a_hi | a_lo | a_hi]
        tmem_st8(col, hi);
        tmem_st8(col + blk, lo);
        tmem_st8(col + 2 * blk, hi);
      } else {
#pragma unroll
        for (int i = 0; i < 16; ++i) v[i] = to_tf32(h[i]);
        tmem_st16(ta2 + my_lane + c0, v);
      }
    }
    asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    if (t == 0) issue_mma2();
    // ---- inputs of the next tile while the layer-2 MMAs run
    if (has_next) convert(next);
    mbar_wait(&mbar2, parity2);
    parity2 ^= 1;
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    // the previous tile's bulk store must have finished reading the output staging
    if (t == 0) asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();   // A1 of the next tile is complete; D1 / the hidden operand and the staging buffers are free
    if (t == 0 && has_next) {
      prefetch(next + gridDim.x);
      issue_mma1();
    }
    // ---- epilogue 2 (while the layer-1 MMAs of the next tile run): bias in fp32; a full tile is staged in shared
    //      memory and leaves by one TMA bulk store, a ragged last tile is written row by row
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
              const float4 bv = *(const float4 *)(b2 + c);
              float4 o;
              o.x = __uint_as_float(v[4 * g + 0]) + bv.x;
              o.y = __uint_as_float(v[4 * g + 1]) + bv.y;
              o.z = __uint_as_float(v[4 * g + 2]) + bv.z;
              o.w = __uint_as_float(v[4 * g + 3]) + bv.w;
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
    __syncthreads();   // the output tile is complete in shared memory; D2 is free again
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
  a.blk1 = round_up(h.n_in, 8);
  a.K1 = bf16 ? round_up(3 * a.blk1, 16) : round_up(h.n_in, 8);
  a.K2 = (bf16 ? 3 : 1) * a.Hp;
  a.Np = round_up(h.n_out, 16);
  if (a.Hp > 256 || a.Np > 256) return false;
  // +16 bytes on the K-chunk stride of the A operands staggers the banks of the column-wise input writes
  a.lbo_a1 = kTcRows * 16 + 16;
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
  a.o_xs = take(kTcRows * h.n_in * 4);
  a.o_os = take(kTcRows * h.n_out * 4);
  p.smem = (size_t)off;
  if (p.smem > 200 * 1024) return false;
  a.idesc1 = make_idesc(bf16, kTcRows, a.Hp);
  a.idesc2 = make_idesc(bf16, kTcRows, a.Np);
  // tensor-memory columns: D1 [Hp] | D2 [Np] | hidden A operand (TF32: Hp columns, in place over D1 once a thread has
  // read its row; compensated BF16: three blocks of Hp / 2 columns after D2)
  const int a2_cols = a.K2 * a.esize / 4;
  a.a2col = (a2_cols <= a.Hp) ? 0 : a.Hp + a.Np;
  int cols = 32;
  while (cols < std::max(a.Hp + a.Np, a.a2col + a2_cols)) cols *= 2;
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
    for (int k = 0; k < h.n_in; ++k) put_w(a.im.o_w1, a.lbo_w1, j, k, a.blk1, h.W1[(size_t)j * h.n_in + k]);
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
