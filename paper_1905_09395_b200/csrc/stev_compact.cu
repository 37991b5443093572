// stev_compact.cu -- variable-load retirement between passes (row a6): the cells still active after
// a pass are gathered, order preserved, into the next pass's active list.  Warp ballot + popc inside a warp,
// a shared-memory scan across the warps of a block, and a grid-level exclusive prefix sum of the block totals.
#include "stev_host.h"

namespace stev {

constexpr int kCB = 1024;  // cells per compaction block

__global__ void __launch_bounds__(kCB) compact_count_kernel(const unsigned char *__restrict__ flags, int n,
                                                            int *__restrict__ block_counts) {
  __shared__ int warp_counts[kCB / 32];
  const int i = blockIdx.x * kCB + threadIdx.x;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const bool f = (i < n) && flags[i] != 0;
  const unsigned b = __ballot_sync(0xffffffffu, f);
  if (lane == 0) warp_counts[warp] = __popc(b);
  __syncthreads();
  if (warp == 0) {
    int v = warp_counts[lane];
#pragma unroll
    for (int off = 16; off >= 1; off >>= 1) v += __shfl_xor_sync(0xffffffffu, v, off);
    if (lane == 0) block_counts[blockIdx.x] = v;
  }
}

// single block: exclusive scan of block_counts[0..nb) in place, total to *count_out
__global__ void __launch_bounds__(kCB) compact_scan_kernel(int *__restrict__ block_counts, int nb, int *__restrict__ count_out) {
  __shared__ int warp_sums[kCB / 32];
  __shared__ int carry_s;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  if (threadIdx.x == 0) carry_s = 0;
  __syncthreads();
  for (int base = 0; base < nb; base += kCB) {
    const int i = base + threadIdx.x;
    const int v = (i < nb) ? block_counts[i] : 0;
    int incl = v;
#pragma unroll
    for (int off = 1; off < 32; off <<= 1) {
      int t = __shfl_up_sync(0xffffffffu, incl, off);
      if (lane >= off) incl += t;
    }
    if (lane == 31) warp_sums[warp] = incl;
    __syncthreads();
    if (warp == 0) {
      int ws = warp_sums[lane];
      int wi = ws;
#pragma unroll
      for (int off = 1; off < 32; off <<= 1) {
        int t = __shfl_up_sync(0xffffffffu, wi, off);
        if (lane >= off) wi += t;
      }
      warp_sums[lane] = wi - ws;  // exclusive offsets of the warps
    }
    __syncthreads();
    const int carry = carry_s;
    if (i < nb) block_counts[i] = carry + warp_sums[warp] + incl - v;
    __syncthreads();
    if (threadIdx.x == kCB - 1) carry_s = carry + warp_sums[warp] + incl;
    __syncthreads();
  }
  if (threadIdx.x == 0) *count_out = carry_s;
}

__global__ void __launch_bounds__(kCB) compact_scatter_kernel(const unsigned char *__restrict__ flags,
                                                              const int *__restrict__ list_in, int n,
                                                              const int *__restrict__ block_offsets,
                                                              int *__restrict__ list_out) {
  __shared__ int warp_off[kCB / 32];
  const int i = blockIdx.x * kCB + threadIdx.x;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const bool f = (i < n) && flags[i] != 0;
  const unsigned b = __ballot_sync(0xffffffffu, f);
  if (lane == 0) warp_off[warp] = __popc(b);
  __syncthreads();
  if (warp == 0) {
    const int c = warp_off[lane];
    int incl = c;
#pragma unroll
    for (int off = 1; off < 32; off <<= 1) {
      int t = __shfl_up_sync(0xffffffffu, incl, off);
      if (lane >= off) incl += t;
    }
    warp_off[lane] = incl - c;
  }
  __syncthreads();
  if (f) {
    const int dst = block_offsets[blockIdx.x] + warp_off[warp] + __popc(b & ((1u << lane) - 1u));
    list_out[dst] = list_in ? list_in[i] : i;
  }
}

int compact_launch(const unsigned char *flags, const int *list_in, int n, int *list_out, int *count_out, int *block_counts,
                   cudaStream_t s) {
  const int nb = (n + kCB - 1) / kCB;
  if (n <= 0) {
    STEV_CUDA(cudaMemsetAsync(count_out, 0, 4, s));
    return STEV_OK;
  }
  compact_count_kernel<<<nb, kCB, 0, s>>>(flags, n, block_counts);
  compact_scan_kernel<<<1, kCB, 0, s>>>(block_counts, nb, count_out);
  compact_scatter_kernel<<<nb, kCB, 0, s>>>(flags, list_in, n, block_counts, list_out);
  STEV_CUDA(cudaGetLastError());
  return STEV_OK;
}

}  // namespace stev

extern "C" int stev_compact_active(const uint8_t *flags, const int32_t *list_in, int32_t n, int32_t *list_out,
                                   int32_t *count_out, void *scratch, size_t scratch_bytes, void *cuda_stream) {
  if (n < 0 || (n > 0 && (!flags || !list_out)) || !count_out) {
    stev::set_error("stev_compact_active: bad argument");
    return STEV_EINVAL;
  }
  if (!scratch || scratch_bytes < 4 * ((size_t)n / 1024 + 2)) {
    stev::set_error("stev_compact_active: scratch too small");
    return STEV_EWORKSPACE;
  }
  return stev::compact_launch(flags, list_in, n, list_out, count_out, (int *)scratch, (cudaStream_t)cuda_stream);
}
