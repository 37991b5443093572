// stev_compact.cu -- variable-load retirement between passes (row a6): the cells still active after
// a pass are gathered, order preserved, into the next pass's active list.  Warp ballot + popc inside a warp,
// a shared-memory scan across the warps of a block, and a grid-level exclusive prefix sum of the block totals.
#include <algorithm>

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

// ---------------------------------------------------------------------------------------------------------
// Launch order of the cells (scheduling only): cells finish after very different numbers of
// steps and the step count grows with temperature, so the persistent kernels pull the hottest cells first -- the
// long integrations start at once and the short ones fill in behind them, instead of a few long cells running alone at
// the end.  Counting sort on a 4096-bucket temperature scale (descending), order within a bucket arbitrary: results
// do not depend on the order, only the schedule does.
// ---------------------------------------------------------------------------------------------------------
__device__ __forceinline__ int order_bucket(double T) {
  double x = (T - 200.0) * (double)kOrderBuckets / 3800.0;   // 200 K .. 4000 K; everything else (NaN too) in the end buckets
  int b = (x >= 0.0) ? ((x < (double)(kOrderBuckets - 1)) ? (int)x : kOrderBuckets - 1) : 0;
  return kOrderBuckets - 1 - b;
}

// `group` consecutive cells (1, or 4 = one 32-byte sector of every fp64 row of the state) share one key, the
// temperature of their hottest cell, and stay together in the list: the lanes that pull them touch the same sectors of
// T, p and the S rows of Y at about the same time, so each sector is fetched from DRAM once instead of once per cell.
__device__ __forceinline__ int order_group_bucket(const double *__restrict__ T, long long i0, int cnt) {
  int b = kOrderBuckets - 1;
  for (int k = 0; k < cnt; ++k) b = min(b, order_bucket(T[i0 + k]));   // smallest bucket = hottest cell
  return b;
}

__global__ void __launch_bounds__(256) order_hist_kernel(const double *__restrict__ T, long long n, int group,
                                                         int *__restrict__ hist) {
  __shared__ int h[kOrderBuckets];
  for (int i = threadIdx.x; i < kOrderBuckets; i += 256) h[i] = 0;
  __syncthreads();
  const long long n_groups = (n + group - 1) / group;
  for (long long g = (long long)blockIdx.x * 256 + threadIdx.x; g < n_groups; g += (long long)gridDim.x * 256) {
    const long long i0 = g * group;
    const int cnt = (int)min((long long)group, n - i0);
    atomicAdd(&h[order_group_bucket(T, i0, cnt)], cnt);
  }
  __syncthreads();
  for (int i = threadIdx.x; i < kOrderBuckets; i += 256)
    if (h[i]) atomicAdd(&hist[i], h[i]);
}

__global__ void __launch_bounds__(256) order_scatter_kernel(const double *__restrict__ T, long long n, int group,
                                                            int *__restrict__ offsets, int *__restrict__ list) {
  const long long n_groups = (n + group - 1) / group;
  for (long long g = (long long)blockIdx.x * 256 + threadIdx.x; g < n_groups; g += (long long)gridDim.x * 256) {
    const long long i0 = g * group;
    const int cnt = (int)min((long long)group, n - i0);
    const int dst = atomicAdd(&offsets[order_group_bucket(T, i0, cnt)], cnt);
    for (int k = 0; k < cnt; ++k) list[dst + k] = (int)(i0 + k);
  }
}

// hist: kOrderBuckets + 1 ints of scratch; list: n ints
int order_cells_launch(const double *T, long long n, int group, int *list, int *hist, cudaStream_t s) {
  STEV_CUDA(cudaMemsetAsync(hist, 0, sizeof(int) * (kOrderBuckets + 1), s));
  const long long n_groups = (n + group - 1) / group;
  const int blocks = (int)std::min<long long>((n_groups + 255) / 256, 4 * (long long)device_sm_count());
  order_hist_kernel<<<blocks, 256, 0, s>>>(T, n, group, hist);
  compact_scan_kernel<<<1, kCB, 0, s>>>(hist, kOrderBuckets, hist + kOrderBuckets);   // exclusive scan in place
  order_scatter_kernel<<<blocks, 256, 0, s>>>(T, n, group, hist, list);
  STEV_CUDA(cudaGetLastError());
  return STEV_OK;
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
