// stev_aux.cu -- test exports and microbenchmarks: DFT magnitudes, contract exp/log on arrays, FP64 throughput
// probes used as roofline denominators, and the standalone fp32 (CUDA-core) estimator forward pass.
#include "stev_host.h"

namespace stev {

// |DFT| of 13-sample windows, bins 0..6 (Eq 9), same sums as the integrator's test.
template <int M>
__device__ __forceinline__ double dft_bin_mag(const double (&x)[kWindow]) {
  return sqrt(dft_bin_sq<M>(x));
}

__global__ void dft_mag_kernel(const double *__restrict__ ring, long long n, double *__restrict__ D) {
  const long long c = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= n) return;
  double x[kWindow];
#pragma unroll
  for (int k = 0; k < kWindow; ++k) x[k] = ring[c * kWindow + k];
  double d0 = 0.0;
#pragma unroll
  for (int k = 0; k < kWindow; ++k) d0 = d0 + x[k];
  double *o = D + c * 7;
  o[0] = fabs(d0);
  o[1] = dft_bin_mag<1>(x);
  o[2] = dft_bin_mag<2>(x);
  o[3] = dft_bin_mag<3>(x);
  o[4] = dft_bin_mag<4>(x);
  o[5] = dft_bin_mag<5>(x);
  o[6] = dft_bin_mag<6>(x);
}

__global__ void exp_log_kernel(const double *__restrict__ x, long long n, double *__restrict__ e, double *__restrict__ l) {
  const long long c = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= n) return;
  if (e) e[c] = cexp(x[c]);
  if (l) l[c] = clog(x[c]);
}

// FP64 throughput probes.  kind 0: 8 independent DFMA chains per thread; kind 1: 4 independent contract exps.
__global__ void __launch_bounds__(256) microbench_kernel(int kind, int iters, double seed, double *sink) {
  double a0 = seed + threadIdx.x * 1e-9, a1 = a0 + 1e-3, a2 = a0 + 2e-3, a3 = a0 + 3e-3;
  double a4 = a0 + 4e-3, a5 = a0 + 5e-3, a6 = a0 + 6e-3, a7 = a0 + 7e-3;
  const double m = 0.999999, c = 1e-7;
  if (kind == 0) {
    for (int i = 0; i < iters; ++i) {
      a0 = fma_rn(a0, m, c); a1 = fma_rn(a1, m, c); a2 = fma_rn(a2, m, c); a3 = fma_rn(a3, m, c);
      a4 = fma_rn(a4, m, c); a5 = fma_rn(a5, m, c); a6 = fma_rn(a6, m, c); a7 = fma_rn(a7, m, c);
    }
  } else if (kind == 1) {
    for (int i = 0; i < iters; ++i) {
      a0 = cexp(a0 * -0.5); a1 = cexp(a1 * -0.5); a2 = cexp(a2 * -0.5); a3 = cexp(a3 * -0.5);
    }
  } else {
    // kind 2: one dependent DFMA chain per thread (latency probe; launched with one warp per SM)
#pragma unroll 16
    for (int i = 0; i < 8 * iters; ++i) a0 = fma_rn(a0, m, c);
  }
  const double r = ((a0 + a1) + (a2 + a3)) + ((a4 + a5) + (a6 + a7));
  if (r == 123456.789) sink[0] = r;
}

// Standalone estimator forward pass on fp32 CUDA cores (R18): one thread per row, rows staged
// through shared memory for coalescing; per output the accumulation order is the contract's (index order, fmaf).
// params: in_shift[n_in], in_scale[n_in], W1T[n_in][H], b1[H], W2T[H][n_out], b2[n_out]
constexpr int kEstRows = 128;
__global__ void __launch_bounds__(kEstRows) estimator_fp32_kernel(const float *__restrict__ params, int n_in, int H, int n_out,
                                                                  int act, const float *__restrict__ X, long long n,
                                                                  float *__restrict__ out) {
  extern __shared__ float sm[];
  const int n_par = 2 * n_in + n_in * H + H + H * n_out + n_out;
  float *sp = sm;                                  // parameters
  float *sx = sp + ((n_par + 3) & ~3);             // [kEstRows][n_in + 1]  (padded rows)
  float *sh = sx + kEstRows * (n_in + 1);          // [H][kEstRows]
  float *so = sh + H * kEstRows;                   // [kEstRows][n_out + 1]
  for (int i = threadIdx.x; i < n_par; i += kEstRows) sp[i] = params[i];
  const float *shift = sp, *scale = sp + n_in, *W1T = sp + 2 * n_in, *b1 = W1T + n_in * H, *W2T = b1 + H, *b2 = W2T + H * n_out;
  for (long long row0 = (long long)blockIdx.x * kEstRows; row0 < n; row0 += (long long)gridDim.x * kEstRows) {
    const int rows = (int)((n - row0 < kEstRows) ? (n - row0) : kEstRows);
    __syncthreads();
    for (int i = threadIdx.x; i < rows * n_in; i += kEstRows) sx[(i / n_in) * (n_in + 1) + i % n_in] = X[row0 * n_in + i];
    __syncthreads();
    const int r = threadIdx.x;
    if (r < rows) {
      for (int j = 0; j < H; ++j) {
        float z = b1[j];
        for (int k = 0; k < n_in; ++k) {
          const float x = (sx[r * (n_in + 1) + k] - shift[k]) * scale[k];
          z = __fmaf_rn(W1T[k * H + j], x, z);
        }
        const double zd = (double)z;
        float a;
        if (act == 0) a = (float)(1.0 - 2.0 / (1.0 + cexp(2.0 * zd)));
        else a = (float)(1.0 / (1.0 + cexp(-zd)));
        sh[j * kEstRows + r] = a;
      }
      for (int o = 0; o < n_out; ++o) {
        float y = b2[o];
        for (int j = 0; j < H; ++j) y = __fmaf_rn(W2T[j * n_out + o], sh[j * kEstRows + r], y);
        so[r * (n_out + 1) + o] = y;
      }
    }
    __syncthreads();
    for (int i = threadIdx.x; i < rows * n_out; i += kEstRows) out[row0 * n_out + i] = so[(i / n_out) * (n_out + 1) + i % n_out];
  }
}

int estimator_eval_tensor(const stev_estimator *e, long long n, const float *X, float *out, int precision, cudaStream_t s);

}  // namespace stev

using namespace stev;

extern "C" {

int stev_dft_mag(const double *ring, int64_t n, double *D, void *cuda_stream) {
  if (n < 0 || (n > 0 && (!ring || !D))) { set_error("stev_dft_mag: bad argument"); return STEV_EINVAL; }
  if (n == 0) return STEV_OK;
  dft_mag_kernel<<<(unsigned)((n + 127) / 128), 128, 0, (cudaStream_t)cuda_stream>>>(ring, n, D);
  STEV_CUDA(cudaGetLastError());
  return STEV_OK;
}

int stev_contract_exp_log(const double *x, int64_t n, double *exp_out, double *log_out, void *cuda_stream) {
  if (n < 0 || (n > 0 && !x)) { set_error("stev_contract_exp_log: bad argument"); return STEV_EINVAL; }
  if (n == 0) return STEV_OK;
  exp_log_kernel<<<(unsigned)((n + 255) / 256), 256, 0, (cudaStream_t)cuda_stream>>>(x, n, exp_out, log_out);
  STEV_CUDA(cudaGetLastError());
  return STEV_OK;
}

int stev_microbench(int32_t kind, int32_t iters, double *ops_per_s, void *cuda_stream) {
  if ((kind < 0 || kind > 2) || iters < 1 || !ops_per_s) { set_error("stev_microbench: bad argument"); return STEV_EINVAL; }
  cudaStream_t s = (cudaStream_t)cuda_stream;
  double *sink = nullptr;
  STEV_CUDA(cudaMalloc(&sink, 8));
  const int blocks = (kind == 2) ? device_sm_count() : device_sm_count() * 8, threads = (kind == 2) ? 32 : 256;
  cudaEvent_t e0, e1;
  STEV_CUDA(cudaEventCreate(&e0));
  STEV_CUDA(cudaEventCreate(&e1));
  microbench_kernel<<<blocks, threads, 0, s>>>(kind, iters, 0.5, sink);  // warm-up
  STEV_CUDA(cudaEventRecord(e0, s));
  microbench_kernel<<<blocks, threads, 0, s>>>(kind, iters, 0.5, sink);
  STEV_CUDA(cudaEventRecord(e1, s));
  STEV_CUDA(cudaEventSynchronize(e1));
  float ms = 0.f;
  STEV_CUDA(cudaEventElapsedTime(&ms, e0, e1));
  const double per_thread = (kind == 1) ? 4.0 * iters : 8.0 * iters;
  *ops_per_s = per_thread * (double)blocks * threads / (ms * 1e-3);
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  cudaFree(sink);
  return STEV_OK;
}

int stev_estimator_eval(const stev_estimator *e, int64_t n, const float *X, float *out, int32_t precision, void *cuda_stream) {
  if (!e || n < 0 || (n > 0 && (!X || !out))) { set_error("stev_estimator_eval: bad argument"); return STEV_EINVAL; }
  if (n == 0) return STEV_OK;
  cudaStream_t s = (cudaStream_t)cuda_stream;
  const HostEstimator &h = e->host;
  if (precision == STEV_PREC_FP32) {
    const int n_par = 2 * h.n_in + h.n_in * h.H + h.H + h.H * h.n_out + h.n_out;
    const size_t smem = 4 * ((size_t)((n_par + 3) & ~3) + kEstRows * (h.n_in + 1) + (size_t)h.H * kEstRows + kEstRows * (h.n_out + 1));
    if (smem > 227 * 1024) { set_error("stev_estimator_eval: network too large for the fp32 kernel"); return STEV_EINVAL; }
    STEV_CUDA(cudaFuncSetAttribute((const void *)estimator_fp32_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    long long blocks = (n + kEstRows - 1) / kEstRows;
    const long long cap = (long long)device_sm_count() * 2;
    if (blocks > cap) blocks = cap;
    estimator_fp32_kernel<<<(unsigned)blocks, kEstRows, smem, s>>>(e->d_params, h.n_in, h.H, h.n_out, h.act, X, n, out);
    STEV_CUDA(cudaGetLastError());
    return STEV_OK;
  }
  if (precision == STEV_PREC_TF32 || precision == STEV_PREC_BF16) return estimator_eval_tensor(e, n, X, out, precision, s);
  set_error("stev_estimator_eval: unknown precision");
  return STEV_EINVAL;
}

}  // extern "C"
