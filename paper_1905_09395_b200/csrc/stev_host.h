// stev_host.h -- host-side handle types and helpers shared by the translation units of libstev_b200.so.
#pragma once
#include <cstdint>
#include <string>
#include <vector>

#include <cuda_runtime.h>

#include "../../include/stev.h"
#include "stev_ls.cuh"
#include "stev_device.cuh"

struct stev_estimator;

namespace stev {

void set_error(const std::string &msg);
int cuda_fail(cudaError_t e, const char *what);
#define STEV_CUDA(call)                                        \
  do {                                                         \
    cudaError_t e__ = (call);                                  \
    if (e__ != cudaSuccess) return ::stev::cuda_fail(e__, #call); \
  } while (0)

struct HostEstimator {
  int n_in = 0, H = 0, n_out = 0, act = 0, input_map = 0;
  float h_ref_T = 1000.f;
  std::vector<float> in_shift, in_scale, W1, b1, W2, b2;  // caller's row-major layouts
};

// Host copy of a mechanism in the caller's ordering plus derived quantities.
struct HostMechanism {
  int S = 0, R = 0, Rrev = 0;
  std::vector<double> W, nasa_lo, nasa_hi, t_mid, A, b, Ea;
  std::vector<uint8_t> reversible;
  std::vector<int> reac_ptr, reac_sp, reac_nu, prod_ptr, prod_sp, prod_nu;
  bool has_real = false;         // real stoichiometric coefficients / rate-law exponents given
  std::vector<double> reac_coef, prod_coef, reac_order, prod_order;   // per CSR entry, always filled (defaults applied)
  std::vector<int> internal_of;  // caller reaction index -> internal index (reversible first)
  std::vector<int> orig_of;      // internal -> caller
};

// Builds the table image for a mechanism and, optionally, an estimator.
void build_table_image(const HostMechanism &m, const HostEstimator *e, std::vector<unsigned char> &image, DevTables &tb,
                       bool f32 = false);

struct LaunchConfig {
  int G = 1, threads = 128, cells_per_block = 128, blocks_per_sm = 1;
  size_t smem = 0;
  CellLayout cl{};
};
// Chooses lanes per cell, block shape and the per-cell shared-memory layout.  Returns false if nothing fits.
bool choose_config(const DevTables &tb, int lanes_per_cell_request, LaunchConfig &cfg, int bytes_per_real = 8);

int device_sm_count();

int estimator_tensor_prepare(stev_estimator *e);

// Lock-step integrator (stev_ls.cuh / stev_ls.cu): all cells of a block step together.  build_ls_image returns false if
// the mechanism is outside its limits (more than two factors per reaction side, tables too large for shared memory).
bool build_ls_image(const HostMechanism &m, const HostEstimator *e, std::vector<unsigned char> &image, LsTables &tb, bool f32 = false);
// allow_static: use the instantiation with compile-time dimensions if the shape list has one (*is_static says which ran)
int integrate_ls_launch(const LsTables &tb, const unsigned char *d_table, const SolverConsts &sc, double t_f, long long n,
                        long long ld, double *T, const double *p, double *Y, int *steps, unsigned char *status, int *counters,
                        cudaStream_t s, int *blocks_out, size_t *smem_out, const int *list, bool allow_static, bool *is_static);

// Launch order of the cells, hottest first (stev_compact.cu).  hist: kOrderBuckets + 1 ints of scratch; list: n ints.
constexpr int kOrderBuckets = 4096;
int order_cells_launch(const double *T, long long n, int group, int *list, int *hist, cudaStream_t s);
// group size of the launch order for stev_params.order_cells (1: by the size of the state against L2; 2: 1; 3: 4; 4: 8)
inline int order_group(int order_cells, long long n, int S) {
  if (order_cells == 2) return 1;
  if (order_cells == 3) return 4;
  if (order_cells == 4) return 8;
  return ((double)n * (double)(S + 2) * 8.0 > 64.0 * 1024.0 * 1024.0) ? 8 : 1;
}

}  // namespace stev

struct stev_mechanism {
  stev::HostMechanism host;
  stev::DevTables tb{};
  unsigned char *d_table = nullptr;
  stev::DevTables tb32{};                // the same image with every real table rounded to float (state_precision FP32)
  unsigned char *d_table32 = nullptr;
  bool ls_ok = false;                    // image of the lock-step kernel (NASA-7 thermo)
  stev::LsTables ls_tb{};
  unsigned char *d_ls_table = nullptr;
  bool ls32_ok = false;                  // the same for the binary32 state path
  stev::LsTables ls_tb32{};
  unsigned char *d_ls_table32 = nullptr;
};

struct stev_estimator {
  stev::HostEstimator host;
  const stev_mechanism *mech = nullptr;  // the mechanism it was loaded against (may be null)
  stev::DevTables tb{};                  // mechanism + estimator image (only if mech != null)
  unsigned char *d_table = nullptr;
  stev::DevTables tb32{};
  unsigned char *d_table32 = nullptr;
  bool ls_ok = false;                    // image of the lock-step kernel (MLP thermo)
  stev::LsTables ls_tb{};
  unsigned char *d_ls_table = nullptr;
  bool ls32_ok = false;
  stev::LsTables ls_tb32{};
  unsigned char *d_ls_table32 = nullptr;
  // standalone evaluation (stev_estimator_eval): device copies in kernel-friendly layouts
  float *d_params = nullptr;             // in_shift, in_scale, W1T [n_in][H], b1, W2T [H][n_out], b2
  size_t params_floats = 0;
  // tensor-core path (stev_mlp_tc.cu): weight images in the canonical UMMA layout, [0] TF32, [1] BF16
  bool tc_ok[2] = {false, false};
  unsigned char *d_tc_image[2] = {nullptr, nullptr};
};
