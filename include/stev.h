/*
 * stev.h -- C ABI of the B200-native STEV library (libstev_b200.so).
 *
 * STEV = the Stabilized, Explicit, Variable-load integrator for stiff chemical kinetics of
 * Buchheit, Owoyele, Jordan, Van Essendelft (arxiv 1905.09395).  Citations below are
 * "PAPER.md:LINE (section / equation)" into the paper text; "R<n>" are the readings listed in
 * DESIGN.md section 3 where the paper is silent.
 *
 * The paper couples its solver to a CFD code through a C link that receives raw memory pointers and
 * returns results by reference, as a drop-in for the CFD code's stiff solver.
 * This header is that link for the CUDA implementation: plain C, POD structs, raw pointers.
 *
 * Conventions
 *   - Units are cgs-mol ("cm, s, mol, cal"): p in dyn/cm^2, Ea in cal/mol, A in
 *     (cm^3/mol)^(order-1)/s, W in g/mol.
 *   - "host" / "device" next to a pointer says where the memory lives.  Descriptor arrays are HOST
 *     memory; the library copies them, the caller may free them after the call returns.
 *   - Per-cell arrays (T, p, Y, steps, status, workspace) are DEVICE memory owned by the caller
 *     (e.g. allocated by PyTorch); the library never allocates per-cell memory in stev_integrate.
 *   - Mass fractions are species-major: Y[i*ld + c] is species i of cell c, ld >= n_cells.
 *   - Every entry point returns an int: 0 = OK, < 0 = error (nothing written), > 0 = completed with a
 *     warning.  No exceptions, no aborts, nothing printed.  stev_last_error() gives the message.
 *   - stev_integrate enqueues work on `cuda_stream`; by default it synchronises that stream before returning (outputs
 *     valid on return, warning code returned); with stev_params.nonblocking = 1 it returns right after enqueueing a
 *     single-pass launch and stev_integrate_finish() delivers the return code.
 */
#ifndef STEV_H
#define STEV_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#if defined(__GNUC__)
#define STEV_API __attribute__((visibility("default")))
#else
#define STEV_API
#endif

#define STEV_OK 0
#define STEV_EINVAL (-1)     /* bad argument / malformed or non-conserving mechanism / unsupported size */
#define STEV_EWORKSPACE (-2) /* workspace too small or NULL */
#define STEV_ECUDA (-3)      /* CUDA runtime error (message in stev_last_error) */
#define STEV_WMAXSTEPS 1     /* some cells stopped at max_steps: status 1, state = state at t_reached < dt_cfd (R20) */
#define STEV_WNONFINITE 2    /* some cells produced a non-finite T or Y: status 2 */

#define STEV_ACT_TANH 0
#define STEV_ACT_SIGMOID 1   /* the paper's choice */
#define STEV_IN_T 0          /* estimator input: (T)                 -- PAPER.md:126 "inputs are the temperatures" */
#define STEV_IN_T_P_Y 1      /* estimator input: (T, p, Y_0..Y_S-1)  -- BASELINE.json config 4 */
#define STEV_PREC_FP32 0     /* fp32 CUDA-core path, bit-reproducible (R18) */
#define STEV_PREC_TF32 1     /* tcgen05 kind::tf32, fp32 accumulate in TMEM */
#define STEV_PREC_BF16 2     /* tcgen05 kind::f16 with bf16 operands, fp32 accumulate in TMEM */
#define STEV_STATE_FP64 0    /* state, rates and DFT in binary64 (BASELINE.json; the default) */
#define STEV_STATE_FP32 1    /* state, rates and DFT in binary32, as the paper ran it; in/out arrays stay fp64 */
#define STEV_ENERGY_ADIABATIC 0 /* constant-pressure adiabatic temperature equation (R15) */
#define STEV_ENERGY_ISOTHERMAL 1

#define STEV_DFT_WINDOW 13   /* "the thirteen most recent changes in reaction progress" */
#define STEV_MAX_SPECIES 64
#define STEV_MAX_REACTIONS 512

typedef struct stev_mechanism stev_mechanism; /* opaque, library-owned, immutable, usable from any stream */
typedef struct stev_estimator stev_estimator; /* opaque, library-owned, immutable */

/* Species, NASA-7 thermodynamics (Eqs 15-16) and Arrhenius mass-action reactions
 * (Eqs 28-30).  All pointers: host.  Each reaction has 1..2 reactant entries and 1..2
 * product entries (CSR), integer stoichiometric coefficients 1..3 (or real ones, below), no species on both sides. */
typedef struct {
  int32_t n_species, n_elements, n_reactions;
  const double *mol_weight;        /* [S] g/mol */
  const double *elem_comp;         /* [S*E] atoms of element e in species i, or NULL; used only to validate
                                      element conservation of every reaction (STEV_EINVAL if violated) */
  const double *nasa_lo, *nasa_hi; /* [S*7] a1..a7 for T < t_mid / T >= t_mid (R17) */
  const double *t_mid;             /* [S] K */
  const double *A, *b, *Ea;        /* [R] k_f = A T^b exp(-Ea / (R_cal T)) */
  const uint8_t *reversible;       /* [R] 1: reverse rate from K_c (Eq 30), 0: irreversible */
  const int32_t *reac_ptr, *reac_species, *reac_nu; /* [R+1], [nnz], [nnz] */
  const int32_t *prod_ptr, *prod_species, *prod_nu;
  /* Optional, host, one double per CSR entry, each may be NULL (Eqs 26-29: the BFER methane mechanism has
   * CH4 + 1.5 O2 -> CO + 2 H2O with the rate k C_CH4^0.5 C_O2^0.65, and CO + 0.5 O2 <=> CO2):
   *   reac_coef / prod_coef    real stoichiometric coefficients (> 0) used in the species source terms, the reaction's
   *                            Gibbs energy and Delta-nu of Eq 30; default (double) reac_nu / prod_nu
   *   reac_order / prod_order  exponent (>= 0) of the species' concentration in the forward / reverse rate law; default the
   *                            coefficient.  Exponents 1, 2, 3 multiply; any other is exp(x log C), and 0 for C <= 0 (R22).
   * A mechanism with any of these runs on the shared-memory-history kernel (lanes_per_cell 0 or 1..32) only. */
  const double *reac_coef, *prod_coef, *reac_order, *prod_order;
} stev_mechanism_desc;

/* Shallow MLP property estimator (Fig 2): one hidden layer, linear output.
 * float32 host arrays, row-major.  x_k = ((float)raw_k - in_shift_k) * in_scale_k;
 * hidden_j = act(b1_j + sum_k W1[j][k] x_k); out_o = b2_o + sum_j W2[o][j] hidden_j.
 * Attached to the integrator it must have n_out = 2S: out[i] = cp_i/R, out[S+i] = h_i/(R h_ref_temperature). */
typedef struct {
  int32_t n_in, n_hidden, n_out;   /* n_in <= 64, n_hidden <= 128 (multiple of 8), n_out <= 256 */
  int32_t activation;              /* STEV_ACT_* */
  int32_t input_map;               /* STEV_IN_*; n_in must be 1 or 2+S accordingly */
  const float *in_shift, *in_scale;
  const float *W1, *b1, *W2, *b2;  /* [H*n_in], [H], [n_out*H], [n_out] */
  float h_ref_temperature;
} stev_estimator_desc;

/* Solver constants.  Defaults (stev_params_default) are the readings R3-R20. */
typedef struct {
  double y_step_max;   /* Y_step^max of Eq 3, PAPER.md:40-51 (R3: 1e-2) */
  double delta_max;    /* delta^max of Eq 4, PAPER.md:43-57 (R4: 1e-2 -> at least 100 steps) */
  double alpha;        /* species limit factor of Eq 7, PAPER.md:65-67 (1e-5; 0 disables gamma) */
  double tol_ring;     /* Tol_ring of Eq 12, PAPER.md:87-95 (R12: 0.5) */
  double tol_freq;     /* Tol_freq of Eq 12 (R12: 0.1, dimensionless because of R9) */
  double r_fac;        /* r_fac of Eq 12 (R12: 2.0; must be > 1) */
  double rof_min;      /* lower clamp of rOF, "0 < rOF" (R13: 2^-100) */
  int32_t dft_window;  /* length of the history of Eq 8: 13, "the thirteen most recent"; other values: STEV_EINVAL */
  int32_t dft_first_high_bin; /* n of Eq 10, high bins are n..6 (R10: 4); 1..6 */
  int32_t dft_enable;  /* 0 switches section 2.3 off (rOF stays 1) */
  int32_t max_steps;   /* per cell (R20: 200000) */
  int32_t energy_mode; /* STEV_ENERGY_* */
  int32_t estimator_precision; /* STEV_PREC_*: precision of the attached estimator INSIDE stev_integrate.  Only STEV_PREC_FP32 (the
                             bit-reproducible CUDA-core path, R18) is accepted there; TF32 / BF16 return STEV_EINVAL: a
                             tensor-core contraction needs >= 64 cells at the same phase per MMA where a block holds at most 32,
                             and the estimator is 3 % (config 3) to 12 % (config 4) of the integrator's issued instructions
                             (DESIGN.md section 7.4).  stev_estimator_eval runs all three. */
  int32_t state_precision; /* STEV_STATE_*: FP32 runs the whole step in binary32 with its own arithmetic contract
                             (DESIGN.md section 5b); checked against the oracle's binary32 mode */
  /* scheduling only: results do not depend on these */
  int32_t chunk_steps;    /* 0: every cell runs to completion in one pass; > 0: a pass advances each active
                             cell at most this many steps, unfinished cells are spilled to the workspace and the
                             active-cell list is compacted before the next pass */
  int32_t lanes_per_cell; /* 0 = the lock-step kernel wherever the call fits it, else the shared-memory-history kernel with the
                             lane count chosen from (S, R).  1,2,4,8,16,32 = lanes cooperating on one cell, DFT history in
                             shared memory (any mechanism, any chunk_steps).
                             512 = lock-step block: up to 32 cells of a block step together, work flattened over (reaction,
                                  cell) and (species, cell) pairs, one warp for the scalar chains of all cells, DFT history in
                                  tensor memory.  Needs chunk_steps = 0, at most two factors per reaction side, integer
                                  coefficients and orders, <= 64 species, <= 1920 reversible reactions (3840 in binary32);
                                  STEV_EINVAL otherwise.  513 = the same with run-time dimensions only (the instantiation any
                                  mechanism outside the shape list runs).  Other values: STEV_EINVAL. */
  int32_t nonblocking;    /* 0: stev_integrate returns after the stream has drained, with the final return code.  1: if the call
                             is a single kernel pass (chunk_steps = 0) it only enqueues on the stream and returns STEV_OK;
                             outputs are valid after the caller synchronises the stream, and stev_integrate_finish() returns
                             the warning code (the CFD code may overlap its own work) */
  int32_t order_cells;    /* 1 (default): the persistent kernels pull the cells in order of decreasing temperature
                             (a counting sort on the device before the launch) -- step counts grow with temperature,
                             so the long integrations start first and do not end up running alone.
                             While the state (n x (S + 2) doubles) is at most 64 MiB, i.e. stays in L2, the order is cell
                             by cell; above that, aligned groups of eight consecutive cells (one 64-byte DRAM access = two
                             32-byte sectors of T, p and every row of Y) are keyed by their hottest cell and stay together,
                             so each sector is fetched from HBM once instead of once per cell.  2: cell by cell at any size; 3: groups of
                             four at any size; 4: groups of eight (two sectors per row) at any size; 0: index order.  Scheduling only: results do not depend on it. */
} stev_params;

/* Counters of the last stev_integrate / stev_integrate_host call on this thread. */
typedef struct {
  int32_t passes;            /* integrator kernel launches */
  int32_t kernel_launches;   /* all kernels launched (integrator + compaction + init) */
  int32_t lanes_per_cell, threads_per_block, cells_per_block, blocks;
  int64_t smem_bytes;        /* dynamic shared memory per block */
  int64_t total_steps;       /* sum of per-cell step counts (filled by stev_integrate_host only; else -1) */
  int32_t specialised;       /* 1: the kernel instantiation with this mechanism's dimensions as compile-time constants ran */
  int32_t reserved;
} stev_stats;

STEV_API void stev_params_default(stev_params *p);

/* Create / destroy.  PAPER.md:113-120, 212-229.  Returns STEV_EINVAL for sizes above STEV_MAX_*, more than two
 * entries per reaction side, coefficients outside 1..3, non-positive W or A, or element imbalance. */
STEV_API int stev_mechanism_create(const stev_mechanism_desc *desc, stev_mechanism **out);
STEV_API void stev_mechanism_destroy(stev_mechanism *m);
STEV_API int stev_mechanism_sizes(const stev_mechanism *m, int32_t *n_species, int32_t *n_reactions, int32_t *n_reversible);

/* PAPER.md:120-136.  `m` may be NULL for an estimator used only through stev_estimator_eval. */
STEV_API int stev_estimator_load(const stev_mechanism *m, const stev_estimator_desc *desc, stev_estimator **out);
STEV_API void stev_estimator_destroy(stev_estimator *e);

/* Bytes of device workspace stev_integrate needs for n_cells (depends on chunk_steps). */
STEV_API size_t stev_workspace_bytes(const stev_mechanism *m, const stev_estimator *e, const stev_params *p, int64_t n_cells);

/* The hot path: advance n_cells independent cells from t = 0 to t = dt_cfd.
 *   T      [n_cells]      device, in/out   temperature, K
 *   p      [n_cells]      device, in       pressure, dyn/cm^2 (constant over the step, R15)
 *   Y      [S][ld]        device, in/out   mass fractions, species-major
 *   steps_out  [n_cells]  device, out      integrator steps taken by each cell
 *   status_out [n_cells]  device, out, may be NULL   0 reached dt_cfd, 1 stopped at max_steps, 2 non-finite
 *   workspace             device, >= stev_workspace_bytes(...), 256-byte aligned
 *   cuda_stream           cudaStream_t (NULL = default stream)
 * estimator == NULL evaluates cp and h from the NASA-7 polynomials.  n_cells == 0 is a no-op. */
STEV_API int stev_integrate(const stev_mechanism *m, const stev_estimator *estimator, const stev_params *p, int64_t n_cells,
                   int64_t ld, double *T, const double *pressure, double *Y, double dt_cfd, int32_t *steps_out,
                   uint8_t *status_out, void *workspace, size_t workspace_bytes, void *cuda_stream);

/* After a nonblocking stev_integrate on `cuda_stream` with this workspace: synchronises the stream and returns what the
 * blocking call would have returned (STEV_OK, STEV_WMAXSTEPS, STEV_WNONFINITE, or STEV_ECUDA). */
STEV_API int stev_integrate_finish(void *workspace, void *cuda_stream);

/* stev_integrate for callers that cannot allocate device memory (code under CUDA graph capture, serving loops, harnesses
 * that forbid cudaMalloc): no workspace argument.  The scratch the integrator needs (its queue head / worst-status
 * counters, the launch order of the cells and the histogram of the counting sort that produces it) sits in ONE
 * file-scope device array of the library, sizeof = 256 + 4 STEV_STATIC_MAX_CELLS + 16,640 bytes (about 1.02 MiB), which
 * every GPU that loads the library holds until the process exits.  The call allocates nothing (no cudaMalloc, cudaFree
 * or allocating library routine): it clears the counters with cudaMemsetAsync, rewrites the launch order in full and
 * launches the lock-step kernel of stev_integrate (same arithmetic, bit-identical results).
 *   - n_cells > STEV_STATIC_MAX_CELLS: STEV_EINVAL (split the field, or use stev_integrate with your own workspace).
 *   - Only what the lock-step kernel takes: chunk_steps = 0, lanes_per_cell 0 / 512 / 513, at most two factors per
 *     reaction side, integer coefficients; otherwise STEV_EINVAL.
 *   - Every call on a device shares the array, and it keeps the previous call's contents.  Calls that overlap on the
 *     same GPU (two streams, two host threads) RACE on it: serialise them (one stream, or an event between them).
 *   - p->nonblocking = 1 only enqueues and returns STEV_OK; read the per-cell status_out after synchronising.
 * All other arguments, layouts and return codes are those of stev_integrate. */
#define STEV_STATIC_MAX_CELLS 262144
STEV_API int stev_integrate_static(const stev_mechanism *m, const stev_estimator *estimator, const stev_params *p,
                          int64_t n_cells, int64_t ld, double *T, const double *pressure, double *Y, double dt_cfd,
                          int32_t *steps_out, uint8_t *status_out, void *cuda_stream);

/* Same call with HOST buffers (the paper's calling convention: the CFD code hands over host
 * memory and gets the state back): allocates device buffers, copies in, integrates, copies out. */
STEV_API int stev_integrate_host(const stev_mechanism *m, const stev_estimator *estimator, const stev_params *p,
                        int64_t n_cells, int64_t ld, double *T, const double *pressure, double *Y, double dt_cfd,
                        int32_t *steps_out, uint8_t *status_out);

STEV_API void stev_last_stats(stev_stats *out);

/* Test exports (device pointers, same layouts). */
/* Right-hand side only: dYdt [S][ld], dTdt [n], q [R][ld]; rOF [R][ld] or NULL (= ones).  PAPER.md:61-67, 93, 212-218. */
STEV_API int stev_rates_eval(const stev_mechanism *m, const stev_estimator *estimator, const stev_params *p, int64_t n_cells,
                    int64_t ld, const double *T, const double *pressure, const double *Y, const double *rOF,
                    double *dYdt, double *dTdt, double *q, void *cuda_stream);
/* Estimator forward pass: X [n][n_in] raw inputs (float, device), out [n][n_out] (float, device).  PAPER.md:126.
 * The STEV_PREC_FP32 kernel keeps the network and a tile of 128 rows in shared memory:
 * 4 (n_params + 128 (n_in + n_hidden + n_out + 2)) bytes, n_params = n_hidden (n_in + 1) + n_out (n_hidden + 1) + 2 n_in,
 * must fit 227 KB, else STEV_EINVAL: the largest sizes the descriptor admits (64-128-256: 387 KB) do not, 22-64-40
 * (80 KB) and 1-32-106 do.  The TF32 / BF16 paths have their own bound (weight image + one input and one output tile
 * within 200 KB of shared memory, accumulators within 512 tensor-memory columns) and return STEV_EINVAL beyond it. */
STEV_API int stev_estimator_eval(const stev_estimator *e, int64_t n, const float *X, float *out, int32_t precision,
                        void *cuda_stream);
/* Variable-load compaction: list_out = [list_in[k] (or k if list_in is NULL) for k in 0..n-1 if
 * flags[k] != 0], order preserved; *count_out (device int32) = its length.  scratch: device, >= 4*(n/1024+2) bytes. */
STEV_API int stev_compact_active(const uint8_t *flags, const int32_t *list_in, int32_t n, int32_t *list_out,
                        int32_t *count_out, void *scratch, size_t scratch_bytes, void *cuda_stream);
/* |DFT| magnitudes of 13-sample windows (Eq 9): ring [n][13] device -> D [n][7] device (bins 0..6). */
STEV_API int stev_dft_mag(const double *ring, int64_t n, double *D, void *cuda_stream);
/* The arithmetic contract's exp / log on device arrays. */
STEV_API int stev_contract_exp_log(const double *x, int64_t n, double *exp_out, double *log_out, void *cuda_stream);
/* Microbenchmarks used for the roofline denominators: kind 0 runs 8 x `iters` independent DFMAs per thread on a full
 * grid, kind 1 4 x `iters` contract exps; kind 2 runs one dependent chain of 8 x `iters` DFMAs in one warp per SM (a
 * latency probe: ops per second per thread = clock / DFMA latency).  Returns operations per second in *ops_per_s. */
STEV_API int stev_microbench(int32_t kind, int32_t iters, double *ops_per_s, void *cuda_stream);

STEV_API const char *stev_last_error(void); /* thread-local, valid until the next call on this thread */
STEV_API const char *stev_version(void);

#ifdef __cplusplus
}
#endif
#endif /* STEV_H */
