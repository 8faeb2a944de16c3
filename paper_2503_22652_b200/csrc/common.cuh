// Internal definitions shared by the translation units of librchfsi.so.
// Nothing here is visible across the C ABI (include/rchfsi.h).
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <cuda_bf16.h>
#include <cublas_v2.h>
#include <cusolverDn.h>
#include <stdint.h>
#include <map>
#include <string>
#include <vector>
#include "rchfsi.h"

// Timing probes that switch parts of the tensor-core kernels off (RCHFSI_TC_DEBUG) exist only in builds
// with -DRCHFSI_PROBES; the shipped library compiles them out (PROBE folds to 0).
#ifdef RCHFSI_PROBES
#define PROBE(mode, bits) ((mode) & (bits))
#else
#define PROBE(mode, bits) 0
#endif

namespace rchfsi {

// One recurrence step's scalars, Alg. 3 loop body:
//   out = a * T * (dinv_out ? dinv[i] : 1) + b * RY + cp * RX + (has_G ? a * G * LY[j] : 0)
struct StepCoef {
  double a, b, cp;
};

// Low-precision device copy of an operator for the tensor-core paths.
struct LowpCopy {
  int prec = -1;          // RCHFSI_TF32 / RCHFSI_BF16 / RCHFSI_FP32
  bool folded = false;    // columns pre-scaled by dinv (A * diag(dinv))
  bool stale = false;     // rchfsi_operator_changed: the buffer stays, its contents are rebuilt on the next use
  void *data = nullptr;   // dense: [m_pad][k_pad]; FE: [n_cells][a_pad][k_pad]
  int64_t ld = 0;         // padded K extent (elements)
  int64_t rows_pad = 0;   // padded row extent per matrix
  size_t bytes = 0;
};

// Cached TMA descriptor (encoding one costs microseconds of host time per step otherwise).
struct TmapEntry {
  const void *base;
  uint64_t rows, cols, pitch;
  uint32_t box_cols, box_rows;
  int elem_bytes, bf16, atom32;
  CUtensorMap map;
};

// Test / tuning knobs, read from the environment ONCE in rchfsi_create (never on the per-step launch path).
struct Knobs {
  bool fe_shadow_pair = false;   // RCHFSI_FE_SHADOW_PAIR: two operand-shadow buffers instead of the in-place one
  bool fe_legacy = false;        // RCHFSI_FE_LEGACY: the one-tile-per-CTA FE kernel also for BF16 (A/B against the pipelined one)
  int dense_bn = 0;              // RCHFSI_DENSE_BN: 64 / 128 / 256, 0 = automatic
  int dense_ks = 0;              // RCHFSI_DENSE_KS: K splits 1 / 2 / 4 / 8, 0 = automatic
  int dense_mc = -1;             // RCHFSI_DENSE_MC: operator-tile multicast on / off, -1 = automatic
  int rr_chunked = -1;           // RCHFSI_RR_CHUNKED: force the memory-light Rayleigh-Ritz on / off
  bool rr_fe_simt = false;       // RCHFSI_RR_FE_SIMT: FE applies of the Rayleigh-Ritz through the hand-written FP64 kernel
  bool rr_fe_batched = false;    // RCHFSI_RR_FE_BATCHED: shared cell matrix through the batched GEMM as well (A/B knob)
  bool rr_timing = false;        // RCHFSI_RR_TIMING: print phase times of the Rayleigh-Ritz to stderr
  int rr_split = -1;             // RCHFSI_RR_SPLIT: rotation X = Y E on the INT8 tensor pipe (rr_i8.cu): 0 off, 1 forced, -1 = automatic
  int rr_gram_i8 = -1;           // RCHFSI_RR_GRAM_I8: Gram products Y^T (Op Y) on the INT8 tensor pipe: 0 off, 1 forced, -1 = automatic
  int rr_i8_bn = 128;            // RCHFSI_RR_I8_BN: 128 = two-pass N_mma = 128 kernel (default), 64 = single-pass N_mma = 64 kernels
  int rr_i8_rows = 0;            // RCHFSI_RR_I8_ROWS: cap on the rows of one digit-plane chunk (tests: forces several chunks)
  int host_chunk = 0;            // RCHFSI_HOST_CHUNK: column-chunk width of rchfsi_filter_host (multiple of 128), 0 = automatic
  int tc_debug = 0;              // RCHFSI_TC_DEBUG (only in -DRCHFSI_PROBES builds)
};

// rr_i8.cu: a device buffer lent for digit planes, and the planes of the column-slab Gram products
struct I8Buf { void *ptr; size_t bytes; };
struct I8GramState { bool active = false; int8_t *yp[7] = {}, *zp[7] = {}; int64_t Rp = 0; int32_t max_w = 0; };

// How rchfsi_filter lays out its blocks for (operator, block width, options): which fused kernel runs, which
// precision the operand block has, whether an operand shadow exists.  Decided from the descriptor alone so that
// rchfsi_workspace_bytes can plan without a handle.
struct Plan {
  int store;     // storage precision of R_X, R_Y, G
  int operand;   // precision of the block the operator kernel reads
  int tprec;     // precision of the unfused operator output T
  bool shadow;   // operand block is a separate buffer
  int fused;     // 0 unfused SIMT, 1 CSR fused, 2 dense tensor-core, 3 FE tensor-core
  bool panel;    // library-owned blocks in panel layout [ceil(N/128)][m][128] (FE tensor-core path)
  bool shadow_inplace;   // one shadow buffer, overwritten in place by the fused FE step
};
struct Knobs;
Plan make_plan(const rchfsi_operator &A, int32_t N, const rchfsi_options &opt, const Knobs &kn);

// State of a filter call between rchfsi_filter_begin and rchfsi_filter_end (rchfsi_filter runs the three in one go;
// the step-wise entry points exist so that a row-sharded caller can exchange interface rows between the steps)
struct FilterRun {
  bool active = false;
  bool chfsi = false, gf32 = false;
  Plan pl{};
  double *X = nullptr;
  int32_t degree = 0, k = 0;            // k = index of the NEXT step to run (2 .. degree)
  double e = 0, c = 0, sigma1 = 0, gamma = 0, sigma = 0;
  void *RX = nullptr, *RY = nullptr, *Wcur = nullptr, *Wnext = nullptr;
  const void *Gst = nullptr;
  bool g_lib = false;                   // Gst is the library's copy (library layout); else the caller's row-major block
  uint64_t apply_index = 0;
  StepCoef last{};                      // coefficients of the step that ran last
  const double *last_LY = nullptr;      // its Lambda_Y row
};

// A piece of caller-provided device memory the handle carves its buffers from (rchfsi_add_workspace)
struct WorkspaceSegment {
  char *base;
  size_t size, used;
};

struct DeviceOperator {
  rchfsi_operator d{};    // caller's descriptor (device pointers, borrowed)
  bool present = false;
};

// FE colouring (host-built at create): cells of one colour share no node.
struct FeColoring {
  int n_colors = 0;
  std::vector<int64_t> color_begin;   // [n_colors + 1] into cell_order
  int32_t *cell_order = nullptr;      // device [n_cells], cells grouped by colour
  uint8_t *flags = nullptr;           // device [n_cells][n_loc]: bit0 first toucher, bit1 last toucher
  std::vector<int32_t> h_order;       // host copies, built (and the mesh validated) in rchfsi_create; uploaded into the
  std::vector<uint8_t> h_flags;       // workspace on first use
};

}  // namespace rchfsi

struct rchfsi_ctx {
  rchfsi::DeviceOperator A, B;
  const double *dinv = nullptr;
  int64_t m = 0;
  int32_t N = 0;        // ACTIVE block width of the current call (= N_cap except inside a column chunk of filter_host)
  int32_t N_cap = 0;    // block width the handle was created for: every workspace block is sized for it
  rchfsi_options opt{};
  cudaStream_t stream = nullptr;
  cublasHandle_t cublas = nullptr;
  cusolverDnHandle_t cusolver = nullptr;
  std::string err;
  int64_t launches = 0;
  int num_sms = 0;                       // multiprocessors of the current device (persistent-kernel grids)

  // filter workspace (storage precision), lazily allocated
  void *RX = nullptr, *RY = nullptr;      // [m][N] store_prec
  void *Gs = nullptr;                     // [m][N] store_prec copy of G (store FP32 only)
  void *Wa = nullptr, *Wb = nullptr;      // operand-precision shadows of R_Y (when needed)
  void *T = nullptr;                      // [m][N] operator output for the unfused paths
  double *Gtmp = nullptr;                 // [m][N] FP64 when G == NULL is computed here
  double *lam_table = nullptr;            // [(p_max+1)][N]
  int32_t lam_table_p = 0;
  double *colnorm = nullptr;              // [2][N]
  std::vector<rchfsi::LowpCopy> lowp;
  std::vector<rchfsi::TmapEntry> tmaps;
  rchfsi::Knobs knobs;
  std::map<const void *, int> func_smem;   // per handle (= per device): dynamic shared memory opted in per kernel
  rchfsi::FeColoring coloring;

  // Rayleigh-Ritz workspace
  double *rr1 = nullptr, *rr2 = nullptr, *rr3 = nullptr;   // [m][N] FP64
  double *rrc1 = nullptr, *rrc2 = nullptr, *rrp = nullptr; // chunked variant: [m][cw] x 2, [rp][N]
  int32_t rr_cw = 0; int64_t rr_rp = 0;
  float *Gsolve32 = nullptr;                               // [m][N] FP32 residual block of rchfsi_solve (chunked mode)
  double *feg_W = nullptr, *feg_T = nullptr, *feg_A = nullptr;  // fe_rr.cu scratch: gathered operand, product, FP64 cell batch
  const double **feg_ptrs = nullptr;                        // [3][feg_ptr_cap] pointer arrays of the batched GEMM
  const double *feg_A_full = nullptr;                       // FP64 copy of all FP32 cell matrices, lent for one Rayleigh-Ritz
  size_t feg_w_bytes = 0, feg_W_bytes = 0, feg_T_bytes = 0; int64_t feg_a_cells = 0, feg_ptr_cap = 0; int32_t feg_N = 0;
  double *Ha = nullptr, *Hb = nullptr;                     // [N][N]
  void *i8_cols = nullptr, *i8_hpart = nullptr; size_t i8_hpart_bytes = 0;   // rr_i8.cu: column maxima / exponents, K-split partial Gram sums
  rchfsi::I8GramState i8g;                                  // transposed digit planes of Y of the memory-light Rayleigh-Ritz
  size_t RX_bytes = 0, RY_bytes = 0, Wa_bytes = 0;        // sizes of the filter's blocks (lent to the Rayleigh-Ritz between filters)
  void *i8_E = nullptr;                                    // rr_i8.cu: digit planes + exponents of the eigenvector matrix
  double *ritz_dev = nullptr, *res_dev = nullptr;          // [N]
  double *sy_work = nullptr; int sy_lwork = 0; int *sy_info = nullptr;

  // host-buffer entry point (rchfsi_filter_host): column chunks of the block travel host -> device on in_stream,
  // are filtered on the main stream and return on out_stream, three staging sets in rotation.  Alg. 3 reads X only
  // in its last line, so the main stream waits for the chunk's X (ev_x) only before the finish kernel.
  static constexpr int HOST_SETS = 3;
  double *hX[HOST_SETS] = {nullptr, nullptr, nullptr};
  void *hG[HOST_SETS] = {nullptr, nullptr, nullptr};
  double *hritz = nullptr;
  int32_t host_chunk = 0;                  // staging width (columns) the sets were allocated for
  cudaStream_t in_stream = nullptr, out_stream = nullptr;
  cudaEvent_t ev_g[HOST_SETS] = {nullptr, nullptr, nullptr}, ev_xin[HOST_SETS] = {nullptr, nullptr, nullptr},
              ev_done[HOST_SETS] = {nullptr, nullptr, nullptr}, ev_free[HOST_SETS] = {nullptr, nullptr, nullptr};
  cudaEvent_t ev_x = nullptr;              // the X event the running filter has to wait for (one of ev_xin)
  bool x_pending = false;

  // rchfsi_estimate_bounds scratch (bounds.cu)
  double *bnd_buf = nullptr, *bnd_cell = nullptr, *bnd_work = nullptr;

  rchfsi::FilterRun run;
  // interface exchange of a row-sharded filter (interface.cu): saved old R_X rows and the recomputed base term
  void *if_old = nullptr, *if_base = nullptr;
  size_t if_cap = 0, if_old_cap = 0, if_base_cap = 0;   // rows x N_cap elements the buffers hold

  // instrumentation
  cudaEvent_t ev_step0 = nullptr, ev_step1 = nullptr;
  int32_t last_steps = 0;

  // caller-provided workspace (rchfsi_add_workspace): every device buffer of the handle is carved from these
  // segments; the library itself never calls cudaMalloc
  std::vector<rchfsi::WorkspaceSegment> segments;
  size_t shortfall = 0;        // bytes of the allocation that did not fit (rchfsi_workspace_shortfall)
  size_t ws_used = 0;          // bytes handed out so far
};

namespace rchfsi {

#define RCHFSI_CUDA_CHECK(h, expr)                                                        \
  do {                                                                                    \
    cudaError_t _e = (expr);                                                              \
    if (_e != cudaSuccess) {                                                              \
      (h)->err = std::string(#expr) + ": " + cudaGetErrorString(_e);                      \
      return (_e == cudaErrorMemoryAllocation) ? RCHFSI_ENOMEM : RCHFSI_ECUDA;            \
    }                                                                                     \
  } while (0)

#define RCHFSI_TRY(expr)                        \
  do {                                          \
    rchfsi_status _s = (expr);                  \
    if (_s != RCHFSI_OK) return _s;             \
  } while (0)

rchfsi_status dev_alloc(rchfsi_ctx *h, void **p, size_t bytes);
// cudaFuncSetAttribute(MaxDynamicSharedMemorySize) once per (handle, kernel)
rchfsi_status ensure_func_smem(rchfsi_ctx *h, const void *func, int bytes);
static inline int64_t cdiv(int64_t a, int64_t b) { return (a + b - 1) / b; }

#define LAUNCH_CHECK(h)                                                                   \
  do {                                                                                    \
    (h)->launches++;                                                                      \
    cudaError_t _e = cudaGetLastError();                                                  \
    if (_e != cudaSuccess) {                                                              \
      (h)->err = std::string("kernel launch: ") + cudaGetErrorString(_e) + " at " +      \
                 __FILE__ + ":" + std::to_string(__LINE__);                               \
      return RCHFSI_ECUDA;                                                                \
    }                                                                                     \
  } while (0)

inline size_t prec_bytes(int prec) {
  return prec == RCHFSI_FP64 ? 8 : (prec == RCHFSI_BF16 ? 2 : 4);
}

// ---- kernels_simt.cu ------------------------------------------------------------------
// T = A * (dinv_in ? diag(dinv) : I) * W for W, T of element type TW / TO in {double, float}.
// For FE the output is accumulated with atomics into a zeroed T.
template <typename TC>
rchfsi_status op_apply_simt(rchfsi_ctx *h, const rchfsi_operator &op, const double *dinv_in,
                            const TC *W, TC *T, int32_t N, int64_t ldw = 0, int64_t ldt = 0);

// Lambda_k table, k = 0..p (eq. (12)): table[k][j].
rchfsi_status lambda_table(rchfsi_ctx *h, const double *ritz, int32_t N, int32_t p, double e,
                           double c, double sigma1, double *table);

// Element-wise pieces of Alg. 2 / Alg. 3 (storage type S, operand shadow type O, T type TT).
struct StepArgs {
  StepCoef k;
  const void *T;        // operator output
  const void *RY;       // storage
  void *RX;             // storage, in: R_X (old), out: R_X (new)
  const void *G;        // storage or NULL
  const double *LY;     // Lambda_Y row of the table (device) or NULL
  const double *dinv_out;  // CHFSI: row scaling of T, else NULL
  void *Wnext;          // operand-precision shadow of the new block, or NULL
  int64_t m;
  int32_t N;
};
rchfsi_status step_elementwise(rchfsi_ctx *h, int store_prec, int t_prec, int shadow_prec,
                               const StepArgs &a);
// dst(store) = alpha * src(FP64) (+ shadow), used for R_Y = (sigma_1/e) G and G copies
rchfsi_status scale_convert(rchfsi_ctx *h, int store_prec, int shadow_prec, double alpha,
                            const void *src, void *dst, void *shadow, int64_t m, int32_t N, int64_t pm = 0,
                            int src_prec = RCHFSI_FP64);
// CHFSI first step: Y = alpha * (dinv * T - c X)
rchfsi_status chfsi_first(rchfsi_ctx *h, int store_prec, int t_prec, int shadow_prec, double alpha,
                          double c, const void *T, const double *dinv, const double *X, void *Y,
                          void *shadow, int64_t m, int32_t N);
// RCHFSI finish: X = dinv * RY + X * LY (PAPER.md:263 last line); CHFSI finish: X = RY
rchfsi_status finish_block(rchfsi_ctx *h, int store_prec, const void *RY, const double *dinv,
                           const double *LY, double *X, int64_t m, int32_t N, int64_t pm = 0);
// column 2-norms (sum of squares accumulated in FP64 with atomics into a zeroed array)
rchfsi_status column_sumsq(rchfsi_ctx *h, int prec, const void *V, int64_t m, int32_t N,
                           double *sumsq);
rchfsi_status scale_columns_inv_norm(rchfsi_ctx *h, double *V, int64_t m, int32_t N,
                                     const double *sumsq);
// T_j += eps ||T_j|| g_j / ||g_j||, g = counter-based Gaussian (S11)
rchfsi_status add_column_noise(rchfsi_ctx *h, int t_prec, void *T, int64_t m, int32_t N, double eps,
                               uint64_t seed, uint64_t apply_index, double *scratch2N);
// G = AX - BX diag(ritz), res_j = ||G_j||
rchfsi_status residual_block(rchfsi_ctx *h, const double *AX, const double *BX, const double *ritz,
                             double *G, double *res, int64_t m, int32_t N);
rchfsi_status residual_window(rchfsi_ctx *h, const double *AX, int64_t lda, const double *BX, int64_t ldb,
                              const double *ritz, void *G, int64_t ldg, int g_prec, double *res2, int64_t m, int32_t w);
rchfsi_status sqrt_inplace(rchfsi_ctx *h, double *v, int32_t N);
rchfsi_status symmetrize(rchfsi_ctx *h, double *H, int32_t N);
rchfsi_status fe_check_symmetric(rchfsi_ctx *h, const rchfsi_operator &op, double *max_asym_host);

// ---- fused paths (return RCHFSI_EINVAL if the configuration is not supported so the caller
// can fall back to the unfused sequence) -------------------------------------------------
struct FusedStep {
  StepCoef k;
  const void *W;        // operand block (shadow or R_Y itself)
  const void *RY;
  void *RX;
  const void *G;
  const double *LY;
  void *Wnext;
  int apply_prec, store_prec;
  bool chfsi;           // dinv applied to the output rows instead of the input
  bool g_rowmajor;      // G is the caller's row-major [m][N] block even though R_X / R_Y use the panel layout
};
bool csr_fused_supported(const rchfsi_operator &A, int32_t N, const rchfsi_options &opt);
rchfsi_status csr_fused_step(rchfsi_ctx *h, const FusedStep &s);
bool dense_tc_supported(const rchfsi_operator &A, int32_t N, const rchfsi_options &opt);
rchfsi_status dense_tc_step(rchfsi_ctx *h, const FusedStep &s);
bool fe_tc_supported(const rchfsi_operator &A, int32_t N, const rchfsi_options &opt);
// bytes of the reduced-precision operator copy each fused path keeps (0 when the path does not apply)
size_t csr_lowp_bytes(const rchfsi_operator &A);
size_t dense_lowp_bytes(const rchfsi_operator &A, int prec);
size_t fe_lowp_bytes(const rchfsi_operator &A, int prec);
// scratch of the batched-GEMM FE applies of the Rayleigh-Ritz for an N-column block
size_t fe_rr_scratch_bytes(const rchfsi_operator &op, int32_t N, int64_t max_cells_per_colour);
rchfsi_status fe_tc_step(rchfsi_ctx *h, const FusedStep &s);
// allocate (and build) what the fused step of this plan needs before the first step: rchfsi_solve calls them up front,
// so that a workspace that is too small shows as ENOMEM before any caller block has been changed
rchfsi_status csr_fused_prepare(rchfsi_ctx *h, bool chfsi);
rchfsi_status dense_tc_prepare(rchfsi_ctx *h, int apply_prec, bool chfsi);
rchfsi_status fe_tc_prepare(rchfsi_ctx *h, int apply_prec, bool chfsi);

// ---- fe_rr.cu / fe_tc.cu ---------------------------------------------------------------
rchfsi_status fe_build_coloring(rchfsi_ctx *h);    // host side: colours, order, flags; validates conn (create time)
rchfsi_status fe_ensure_coloring(rchfsi_ctx *h);   // device side: uploads order and flags into the workspace (first use)
bool fe_apply_gemm_supported(const rchfsi_ctx *h, const rchfsi_operator &op);
// T = Op W in FP64 through gather -> batched DGEMM -> coloured scatter (Rayleigh-Ritz only)
rchfsi_status fe_apply_gemm(rchfsi_ctx *h, const rchfsi_operator &op, const double *W, double *T, int32_t N,
                            int64_t ldw = 0, int64_t ldt = 0);
size_t fe_rr_fp64_cells_bytes(const rchfsi_ctx *h);            // 0 unless A is an FP32-only FE operator
rchfsi_status fe_rr_lend_fp64_cells(rchfsi_ctx *h, void *buf); // valid until the caller resets h->feg_A_full

// ---- rr.cu -----------------------------------------------------------------------------
rchfsi_status rayleigh_ritz_impl(rchfsi_ctx *h, double *Y, double *ritz_out, double *G_out,
                                 double *res_out);
// Memory-light variant (SURVEY 8(d) config-5 plan): Gram matrices over column chunks, rotation by row panels in
// place, residual block recomputed per column chunk and written in g_prec (FP64 or FP32).
rchfsi_status rayleigh_ritz_chunked(rchfsi_ctx *h, double *Y, double *ritz_out, void *G_out, int g_prec,
                                    double *res_out);
bool rr_wants_chunked(rchfsi_ctx *h);
rchfsi_status rotate_in_place(rchfsi_ctx *h, double *Y, const double *E);   // rchfsi_rotate
rchfsi_status rr_preallocate(rchfsi_ctx *h, bool chunked);                  // every buffer of a Rayleigh-Ritz, nothing computed
rchfsi_status fe_rr_preallocate(rchfsi_ctx *h, const rchfsi_operator &op, int32_t N);
rchfsi_status rr_i8_preallocate(rchfsi_ctx *h, bool chunked, int32_t cw);

// ---- rr_i8.cu: rotation X = Y E on the INT8 tensor pipe (error-free digit split of the FP64 operands) ----
bool rotate_i8_supported(const rchfsi_ctx *h);
bool rr_i8_scratch_ok(const rchfsi_ctx *h, size_t bytes);   // enough scratch for one 128-row chunk of digit planes
size_t rotate_i8_fixed_bytes(int32_t N);        // digit planes of E, held by the handle
// Out[r][:] = In[r][:] E for r < rows (E column-major N x N); Out may be In; `scratch` holds one row chunk's planes
rchfsi_status rotate_i8(rchfsi_ctx *h, const double *In, int64_t rows, const double *E, double *Out, void *scratch,
                        size_t scratch_bytes);
// Gram products H = Y^T Z (lower triangle, column-major) with the same digit split, contraction over the rows
bool gram_i8_supported(const rchfsi_ctx *h);
size_t rr_i8_plan_bytes(int64_t m, int32_t N);   // digit planes of E, column exponents, K-split partial sums
rchfsi_status gram_i8_full(rchfsi_ctx *h, const double *Y, const double *AY, const double *BY, double *Ha, double *Hb,
                           void *scratch, size_t scratch_bytes);
bool carve_buf(std::vector<I8Buf> &bufs, size_t bytes, void **out);   // first fit, 256-byte aligned; consumes what it returns
bool gram_i8_begin(rchfsi_ctx *h, const double *Y, std::vector<I8Buf> &bufs, int32_t max_w, rchfsi_status *st);
rchfsi_status gram_i8_slab(rchfsi_ctx *h, const double *Y, const double *Z1, const double *Z2, int64_t ldz, int32_t w, int32_t zc0,
                           double *Ha, double *Hb);

}  // namespace rchfsi
