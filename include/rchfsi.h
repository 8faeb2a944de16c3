/* rchfsi.h -- C ABI of the B200-native R-ChFSI filter library.
 *
 * Method: "Residual-based Chebyshev filtered subspace iteration for Hermitian
 * eigenvalue problems tolerant to inexact matrix-vector products" (arxiv 2503.22652).
 * Citations are PAPER.md:LINE of the paper text this library was written from.
 *
 * Notation (SURVEY.md notation warning): the problem is
 * A u = lambda B u with A Hermitian (real symmetric here), B SPD, m = matrix dimension,
 * n_wanted = number of wanted lowest eigenpairs, N = block width (>= n_wanted),
 * p = Chebyshev degree.  D^-1 is a cheap diagonal approximation of B^-1 (PAPER.md:164,
 * 325) used ONLY inside the filter recurrence.
 *
 * Conventions
 *  - Every function returns an rchfsi_status; nothing throws across the ABI.
 *    rchfsi_last_error(handle) returns a static/handle-owned message for the last failure.
 *  - Pointers documented "device" are CUDA device pointers on the current device and are
 *    OWNED BY THE CALLER.  The library BORROWS the operator arrays and dinv_diag for the
 *    lifetime of the handle and X / ritz / G for the duration of the call.  Pointers
 *    documented "host" are ordinary host pointers.
 *  - Blocks of vectors are row-major [m][N] with the N columns contiguous (one row of N
 *    values per matrix row), FP64, 16-byte aligned.
 *  - All device work is enqueued on the cudaStream_t given at create time (passed as
 *    void*, NULL = the legacy default stream).  rchfsi_filter and rchfsi_rayleigh_ritz are
 *    asynchronous with respect to the host; rchfsi_solve and the *_host entry points
 *    synchronise the stream before returning.
 *  - The library never allocates device memory.  Its workspace (recurrence blocks, reduced-
 *    precision operator copies, Rayleigh-Ritz temporaries, staging of the host entry point)
 *    is carved from caller-provided device buffers (rchfsi_add_workspace; e.g. torch tensors).
 *    rchfsi_workspace_bytes plans the size of a single sufficient buffer up front; a call that
 *    runs out returns RCHFSI_ENOMEM before it has changed any caller block, reports the missing
 *    bytes (rchfsi_workspace_shortfall) and may simply be repeated after adding a segment.
 *  - There is no CPU fallback: without a CUDA device every compute entry point returns
 *    RCHFSI_ECUDA.
 */
#ifndef RCHFSI_H
#define RCHFSI_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct rchfsi_ctx *rchfsi_handle;

typedef enum {
  RCHFSI_OK = 0,
  RCHFSI_EINVAL = 1,         /* bad argument; outputs untouched */
  RCHFSI_ENOMEM = 2,         /* the workspace is exhausted (rchfsi_workspace_shortfall), or malloc failed */
  RCHFSI_ECUDA = 3,          /* CUDA / cuBLAS / cuSOLVER runtime error, or no device */
  RCHFSI_ENOTCONVERGED = 4,  /* rchfsi_solve hit max_iter; outputs hold the last iterate */
  RCHFSI_EBREAKDOWN = 5      /* Rayleigh-Ritz Gram matrix Y^T B Y not numerically SPD */
} rchfsi_status;

typedef enum { RCHFSI_OP_DENSE = 0, RCHFSI_OP_CSR = 1, RCHFSI_OP_FE = 2 } rchfsi_opkind;

/* Precision of the operator apply A (x) V inside the filter ("the
 * computation of A D^-1 R_Y is done using FP32 arithmetic", TF32 compute mode, BF16).
 * FP64: exact products (parity mode).  FP32: FP32 operands, FP32 FMA on the ALUs.
 * TF32 / BF16: tensor-core operands, FP32 accumulate (dense and FE operators; a CSR
 * operator runs TF32 and BF16 requests as FP32: the sparse product is on the ALUs). */
typedef enum { RCHFSI_FP64 = 0, RCHFSI_FP32 = 1, RCHFSI_TF32 = 2, RCHFSI_BF16 = 3 } rchfsi_prec;

/* RCHFSI_METHOD_CHFSI: Algorithm 2 with H = D^-1 (A (x) .)  (eq. (7) at 170).
 * RCHFSI_METHOD_RCHFSI: Algorithm 3, the recurrence on residuals. */
typedef enum { RCHFSI_METHOD_CHFSI = 0, RCHFSI_METHOD_RCHFSI = 1 } rchfsi_method;

/* A linear operator on R^m.  All arrays are device pointers, FP64 master copies.
 *  DENSE: `dense` row-major m x m with leading dimension lda (>= m), symmetric.
 *  CSR  : rowptr[m+1] (int64), colind[nnz] (int32, any order within a row), vals[nnz].
 *  FE   : A V = sum_c P_c^T A_c P_c V (Remark 4.1): conn[n_cells][n_loc]
 *         holds the global row of each local node (distinct within a cell);
 *         cell_mats is [n_cells][n_loc][n_loc], or ONE [n_loc][n_loc] matrix shared by
 *         every cell when cell_shared != 0.  Every cell matrix must be symmetric (it is
 *         the element matrix of a symmetric form; A is Hermitian): the
 *         kernels read A_c[b][a] for A_c[a][b].  rchfsi_create verifies this, and that
 *         every row 0..m-1 occurs in conn (EINVAL otherwise: a row no cell touches has
 *         no place in the coloured scatter).
 *         cell_mats_f32, if non-NULL, is the same array in FP32 and may be given INSTEAD
 *         of cell_mats (cell_mats == NULL) when the FP64 copy does not fit (config 5:
 *         13 GB); it is then also what the FP64 Rayleigh-Ritz path reads (widened). */
typedef struct {
  int32_t kind;               /* rchfsi_opkind */
  int64_t m;
  const double *dense;
  int64_t lda;
  const int64_t *rowptr;
  const int32_t *colind;
  const double *vals;
  int64_t nnz;
  int64_t n_cells;
  int32_t n_loc;
  int32_t cell_shared;
  const double *cell_mats;
  const float *cell_mats_f32;
  const int32_t *conn;
} rchfsi_operator;

typedef struct {
  int32_t apply_prec;         /* rchfsi_prec of the operator apply inside the filter */
  int32_t store_prec;         /* RCHFSI_FP64 or RCHFSI_FP32: storage of R_X, R_Y and of the
                                 filter's copy of G (PAPER.md:341 stores them in FP32) */
  int32_t normalize_columns_before_rr; /* scale columns of Y_p to unit 2-norm before the
                                 Gram matrices (reading S6); default 1 */
  int32_t adaptive_bounds;    /* rchfsi_solve: after each Rayleigh-Ritz set lam_T to the
                                 largest and lam_min to the smallest Ritz value (S7) */
  double noise_eps;           /* > 0: debug hook, per-matvec column-scaled Gaussian error
                                 T_j += eps ||T_j|| g_j/||g_j|| inside the filter only
                                 (BASELINE.json configs[0]; reading S11) */
  uint64_t noise_seed;
  int32_t allow_high_degree;  /* the filter refuses degree >= 100 with a reduced-precision apply (the paper finds p = 100,
                                 120 unstable in FP32 / TF32, PAPER.md:347-359 and footnote 5) unless this is set */
  int32_t g_input_f32;        /* nonzero: the G argument of rchfsi_filter points to FP32 values [m][N] (an FP64
                                 residual block does not fit at config 5, SURVEY 8(d) memory plan); needs
                                 store_prec FP32; G is then read in place, no copy is made */
} rchfsi_options;

/* Fill `opt` with the defaults: apply FP64, store FP64, normalize 1, everything else 0. */
void rchfsi_default_options(rchfsi_options *opt);

/* Create a solver context for A x = lambda B x.
 *  A          operator (borrowed).
 *  B          operator or NULL for B = I (the standard problem).
 *  dinv_diag  device, length m: diagonal of D^-1 ~ B^-1; NULL => I.
 *  block_N    block width N (1 <= N <= m).
 *  opt        NULL => defaults.
 *  cuda_stream cudaStream_t as void*.
 * Errors: EINVAL (null/ill-sized arguments, unknown kind/precision, non-symmetric FE cell
 * matrices), ECUDA (no device), ENOMEM. */
rchfsi_status rchfsi_create(rchfsi_handle *out, const rchfsi_operator *A,
                            const rchfsi_operator *B, const double *dinv_diag,
                            int32_t block_N, const rchfsi_options *opt, void *cuda_stream);

rchfsi_status rchfsi_destroy(rchfsi_handle h);

/* The CONTENTS of the operator arrays and of dinv_diag are borrowed too: the filter keeps reduced-precision
 * copies of A (with D^-1 folded in) that are built on first use.  When the caller updates A or dinv_diag in
 * place (the A of an SCF iteration evolves), call this before the next filter: it synchronises
 * the stream and drops the copies so that they are rebuilt.  The sparsity pattern / connectivity must not
 * change (make a new handle for that). */
rchfsi_status rchfsi_operator_changed(rchfsi_handle h);

/* Message for the most recent failure on this handle ("" if none); NULL handle => the
 * message of the last failed rchfsi_create in this thread. */
const char *rchfsi_last_error(rchfsi_handle h);

/* Workspace ("the caller (torch) allocates the workspace").
 * rchfsi_workspace_bytes: bytes of ONE device buffer that is sufficient for the entry points named in `uses`
 *   (bit-or of rchfsi_use) with filter degrees up to max_degree; computed from the descriptors alone (no device
 *   needed).  It enumerates the same buffers as the allocation sites; for the memory-light Rayleigh-Ritz of
 *   rchfsi_solve (chosen when three more FP64 blocks do not fit on the device) less is used.
 * rchfsi_add_workspace: hand `bytes` of device memory (borrowed until rchfsi_destroy; any alignment) to the handle.
 *   May be called several times; buffers never span segments.
 * rchfsi_workspace_shortfall: after an RCHFSI_ENOMEM, the size of a segment that lets the failed allocation
 *   succeed (0 otherwise).  rchfsi_workspace_used: bytes handed out so far. */
typedef enum {
  RCHFSI_USE_FILTER = 1, RCHFSI_USE_RAYLEIGH_RITZ = 2, RCHFSI_USE_SOLVE = 4, RCHFSI_USE_FILTER_HOST = 8,
  RCHFSI_USE_BOUNDS = 16,
  RCHFSI_USE_FILTER_NULL_G = 32   /* rchfsi_filter will be called with G == NULL (two more FP64 blocks) */
} rchfsi_use;
size_t rchfsi_workspace_bytes(const rchfsi_operator *A, const rchfsi_operator *B, int32_t block_N,
                              const rchfsi_options *opt, int32_t uses, int32_t max_degree);
rchfsi_status rchfsi_add_workspace(rchfsi_handle h, void *device_buffer, size_t bytes);
size_t rchfsi_workspace_shortfall(rchfsi_handle h);
size_t rchfsi_workspace_used(rchfsi_handle h);

/* The Chebyshev filter (the hot path).
 *  method RCHFSI (Algorithm 3):
 *     R_X = 0, R_Y = (sigma_1/e) G, Lambda_X = I, Lambda_Y = (sigma_1/e)(Lambda - c I);
 *     for k = 2..p:  R_X <- a A (x) (D^-1 R_Y) + b R_Y + c' R_X + a G Lambda_Y,
 *                    Lambda_X <- a Lambda_Y Lambda + b Lambda_Y + c' Lambda_X, swap;
 *     X <- D^-1 R_Y + X Lambda_Y,
 *     with e, c, sigma_1, sigma_{k+1} = 1/(2/sigma_1 - sigma_k), a = 2 sigma_{k+1}/e,
 *     b = -a c, c' = -sigma_k sigma_{k+1}.
 *  method CHFSI (Algorithm 2, PAPER.md:78-86 with eq. (7) at 170):
 *     Y = (sigma_1/e)(D^-1 A (x) X - c X); for k = 2..p: X <- a D^-1 A (x) Y + b Y + c' X, swap.
 *  X      device [m][N] FP64, in: X^(i); out: the filtered block Y_p (overwritten).
 *  ritz   device [N] FP64: diagonal of Lambda^(i) (RCHFSI only; ignored for CHFSI).
 *  G      device [m][N] FP64: A X - B X Lambda computed with the exact
 *         operators; NULL => computed here in FP64 from A, B, X, ritz (RCHFSI only).
 *  degree p >= 1 (p >= 100 with a reduced-precision apply needs allow_high_degree);
 *  lam_min < lam_T < lam_max (a_low <= lambda_1, [a,b] = [lam_T, lam_max]).
 * Asynchronous.  Errors: EINVAL (bad handle / pointers / degree / bounds), ECUDA, ENOMEM. */
rchfsi_status rchfsi_filter(rchfsi_handle h, int32_t method, double *X, const double *ritz,
                            const double *G, int32_t degree, double lam_min, double lam_T,
                            double lam_max);

/* The same filter in three pieces, for callers that must act between the recurrence steps (the row-sharded
 * multi-GPU filter below): rchfsi_filter == rchfsi_filter_begin; (degree - 1) x rchfsi_filter_step; rchfsi_filter_end.
 *  begin  validates, computes the scalars and the Lambda_k table, sets R_X = 0, R_Y = (sigma_1/e) G;
 *  step   one pass of the loop body: the fused operator + recurrence step, then swap(R_X, R_Y);
 *  end    the last line of Algorithm 3, X <- D^-1 R_Y + X Lambda_Y.  EINVAL while steps are left.
 * rchfsi_filter_steps_left: steps still to run (0 when no filter is in progress). */
rchfsi_status rchfsi_filter_begin(rchfsi_handle h, int32_t method, double *X, const double *ritz, const double *G,
                                  int32_t degree, double lam_min, double lam_T, double lam_max);
rchfsi_status rchfsi_filter_step(rchfsi_handle h);
rchfsi_status rchfsi_filter_end(rchfsi_handle h);
int32_t rchfsi_filter_steps_left(rchfsi_handle h);

/* Row-sharded filter: interface exchange ("nearest-neighbour MPI communication ... in BF16 precision; we
 * term this method TF32B"; "reducing inter-node message sizes by a factor of 4").  Each rank (one process
 * per GPU) creates its handle on a SLAB of the operator -- the cells it owns and every row they touch -- so the rows
 * between two slabs exist on both ranks.  A local rchfsi_filter_step leaves on such a row only this rank's share of the
 * product: R_new = base + a T_r with base = b R_Y + c' R_X + a G Lambda_Y equal on both ranks.  Per step:
 *   rchfsi_interface_save(rows)              BEFORE the step: keeps the R_X rows the step will overwrite;
 *   rchfsi_filter_step
 *   rchfsi_interface_pack(rows, wire, send)  send[i][j] = wire(R_new - base), i over `rows`, j < N ([n_rows][N], wire type);
 *   -- the caller swaps `send` with the neighbour rank (NCCL send/recv, torch.distributed) --
 *   rchfsi_interface_apply(rows, wire, own = send, nbr = received)
 *                                            R_new = base + (own + nbr), both in wire precision, so the two replicas
 *                                            of a row stay bit-identical; refreshes the operand shadow of the rows.
 *  rows       device int32[n_rows]: local row indices of ALL interface rows of this rank (a middle rank: both planes;
 *             the caller sends / receives the two halves of the buffers to / from its two neighbours).
 *  wire_prec  RCHFSI_FP64, RCHFSI_FP32 or RCHFSI_BF16: the precision on the wire.  With BF16 the interface rows see an
 *             O(2^-9) relative error in their share of the product: an inexact matvec (Thm 3.4).
 * METHOD_RCHFSI with G given only (Algorithm 3 has no operator apply outside the loop).  Asynchronous.
 * Errors: EINVAL (no filter in progress, bad rows / wire), ENOMEM (workspace), ECUDA. */
rchfsi_status rchfsi_interface_save(rchfsi_handle h, const int32_t *rows, int32_t n_rows);
rchfsi_status rchfsi_interface_pack(rchfsi_handle h, const int32_t *rows, int32_t n_rows, int32_t wire_prec, void *send_buf);
rchfsi_status rchfsi_interface_apply(rchfsi_handle h, const int32_t *rows, int32_t n_rows, int32_t wire_prec,
                                     const void *own_buf, const void *nbr_buf);

/* Same call with HOST buffers: copies X, ritz (and G if non-NULL) to device scratch,
 * runs rchfsi_filter, copies Y_p back into X_host, synchronises.  G_host holds FP64 values,
 * or FP32 values when the handle was created with g_input_f32. */
rchfsi_status rchfsi_filter_host(rchfsi_handle h, int32_t method, double *X_host,
                                 const double *ritz_host, const double *G_host,
                                 int32_t degree, double lam_min, double lam_T, double lam_max);

/* Rayleigh-Ritz on a non-orthogonal basis, all in FP64 with the
 * exact operators: H_a = Y^T A Y, H_b = Y^T B Y, solve H_a E = H_b E Lambda with
 * E^T H_b E = I and ascending eigenvalues, X = Y E.
 *  Y_in_X_out  device [m][N]: in the basis Y (columns scaled to unit 2-norm first when
 *              normalize_columns_before_rr), out the B-orthonormal Ritz vectors X.
 *  ritz_out    device [N]: Ritz values, ascending.
 *  G_out       device [m][N] or NULL: A X - B X diag(ritz) (the input of Algorithm 3).
 *  resnorm_out device [N] or NULL: r_j = ||A x_j - ritz_j B x_j||_2.
 * Asynchronous except for one host read of the cuSOLVER status (EBREAKDOWN). */
rchfsi_status rchfsi_rayleigh_ritz(rchfsi_handle h, double *Y_in_X_out, double *ritz_out,
                                   double *G_out, double *resnorm_out);

/* The subspace rotation of the Rayleigh-Ritz step on its own ("X = Y E"): Y <- Y E in place, FP64.
 *  Y_in_X_out    device [m][N] row-major.
 *  E_colmajor    device N x N, column-major (the LAPACK / cuSOLVER eigenvector layout), not aliasing Y.
 * Same kernel as inside rchfsi_rayleigh_ritz: the INT8 tensor-pipe product of rr_i8.cu (error-free digit split of both
 * operands, result within a few FP64 ulps of (row max of Y) x (column max of E) per element; N <= 16384);
 * RCHFSI_RR_SPLIT=0 selects cuBLAS dgemm instead.  Asynchronous. */
rchfsi_status rchfsi_rotate(rchfsi_handle h, double *Y_in_X_out, const double *E_colmajor);

/* Algorithm 1, do-while reading: one Rayleigh-Ritz on the initial guess,
 * then repeat { filter; Rayleigh-Ritz; residual test on the n_wanted lowest pairs }.
 *  X            device [m][N]: in the initial guess, out B-orthonormal Ritz vectors.
 *  evals_out    HOST [N]; resnorm_out HOST [N]; iters_out HOST (outer iterations done).
 *  history_out  HOST [max_iter] or NULL: max wanted residual after each iteration.
 * Returns OK when max_{j<n_wanted} r_j < tol, ENOTCONVERGED otherwise. */
rchfsi_status rchfsi_solve(rchfsi_handle h, int32_t method, double *X, int32_t n_wanted,
                           int32_t degree, double lam_min, double lam_T, double lam_max,
                           double tol, int32_t max_iter, double *evals_out,
                           double *resnorm_out, int32_t *iters_out, double *history_out);

/* Estimates of the upper spectral bound lam_max the filter is parameterised by ("parameterised by
 * estimates lam_min, lam_max, lam_T").  The recurrence applies D^-1 A (eq. (7) at PAPER.md:170, Algorithm 3 at 263),
 * so lam_max must bound lam(D^-1 A); it should also bound lam(B^-1 A).  All computed on the device, FP64:
 *   lanczos_*        k-step Lanczos on D^-1/2 A D^-1/2 from a Gaussian start vector drawn from `seed` by the
 *                    counter-based generator of the noise hook: extreme Ritz values theta_min / theta_max (inside the
 *                    spectrum) and lanczos_max = theta_max + beta_k |s_k| (Ritz value + its residual norm);
 *   gershgorin_max   ||D^-1 A||_inf = max_i d_i sum_j |a_ij|: rigorous for lam(D^-1 A), usually loose;
 *   fe_cellwise_max  A and B FE operators on one mesh: max_c lam_max(A_c, B_c) >= lam_max(A, B) over every
 *                    fe_cell_stride-th cell (each cell pencil by cuSOLVER); rigorous for stride 1, NaN when it does
 *                    not apply or fe_cell_stride == 0;
 *   lam_max          recommended value: lanczos_max + 1 %, capped by gershgorin_max, raised to fe_cellwise_max
 *                    (+ 2 % when only a sample of the cells was examined).
 * Synchronises the stream.  Errors: EINVAL (steps outside [2, 512]), ECUDA, ENOMEM, EBREAKDOWN. */
typedef struct {
  double lam_max;
  double lanczos_max;
  double lanczos_theta_max;
  double lanczos_theta_min;
  double gershgorin_max;
  double fe_cellwise_max;
  int32_t lanczos_steps;      /* steps actually taken (fewer on an invariant subspace) */
} rchfsi_bounds;
rchfsi_status rchfsi_estimate_bounds(rchfsi_handle h, int32_t lanczos_steps, int32_t fe_cell_stride, uint64_t seed,
                                     rchfsi_bounds *out);

/* Exact FP64 operator apply, exposed for tests and residual certification:
 * which = 0: out = A V, which = 1: out = B V (B = I copies).  V, out device [m][N]. */
rchfsi_status rchfsi_apply(rchfsi_handle h, int32_t which, const double *V, double *out);

/* Instrumentation: number of kernels this handle has launched since creation, and the
 * CUDA-event time (ms) of the recurrence-step launches of the last rchfsi_filter call
 * (steps_out = number of step launches timed; needs a stream synchronise, which it does). */
int64_t rchfsi_launch_count(rchfsi_handle h);
rchfsi_status rchfsi_last_filter_step_ms(rchfsi_handle h, float *ms_total_out, int32_t *steps_out);

/* ---------------------------------------------------------------------------------------------
 * Allocation-free entry point for callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving
 * loops, harnesses that forbid it).  No handle, no workspace: its scratch is a file-scope __device__ array of
 * RCHFSI_STATIC_SCRATCH_BYTES (148 slots x RCHFSI_STATIC_MAX_N partial sums + a 256-byte header) that every GPU
 * which loads the library holds until the process exits.
 *
 * rchfsi_residual_static: G = AX - BX diag(ritz) (the residual block of Algorithm 3) and
 * r_j = ||A x_j - ritz_j B x_j||_2, FP64, on the CURRENT device.
 *  AX, BX       device [m][N] row-major FP64: A X and B X (pass X itself as BX for a standard problem).
 *  ritz         device [N].
 *  G_out        device [m][N] or NULL, not aliasing an input.  resnorm_out device [N] or NULL; not both NULL.
 *  stream       cudaStream_t (NULL = the default stream).  Asynchronous: one kernel launch, nothing else.
 * N > RCHFSI_STATIC_MAX_N, non-positive sizes or NULL inputs return RCHFSI_EINVAL with outputs untouched
 * (rchfsi_static_last_error, per host thread).  Calls no cudaMalloc / cudaFree / allocating library routine.
 * The partial sums are added in a fixed order, so r_j is bitwise reproducible (the atomicAdd reduction inside
 * rchfsi_rayleigh_ritz is not).  ALL calls on one device share the scratch array, which keeps the last call's
 * contents; the kernel re-arms its ticket counter itself.  Two calls that overlap on the GPU (different streams, or
 * different host threads) race on it: serialise them.  A call whose kernel was aborted leaves the counter undefined.
 *
 * rchfsi_static_setup: takes the array's device address (cudaGetSymbolAddress) and clears the counter for the CURRENT
 * device, once; rchfsi_residual_static does it lazily on first use, but a caller that captures a CUDA graph must call
 * it before the capture starts (the set-up synchronises). */
#define RCHFSI_STATIC_MAX_N 4096
#define RCHFSI_STATIC_SCRATCH_BYTES 4849920
rchfsi_status rchfsi_static_setup(void);
rchfsi_status rchfsi_residual_static(const double *AX, const double *BX, const double *ritz, int64_t m, int32_t N,
                                     double *G_out, double *resnorm_out, void *stream);
const char *rchfsi_static_last_error(void);

/* Library / build identification, e.g. "rchfsi 0.1 sm_100a". */
const char *rchfsi_version(void);

#ifdef __cplusplus
}
#endif
#endif /* RCHFSI_H */
