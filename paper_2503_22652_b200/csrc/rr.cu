// Rayleigh-Ritz on a non-orthogonal basis, FP64 throughout.
// Off the hot path: the Gram products and the rotations run on the INT8 tensor pipe
// (rr_i8.cu; cuBLAS dgemm behind RCHFSI_RR_SPLIT=0 / RCHFSI_RR_GRAM_I8=0 and for problems of a few hundred rows), the
// N x N generalized eigenproblem is cuSOLVER dsygvd; the operator applies are this library's FP64 kernels (FE: gather,
// cuBLAS batched dgemm with the exact cell matrices, coloured scatter).
#include <algorithm>
#include <cstdio>
#include <cstdlib>
#include "common.cuh"

namespace rchfsi {

#define CUBLAS_CHECK(h, expr)                                                   \
  do {                                                                          \
    cublasStatus_t _s = (expr);                                                 \
    if (_s != CUBLAS_STATUS_SUCCESS) {                                          \
      (h)->err = std::string(#expr) + ": cuBLAS status " + std::to_string(_s);  \
      return RCHFSI_ECUDA;                                                      \
    }                                                                           \
  } while (0)
#define CUSOLVER_CHECK(h, expr)                                                   \
  do {                                                                            \
    cusolverStatus_t _s = (expr);                                                 \
    if (_s != CUSOLVER_STATUS_SUCCESS) {                                          \
      (h)->err = std::string(#expr) + ": cuSOLVER status " + std::to_string(_s);  \
      return RCHFSI_ECUDA;                                                        \
    }                                                                             \
  } while (0)

// RCHFSI_RR_TIMING=1: synchronise after each phase and print its wall time to stderr (diagnostic only).
struct PhaseTimer {
  rchfsi_ctx *h;
  bool on;
  cudaEvent_t e0 = nullptr, e1 = nullptr;
  explicit PhaseTimer(rchfsi_ctx *hh) : h(hh), on(hh->knobs.rr_timing) {
    if (on) {
      cudaEventCreate(&e0);
      cudaEventCreate(&e1);
      cudaEventRecord(e0, h->stream);
    }
  }
  void lap(const char *what) {
    if (!on) return;
    cudaEventRecord(e1, h->stream);
    cudaEventSynchronize(e1);
    float ms = 0.f;
    cudaEventElapsedTime(&ms, e0, e1);
    fprintf(stderr, "[rchfsi rr] %-28s %10.3f ms\n", what, ms);
    cudaEventRecord(e0, h->stream);
  }
  ~PhaseTimer() {
    if (on) {
      cudaEventDestroy(e0);
      cudaEventDestroy(e1);
    }
  }
};

static rchfsi_status ensure_rr_workspace(rchfsi_ctx *h, bool full_blocks = true) {
  const size_t blk = sizeof(double) * (size_t)h->m * h->N;
  const size_t nn = sizeof(double) * (size_t)h->N * h->N;
  if (!h->cublas) {
    CUBLAS_CHECK(h, cublasCreate(&h->cublas));
    CUBLAS_CHECK(h, cublasSetStream(h->cublas, h->stream));
    CUBLAS_CHECK(h, cublasSetMathMode(h->cublas, CUBLAS_PEDANTIC_MATH));
  }
  if (!h->cusolver) {
    CUSOLVER_CHECK(h, cusolverDnCreate(&h->cusolver));
    CUSOLVER_CHECK(h, cusolverDnSetStream(h->cusolver, h->stream));
  }
  if (full_blocks) {
    if (!h->rr1) RCHFSI_TRY(dev_alloc(h, (void **)&h->rr1, blk));
    if (!h->rr3) RCHFSI_TRY(dev_alloc(h, (void **)&h->rr3, blk));
    if (h->B.present && !h->rr2) RCHFSI_TRY(dev_alloc(h, (void **)&h->rr2, blk));
  }
  if (!h->Ha) {   // only the lower triangles are ever formed: keep the never-read upper parts defined
    RCHFSI_TRY(dev_alloc(h, (void **)&h->Ha, nn));
    RCHFSI_CUDA_CHECK(h, cudaMemsetAsync(h->Ha, 0, nn, h->stream));
  }
  if (!h->Hb) {
    RCHFSI_TRY(dev_alloc(h, (void **)&h->Hb, nn));
    RCHFSI_CUDA_CHECK(h, cudaMemsetAsync(h->Hb, 0, nn, h->stream));
  }
  if (!h->ritz_dev) RCHFSI_TRY(dev_alloc(h, (void **)&h->ritz_dev, sizeof(double) * h->N));
  if (!h->res_dev) RCHFSI_TRY(dev_alloc(h, (void **)&h->res_dev, sizeof(double) * h->N));
  if (!h->colnorm) RCHFSI_TRY(dev_alloc(h, (void **)&h->colnorm, sizeof(double) * 2 * h->N));
  if (!h->sy_info) RCHFSI_TRY(dev_alloc(h, (void **)&h->sy_info, sizeof(int)));
  if (!h->sy_work) {
    int lwork = 0;
    CUSOLVER_CHECK(h, cusolverDnDsygvd_bufferSize(h->cusolver, CUSOLVER_EIG_TYPE_1, CUSOLVER_EIG_MODE_VECTOR,
                                                  CUBLAS_FILL_MODE_LOWER, h->N, h->Ha, h->N, h->Hb, h->N,
                                                  h->ritz_dev, &lwork));
    h->sy_lwork = lwork;
    RCHFSI_TRY(dev_alloc(h, (void **)&h->sy_work, sizeof(double) * (size_t)std::max(lwork, 1)));
  }
  return RCHFSI_OK;
}

// FP64 operator apply of the Rayleigh-Ritz: FE operators go through the batched-GEMM path of fe_rr.cu when it
// applies (3-4x the hand-written FP64 kernel at config 4), everything else through kernels_simt.cu.
static rchfsi_status apply64(rchfsi_ctx *h, const rchfsi_operator &op, const double *W, double *T, int32_t N,
                             int64_t ldw = 0, int64_t ldt = 0) {
  if (fe_apply_gemm_supported(h, op)) return fe_apply_gemm(h, op, W, T, N, ldw, ldt);
  return op_apply_simt<double>(h, op, nullptr, W, T, N, ldw, ldt);
}

// flops of one operator apply on an N-column block (to choose between re-applying and rotating, below)
static double apply_flops(const rchfsi_operator &op, int32_t N) {
  if (op.kind == RCHFSI_OP_DENSE) return 2.0 * (double)op.m * (double)op.m * N;
  if (op.kind == RCHFSI_OP_CSR) return 2.0 * (double)op.nnz * N;
  return 2.0 * (double)op.n_cells * (double)op.n_loc * (double)op.n_loc * N;
}

// Row-major [m][N] blocks are column-major N x m matrices with leading dimension N.
// Gram: H = U^T V  (N x N).  In the column-major view Uc (N x m): Uc * Vc^T has entry
// (i,j) = sum_r U[r][i] V[r][j], stored column-major = H^T row-major; H is symmetrised after.
// Only the lower triangle (column-major i >= j) is formed, in slabs of GRAM_SLAB columns: U^T V is symmetric up
// to rounding for V = Op U with a symmetric operator, and dsygvd reads the lower triangle only.  Slab [c0, c0+w)
// needs the rows i >= c0, so the work is a little over half of the full product.
constexpr int32_t GRAM_SLAB = 256;
static rchfsi_status gram(rchfsi_ctx *h, const double *U, const double *V, double *H) {
  const double one = 1.0, zero = 0.0;
  const int32_t N = h->N;
  for (int32_t c0 = 0; c0 < N; c0 += GRAM_SLAB) {
    const int32_t w = std::min(GRAM_SLAB, N - c0);
    CUBLAS_CHECK(h, cublasDgemm(h->cublas, CUBLAS_OP_N, CUBLAS_OP_T, N - c0, w, (int)h->m, &one, U + c0, N, V + c0, N,
                                &zero, H + (size_t)c0 * N + c0, N));
    h->launches++;
  }
  return RCHFSI_OK;
}
// Out[r][j] = sum_l In[r][l] E[l][j], E column-major N x N (cuSOLVER layout):
// Outc (N x m) = E^T * Inc.
static rchfsi_status rotate(rchfsi_ctx *h, const double *In, const double *E, double *Out) {
  const double one = 1.0, zero = 0.0;
  CUBLAS_CHECK(h, cublasDgemm(h->cublas, CUBLAS_OP_T, CUBLAS_OP_N, h->N, (int)h->m, h->N, &one, E, h->N, In,
                              h->N, &zero, Out, h->N));
  h->launches++;
  return RCHFSI_OK;
}

rchfsi_status rayleigh_ritz_impl(rchfsi_ctx *h, double *Y, double *ritz_out, double *G_out, double *res_out) {
  RCHFSI_TRY(ensure_rr_workspace(h));
  const int64_t m = h->m;
  const int32_t N = h->N;
  const size_t blk = sizeof(double) * (size_t)m * N;
  cudaStream_t st = h->stream;
  PhaseTimer pt(h);
  if (h->opt.normalize_columns_before_rr) {   // reading S6
    RCHFSI_TRY(column_sumsq(h, RCHFSI_FP64, Y, m, N, h->colnorm));
    RCHFSI_TRY(scale_columns_inv_norm(h, Y, m, N, h->colnorm));
  }
  pt.lap("normalise columns");
  double *AY = h->rr1;
  h->feg_N = std::max(h->feg_N, N);     // FE apply scratch sized once for the whole block
  RCHFSI_TRY(apply64(h, h->A.d, Y, AY, N));
  pt.lap("A Y");
  const double *BY = Y;
  if (h->B.present) {
    RCHFSI_TRY(apply64(h, h->B.d, Y, h->rr2, N));
    BY = h->rr2;
  }
  pt.lap("B Y");
  const bool i8ok = rr_i8_scratch_ok(h, blk);
  if (gram_i8_supported(h) && i8ok) {   // rr3 holds the transposed digit planes until the rotation needs it
    RCHFSI_TRY(gram_i8_full(h, Y, AY, h->B.present ? h->rr2 : nullptr, h->Ha, h->Hb, h->rr3, blk));
    pt.lap("Gram x2 (INT8 tensor pipe, lower)");
  } else {
    RCHFSI_TRY(gram(h, Y, AY, h->Ha));
    RCHFSI_TRY(gram(h, Y, BY, h->Hb));
    pt.lap("Gram x2 (dgemm, lower)");
  }
  // H_a E = H_b E Lambda, E^T H_b E = I, ascending (LAPACK dsygv type 1)
  CUSOLVER_CHECK(h, cusolverDnDsygvd(h->cusolver, CUSOLVER_EIG_TYPE_1, CUSOLVER_EIG_MODE_VECTOR,
                                     CUBLAS_FILL_MODE_LOWER, N, h->Ha, N, h->Hb, N, h->ritz_dev, h->sy_work,
                                     h->sy_lwork, h->sy_info));
  h->launches++;
  int info = 0;
  RCHFSI_CUDA_CHECK(h, cudaMemcpyAsync(&info, h->sy_info, sizeof(int), cudaMemcpyDeviceToHost, st));
  RCHFSI_CUDA_CHECK(h, cudaStreamSynchronize(st));
  if (info != 0) {
    h->err = "Rayleigh-Ritz: dsygvd info = " + std::to_string(info) +
             (info > N ? " (Y^T B Y not positive definite)" : " (eigensolver did not converge)");
    return RCHFSI_EBREAKDOWN;
  }
  pt.lap("dsygvd");
  const double *E = h->Ha;   // eigenvectors overwrite H_a, column-major
  double *T3 = h->rr3;
  // X = Y E
  if (rotate_i8_supported(h) && i8ok) {
    RCHFSI_TRY(rotate_i8(h, Y, m, E, Y, T3, blk));            // in place; T3 holds the digit planes
    pt.lap("X = Y E (INT8 tensor pipe)");
  } else {
    RCHFSI_TRY(rotate(h, Y, E, T3));
    RCHFSI_CUDA_CHECK(h, cudaMemcpyAsync(Y, T3, blk, cudaMemcpyDeviceToDevice, st));
    pt.lap("X = Y E (dgemm + copy)");
  }
  const bool need_res = (G_out != nullptr) || (res_out != nullptr);
  if (need_res) {
    // AX and BX: either rotate the products already at hand, AX = (AY) E, BX = (BY) E (2 m N^2 flops each), or
    // apply the operators to the rotated block again -- whichever is less work (sparse / FE operators: re-apply)
    // (rotations on the INT8 pipe run in place -- the products A Y, B Y are dead afterwards -- with the free block as
    // scratch for the digit planes)
    const double *AX = T3, *BX = Y;
    const double rot_flops = 2.0 * (double)m * (double)N * (double)N;
    const bool rot8 = rotate_i8_supported(h) && i8ok;
    if (apply_flops(h->A.d, N) < rot_flops) {
      RCHFSI_TRY(apply64(h, h->A.d, Y, T3, N));
    } else if (rot8) {
      RCHFSI_TRY(rotate_i8(h, AY, m, E, AY, T3, blk));
      AX = AY;
    } else {
      RCHFSI_TRY(rotate(h, AY, E, T3));
    }
    if (h->B.present) {
      double *spare = (AX == AY) ? T3 : h->rr1;        // the block that holds neither A X nor B Y
      if (apply_flops(h->B.d, N) < rot_flops) {
        RCHFSI_TRY(apply64(h, h->B.d, Y, spare, N));
        BX = spare;
      } else if (rot8) {
        RCHFSI_TRY(rotate_i8(h, h->rr2, m, E, h->rr2, spare, blk));
        BX = h->rr2;
      } else {
        RCHFSI_TRY(rotate(h, h->rr2, E, spare));
        BX = spare;
      }
    }
    pt.lap("AX, BX (re-apply or rotate)");
    RCHFSI_TRY(residual_block(h, AX, BX, h->ritz_dev, G_out, res_out, m, N));
    pt.lap("residual block");
  }
  if (ritz_out && ritz_out != h->ritz_dev)
    RCHFSI_CUDA_CHECK(h, cudaMemcpyAsync(ritz_out, h->ritz_dev, sizeof(double) * N, cudaMemcpyDeviceToDevice, st));
  return RCHFSI_OK;
}

// Y <- Y E for a caller-given E (rchfsi_rotate): row panels through the panel buffer of the chunked variant.
static void choose_row_panel(rchfsi_ctx *h) {
  if (h->rr_rp == 0) {
    int64_t rp = (int64_t)(3.0e9 / (8.0 * (double)h->N));
    h->rr_rp = std::max<int64_t>(256, std::min<int64_t>(h->m, rp));
  }
}
rchfsi_status rotate_in_place(rchfsi_ctx *h, double *Y, const double *E) {
  const int64_t m = h->m;
  const int32_t N = h->N;
  if (!h->cublas) {
    CUBLAS_CHECK(h, cublasCreate(&h->cublas));
    CUBLAS_CHECK(h, cublasSetStream(h->cublas, h->stream));
    CUBLAS_CHECK(h, cublasSetMathMode(h->cublas, CUBLAS_PEDANTIC_MATH));
  }
  choose_row_panel(h);
  if (!h->rrp) RCHFSI_TRY(dev_alloc(h, (void **)&h->rrp, sizeof(double) * (size_t)h->rr_rp * N));
  if (rotate_i8_supported(h) && rr_i8_scratch_ok(h, sizeof(double) * (size_t)h->rr_rp * N))
    return rotate_i8(h, Y, m, E, Y, h->rrp, sizeof(double) * (size_t)h->rr_rp * N);
  const double one = 1.0, zero = 0.0;
  for (int64_t r0 = 0; r0 < m; r0 += h->rr_rp) {
    const int64_t rows = std::min<int64_t>(h->rr_rp, m - r0);
    CUBLAS_CHECK(h, cublasDgemm(h->cublas, CUBLAS_OP_T, CUBLAS_OP_N, N, (int)rows, N, &one, E, N, Y + (size_t)r0 * N, N,
                                &zero, h->rrp, N));
    RCHFSI_CUDA_CHECK(h, cudaMemcpyAsync(Y + (size_t)r0 * N, h->rrp, sizeof(double) * (size_t)rows * N,
                                         cudaMemcpyDeviceToDevice, h->stream));
    h->launches++;
  }
  return RCHFSI_OK;
}

// chunk width and row panel of the memory-light variant, decided once per handle
static void choose_chunks(rchfsi_ctx *h) {
  const int64_t m = h->m;
  const int32_t N = h->N;
  if (h->rr_cw == 0) {
    // two [m][cw] FP64 chunks: 6 GB, or up to a third of the free memory when there is more (wider chunks make the
    // batched FE applies and the Gram GEMMs more efficient)
    size_t free_b = 0, total_b = 0;
    double budget = 6.0e9;
    if (cudaMemGetInfo(&free_b, &total_b) == cudaSuccess) budget = std::max(budget, 0.33 * ((double)free_b - 12.0e9));   // 12 GB kept for the low-precision operator copies and scratch still to come
    int64_t cw = (int64_t)(budget / (16.0 * (double)m));
    if (gram_i8_supported(h) && cw >= 64) {
      // the INT8 Gram kernel takes the slabs of A Y_c and B Y_c side by side in 128-column tiles: keep 2 cw close to a
      // multiple of 128
      const int64_t w8 = cw / 8 * 8;
      const double util = 2.0 * (double)w8 / (double)(cdiv(2 * w8, 128) * 128);
      cw = std::min<int64_t>(N, util >= 0.85 ? w8 : cw / 64 * 64);
    } else {
      cw = std::max<int64_t>(8, std::min<int64_t>(N, cw >= 48 ? cw / 48 * 48 : cw / 8 * 8));   // multiples of the FE column tile
    }
    h->rr_cw = (int32_t)cw;
    choose_row_panel(h);
  }
}

// Every buffer a Rayleigh-Ritz of this handle allocates, without computing anything: rchfsi_solve calls it before its
// first Rayleigh-Ritz, so that a workspace that is too small shows as ENOMEM before X has been touched.
rchfsi_status rr_preallocate(rchfsi_ctx *h, bool chunked) {
  RCHFSI_TRY(ensure_rr_workspace(h, !chunked));
  int32_t width = h->N;
  if (chunked) {
    choose_chunks(h);
    if (!h->rrc1) RCHFSI_TRY(dev_alloc(h, (void **)&h->rrc1, sizeof(double) * (size_t)h->m * h->rr_cw));
    if (!h->rrc2) RCHFSI_TRY(dev_alloc(h, (void **)&h->rrc2, sizeof(double) * (size_t)h->m * h->rr_cw));
    width = h->rr_cw;
  }
  h->feg_N = std::max(h->feg_N, width);
  if (fe_apply_gemm_supported(h, h->A.d)) RCHFSI_TRY(fe_rr_preallocate(h, h->A.d, width));
  if (h->B.present && fe_apply_gemm_supported(h, h->B.d)) RCHFSI_TRY(fe_rr_preallocate(h, h->B.d, width));
  return rr_i8_preallocate(h, chunked, chunked ? h->rr_cw : h->N);
}

// ------------------------------------------------------------------------------------------------
// Chunked variant: no full-size temporary.  Extra device memory: two [m][cw] FP64 chunks and one [rp][N]
// FP64 row panel (about 6 GB + 3 GB at config 5 instead of 3 x 58.5 GB).
bool rr_wants_chunked(rchfsi_ctx *h) {
  if (h->knobs.rr_chunked >= 0) return h->knobs.rr_chunked != 0;               // test / tuning knob
  if (h->rr_cw > 0) return true;                                               // decided earlier for this handle
  if (h->rr1) return false;                                                    // full workspace already there
  size_t free_b = 0, total_b = 0;
  if (cudaMemGetInfo(&free_b, &total_b) != cudaSuccess) return false;
  const size_t blk = sizeof(double) * (size_t)h->m * h->N;
  return free_b < (size_t)(3.3 * (double)blk);
}

rchfsi_status rayleigh_ritz_chunked(rchfsi_ctx *h, double *Y, double *ritz_out, void *G_out, int g_prec,
                                    double *res_out) {
  RCHFSI_TRY(ensure_rr_workspace(h, false));
  const int64_t m = h->m;
  const int32_t N = h->N;
  cudaStream_t st = h->stream;
  choose_chunks(h);
  // (each buffer has its own guard: the call may be repeated after the caller added workspace)
  if (!h->rrc1) RCHFSI_TRY(dev_alloc(h, (void **)&h->rrc1, sizeof(double) * (size_t)m * h->rr_cw));
  if (!h->rrc2) RCHFSI_TRY(dev_alloc(h, (void **)&h->rrc2, sizeof(double) * (size_t)m * h->rr_cw));
  const int32_t cw = h->rr_cw;
  h->feg_N = std::max(h->feg_N, cw);    // FE apply scratch sized once for the chunk width
  const double one = 1.0, zero = 0.0;
  PhaseTimer pt(h);
  if (h->opt.normalize_columns_before_rr) {
    RCHFSI_TRY(column_sumsq(h, RCHFSI_FP64, Y, m, N, h->colnorm));
    RCHFSI_TRY(scale_columns_inv_norm(h, Y, m, N, h->colnorm));
  }
  // Gram matrices, one column chunk of A Y / B Y at a time:  H[:, c0:c0+w] = Y^T (Op Y[:, c0:c0+w]).
  // INT8 tensor pipe (rr_i8.cu) when the filter's blocks -- dead between two filters -- can hold the transposed digit
  // planes of Y (rchfsi_solve allocates them before its first Rayleigh-Ritz); cuBLAS dgemm otherwise (a stand-alone
  // rchfsi_rayleigh_ritz on a handle that has never filtered).
  // The filter's blocks R_X, R_Y and the operand shadow are dead between two filters (the filter re-initialises them):
  // this call borrows them for the transposed digit planes and for an FP64 copy of FP32-only cell matrices.
  struct Borrowed {
    rchfsi_ctx *h;
    ~Borrowed() { h->i8g.active = false; h->feg_A_full = nullptr; }
  } borrowed{h};
  std::vector<I8Buf> bufs;
  if (!h->run.active) {
    if (h->RX) bufs.push_back({h->RX, h->RX_bytes});
    if (h->RY) bufs.push_back({h->RY, h->RY_bytes});
    if (h->Wa) bufs.push_back({h->Wa, h->Wa_bytes});
  }
  bool g8 = false;
  if (gram_i8_supported(h) && !bufs.empty()) {
    rchfsi_status gst = RCHFSI_OK;
    g8 = gram_i8_begin(h, Y, bufs, cw, &gst);
    if (gst != RCHFSI_OK) return gst;
  }
  const uint8_t *cells64 = nullptr;
  if (const size_t cb = fe_rr_fp64_cells_bytes(h)) {     // converted once per call instead of once per batch and chunk
    void *pc = nullptr;
    if (carve_buf(bufs, cb, &pc)) {
      RCHFSI_TRY(fe_rr_lend_fp64_cells(h, pc));
      cells64 = reinterpret_cast<const uint8_t *>(pc);
    }
  }
  // scratch of the rotation (digit planes of a row chunk of Y): the largest borrowed block that does not hold the cell
  // copy -- by then the transposed planes of the Gram products are dead; the row panel only when nothing can be borrowed
  void *rot_buf = nullptr;
  size_t rot_bytes = 0;
  if (!h->run.active)
    for (const I8Buf &b : {I8Buf{h->RX, h->RX_bytes}, I8Buf{h->RY, h->RY_bytes}, I8Buf{h->Wa, h->Wa_bytes}}) {
      const uint8_t *p0 = reinterpret_cast<const uint8_t *>(b.ptr);
      if (p0 && !(cells64 && cells64 >= p0 && cells64 < p0 + b.bytes) && b.bytes > rot_bytes) { rot_buf = b.ptr; rot_bytes = b.bytes; }
    }
  bool rot8 = rotate_i8_supported(h);
  if (!(rot8 && rot_buf && rr_i8_scratch_ok(h, rot_bytes))) {
    if (!h->rrp) RCHFSI_TRY(dev_alloc(h, (void **)&h->rrp, sizeof(double) * (size_t)h->rr_rp * N));
    rot_buf = h->rrp;
    rot_bytes = sizeof(double) * (size_t)h->rr_rp * N;
    rot8 = rot8 && rr_i8_scratch_ok(h, rot_bytes);
  }
  for (int32_t c0 = 0; c0 < N; c0 += cw) {
    const int32_t w = std::min(cw, N - c0);
    // lower triangle only (rows i >= c0 of this column slab): dsygvd reads nothing else
    RCHFSI_TRY(apply64(h, h->A.d, Y + c0, h->rrc1, w, N, w));
    if (h->B.present) RCHFSI_TRY(apply64(h, h->B.d, Y + c0, h->rrc2, w, N, w));
    if (g8) {
      RCHFSI_TRY(gram_i8_slab(h, Y, h->rrc1, h->B.present ? h->rrc2 : nullptr, w, w, c0, h->Ha, h->Hb));
      continue;
    }
    const double *BYc = h->B.present ? h->rrc2 : Y + c0;
    const int64_t ldb = h->B.present ? w : N;
    CUBLAS_CHECK(h, cublasDgemm(h->cublas, CUBLAS_OP_N, CUBLAS_OP_T, N - c0, w, (int)m, &one, Y + c0, N, h->rrc1, w, &zero,
                                h->Ha + (size_t)c0 * N + c0, N));
    CUBLAS_CHECK(h, cublasDgemm(h->cublas, CUBLAS_OP_N, CUBLAS_OP_T, N - c0, w, (int)m, &one, Y + c0, N, BYc, (int)ldb, &zero,
                                h->Hb + (size_t)c0 * N + c0, N));
    h->launches += 2;
  }
  pt.lap("chunked: applies + Gram (lower)");
  CUSOLVER_CHECK(h, cusolverDnDsygvd(h->cusolver, CUSOLVER_EIG_TYPE_1, CUSOLVER_EIG_MODE_VECTOR,
                                     CUBLAS_FILL_MODE_LOWER, N, h->Ha, N, h->Hb, N, h->ritz_dev, h->sy_work,
                                     h->sy_lwork, h->sy_info));
  h->launches++;
  int info = 0;
  RCHFSI_CUDA_CHECK(h, cudaMemcpyAsync(&info, h->sy_info, sizeof(int), cudaMemcpyDeviceToHost, st));
  RCHFSI_CUDA_CHECK(h, cudaStreamSynchronize(st));
  if (info != 0) {
    h->err = "Rayleigh-Ritz: dsygvd info = " + std::to_string(info) +
             (info > N ? " (Y^T B Y not positive definite)" : " (eigensolver did not converge)");
    return RCHFSI_EBREAKDOWN;
  }
  pt.lap("chunked: dsygvd");
  const double *E = h->Ha;
  // X = Y E in place, one row panel at a time (row-major rows r0.. are the columns r0.. of the N x m view)
  if (rot8) {
    RCHFSI_TRY(rotate_i8(h, Y, m, E, Y, rot_buf, rot_bytes));
  } else {
    for (int64_t r0 = 0; r0 < m; r0 += h->rr_rp) {
      const int64_t rows = std::min<int64_t>(h->rr_rp, m - r0);
      CUBLAS_CHECK(h, cublasDgemm(h->cublas, CUBLAS_OP_T, CUBLAS_OP_N, N, (int)rows, N, &one, E, N, Y + (size_t)r0 * N, N,
                                  &zero, h->rrp, N));
      RCHFSI_CUDA_CHECK(h, cudaMemcpyAsync(Y + (size_t)r0 * N, h->rrp, sizeof(double) * (size_t)rows * N,
                                           cudaMemcpyDeviceToDevice, st));
      h->launches++;
    }
  }
  pt.lap("chunked: X = Y E (row panels)");
  if (G_out || res_out) {
    // G = A X - B X Lambda recomputed from the rotated block, chunk by chunk (two more operator applies instead
    // of two more full-size temporaries)
    if (res_out) RCHFSI_CUDA_CHECK(h, cudaMemsetAsync(res_out, 0, sizeof(double) * N, st));
    const size_t gel = (g_prec == RCHFSI_FP32) ? sizeof(float) : sizeof(double);
    for (int32_t c0 = 0; c0 < N; c0 += cw) {
      const int32_t w = std::min(cw, N - c0);
      RCHFSI_TRY(apply64(h, h->A.d, Y + c0, h->rrc1, w, N, w));
      const double *BX = Y + c0;
      int64_t ldb = N;
      if (h->B.present) {
        RCHFSI_TRY(apply64(h, h->B.d, Y + c0, h->rrc2, w, N, w));
        BX = h->rrc2;
        ldb = w;
      }
      void *Gc = G_out ? (void *)(reinterpret_cast<uint8_t *>(G_out) + (size_t)c0 * gel) : nullptr;
      RCHFSI_TRY(residual_window(h, h->rrc1, w, BX, ldb, h->ritz_dev + c0, Gc, N, g_prec, res_out ? res_out + c0 : nullptr, m, w));
    }
    if (res_out) RCHFSI_TRY(sqrt_inplace(h, res_out, N));
    pt.lap("chunked: residual applies");
  }
  if (ritz_out && ritz_out != h->ritz_dev)
    RCHFSI_CUDA_CHECK(h, cudaMemcpyAsync(ritz_out, h->ritz_dev, sizeof(double) * N, cudaMemcpyDeviceToDevice, st));
  return RCHFSI_OK;
}

}  // namespace rchfsi
