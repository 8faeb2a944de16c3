// Rayleigh-Ritz on a non-orthogonal basis, FP64 throughout.
// Off the hot path: the Gram and rotation products are plain library
// GEMMs (cuBLAS dgemm) and the N x N generalized eigenproblem is cuSOLVER dsygvd; the operator
// applies are this library's FP64 kernels.
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

static rchfsi_status ensure_rr_workspace(rchfsi_ctx *h) {
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
  if (!h->rr1) RCHFSI_TRY(dev_alloc(h, (void **)&h->rr1, blk));
  if (!h->rr3) RCHFSI_TRY(dev_alloc(h, (void **)&h->rr3, blk));
  if (h->B.present && !h->rr2) RCHFSI_TRY(dev_alloc(h, (void **)&h->rr2, blk));
  if (!h->Ha) RCHFSI_TRY(dev_alloc(h, (void **)&h->Ha, nn));
  if (!h->Hb) RCHFSI_TRY(dev_alloc(h, (void **)&h->Hb, nn));
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

// Row-major [m][N] blocks are column-major N x m matrices with leading dimension N.
// Gram: H = U^T V  (N x N).  In the column-major view Uc (N x m): Uc * Vc^T has entry
// (i,j) = sum_r U[r][i] V[r][j], stored column-major = H^T row-major; H is symmetrised after.
static rchfsi_status gram(rchfsi_ctx *h, const double *U, const double *V, double *H) {
  const double one = 1.0, zero = 0.0;
  CUBLAS_CHECK(h, cublasDgemm(h->cublas, CUBLAS_OP_N, CUBLAS_OP_T, h->N, h->N, (int)h->m, &one, U, h->N, V,
                              h->N, &zero, H, h->N));
  h->launches++;
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
  if (h->opt.normalize_columns_before_rr) {   // reading S6
    RCHFSI_TRY(column_sumsq(h, RCHFSI_FP64, Y, m, N, h->colnorm));
    RCHFSI_TRY(scale_columns_inv_norm(h, Y, m, N, h->colnorm));
  }
  double *AY = h->rr1;
  RCHFSI_TRY(op_apply_simt<double>(h, h->A.d, nullptr, Y, AY, N));
  const double *BY = Y;
  if (h->B.present) {
    RCHFSI_TRY(op_apply_simt<double>(h, h->B.d, nullptr, Y, h->rr2, N));
    BY = h->rr2;
  }
  RCHFSI_TRY(gram(h, Y, AY, h->Ha));
  RCHFSI_TRY(gram(h, Y, BY, h->Hb));
  RCHFSI_TRY(symmetrize(h, h->Ha, N));
  RCHFSI_TRY(symmetrize(h, h->Hb, N));
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
  const double *E = h->Ha;   // eigenvectors overwrite H_a, column-major
  double *T3 = h->rr3;
  // X = Y E
  RCHFSI_TRY(rotate(h, Y, E, T3));
  RCHFSI_CUDA_CHECK(h, cudaMemcpyAsync(Y, T3, blk, cudaMemcpyDeviceToDevice, st));
  const bool need_res = (G_out != nullptr) || (res_out != nullptr);
  if (need_res) {
    // AX = (AY) E -> T3 ; BX = (BY) E -> rr1 (AY is dead by then) or X itself when B = I
    RCHFSI_TRY(rotate(h, AY, E, T3));
    const double *BX = Y;
    if (h->B.present) {
      RCHFSI_TRY(rotate(h, h->rr2, E, h->rr1));
      BX = h->rr1;
    }
    RCHFSI_TRY(residual_block(h, T3, BX, h->ritz_dev, G_out, res_out, m, N));
  }
  if (ritz_out && ritz_out != h->ritz_dev)
    RCHFSI_CUDA_CHECK(h, cudaMemcpyAsync(ritz_out, h->ritz_dev, sizeof(double) * N, cudaMemcpyDeviceToDevice, st));
  return RCHFSI_OK;
}

}  // namespace rchfsi
