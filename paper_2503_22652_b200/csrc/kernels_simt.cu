// Plain-ALU (SIMT) kernels: exact FP64 operator applies (parity mode and Rayleigh-Ritz), the
// FP32-FMA operator applies, and the element-wise pieces of Algorithms 2 and 3
// (PAPER.md:78-86, 255-263).  The tensor-core paths live in dense_tc.cu / fe_tc.cu.
#include "common.cuh"

namespace rchfsi {

// ------------------------------------------------------------------------------------ dense
// T[i][j] = sum_k A[i][k] * (dinv[k] * W[k][j]); BM x 64 tile, 16x16 threads, (BM/16) x 4 per thread, the next
// K tile prefetched into registers while the current one is multiplied.
// <64, 16> for large problems; <16, 64> when 64-row tiles would leave most SMs idle (config 1: 16 -> 63 CTAs, and
// 16 instead of 63 exposed global-memory round trips along K).
template <typename TC, int BM, int BK>
__global__ void __launch_bounds__(256) dense_apply_kernel(const double *__restrict__ A, int64_t lda,
                                                          const double *__restrict__ dinv,
                                                          const TC *__restrict__ W, TC *__restrict__ T,
                                                          int64_t m, int32_t N, int64_t ldw, int64_t ldt) {
  constexpr int BN = 64, RPT = BM / 16;
  constexpr int NA = BM * BK / 256, NW = BK * BN / 256;
  __shared__ TC As[BK][BM + 4];
  __shared__ TC Ws[BK][BN + 4];
  const int tid = threadIdx.x;
  const int tx = tid & 15, ty = tid >> 4;
  const int64_t i0 = (int64_t)blockIdx.y * BM;
  const int j0 = blockIdx.x * BN;
  TC acc[RPT][4];
#pragma unroll
  for (int r = 0; r < RPT; ++r)
#pragma unroll
    for (int c = 0; c < 4; ++c) acc[r][c] = TC(0);
  TC pa[NA], pw[NW];
  auto fetch = [&](int64_t k0) {
    // A tile: BM rows x BK k, k fastest across threads
#pragma unroll
    for (int l = 0; l < NA; ++l) {
      const int e = tid + l * 256;
      const int r = e / BK, kk = e % BK;
      const int64_t i = i0 + r, k = k0 + kk;
      pa[l] = (i < m && k < m) ? (TC)A[i * lda + k] : TC(0);
    }
    // W tile: BK k x 64 columns, scaled by dinv[k]
#pragma unroll
    for (int l = 0; l < NW; ++l) {
      const int e = tid + l * 256;
      const int kk = e >> 6, c = e & 63;
      const int64_t k = k0 + kk;
      const int jc = j0 + c;
      TC v = TC(0);
      if (k < m && jc < N) {
        v = W[k * ldw + jc];
        if (dinv) v = (TC)dinv[k] * v;
      }
      pw[l] = v;
    }
  };
  fetch(0);
  for (int64_t k0 = 0; k0 < m; k0 += BK) {
#pragma unroll
    for (int l = 0; l < NA; ++l) {
      const int e = tid + l * 256;
      As[e % BK][e / BK] = pa[l];
    }
#pragma unroll
    for (int l = 0; l < NW; ++l) {
      const int e = tid + l * 256;
      Ws[e >> 6][e & 63] = pw[l];
    }
    __syncthreads();
    if (k0 + BK < m) fetch(k0 + BK);
#pragma unroll
    for (int kk = 0; kk < BK; ++kk) {
      TC a[RPT], w[4];
#pragma unroll
      for (int r = 0; r < RPT; ++r) a[r] = As[kk][ty * RPT + r];
#pragma unroll
      for (int c = 0; c < 4; ++c) w[c] = Ws[kk][tx * 4 + c];
#pragma unroll
      for (int r = 0; r < RPT; ++r)
#pragma unroll
        for (int c = 0; c < 4; ++c) acc[r][c] += a[r] * w[c];
    }
    __syncthreads();
  }
#pragma unroll
  for (int r = 0; r < RPT; ++r) {
    int64_t i = i0 + ty * RPT + r;
    if (i >= m) continue;
#pragma unroll
    for (int c = 0; c < 4; ++c) {
      int jj = j0 + tx * 4 + c;
      if (jj < N) T[i * ldt + jj] = acc[r][c];
    }
  }
}

// -------------------------------------------------------------------------------------- CSR
// One thread per (row, VEC consecutive columns): T_i = sum_t vals_t dinv[col_t] W[col_t].
template <typename TC, int VEC>
__global__ void __launch_bounds__(256) csr_apply_kernel(const int64_t *__restrict__ rowptr,
                                                        const int32_t *__restrict__ colind,
                                                        const double *__restrict__ vals,
                                                        const double *__restrict__ dinv,
                                                        const TC *__restrict__ W, TC *__restrict__ T,
                                                        int64_t m, int32_t N, int64_t ldw, int64_t ldt) {
  const int nvec = N / VEC;
  const int64_t total = m * nvec;
  for (int64_t idx = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; idx < total;
       idx += (int64_t)gridDim.x * blockDim.x) {
    const int64_t row = idx / nvec;
    const int v = (int)(idx - row * nvec);
    TC acc[VEC];
#pragma unroll
    for (int q = 0; q < VEC; ++q) acc[q] = TC(0);
    const int64_t t1 = rowptr[row + 1];
    for (int64_t t = rowptr[row]; t < t1; ++t) {
      const int32_t col = colind[t];
      double a = vals[t];
      if (dinv) a *= dinv[col];
      const TC av = (TC)a;
      const TC *w = W + (int64_t)col * ldw + (int64_t)v * VEC;
#pragma unroll
      for (int q = 0; q < VEC; ++q) acc[q] += av * w[q];
    }
    TC *o = T + row * ldt + (int64_t)v * VEC;
#pragma unroll
    for (int q = 0; q < VEC; ++q) o[q] = acc[q];
  }
}

// --------------------------------------------------------------------------------------- FE
// One CTA per (cell, tile of CT columns): gather the n_loc node rows into shared memory,
// T_c[a] = sum_b A_c[b][a] W_c[b] (symmetric cell matrix read coalesced), scatter-add with
// atomics into the zeroed T.
template <typename TC, typename TM, int CT>
__global__ void fe_apply_kernel(const TM *__restrict__ cell_mats, int64_t cell_stride,
                                const int32_t *__restrict__ conn, int32_t n_loc,
                                const double *__restrict__ dinv, const TC *__restrict__ W,
                                TC *__restrict__ T, int32_t N, int64_t ldw, int64_t ldt) {
  extern __shared__ __align__(16) unsigned char fe_smem[];
  TC *Ws = reinterpret_cast<TC *>(fe_smem);              // [n_loc][CT]
  const int64_t cell = blockIdx.y;
  const int j0 = blockIdx.x * CT;
  const int32_t *cn = conn + cell * n_loc;
  for (int e = threadIdx.x; e < n_loc * CT; e += blockDim.x) {
    int b = e / CT, c = e - b * CT;
    int j = j0 + c;
    int64_t row = cn[b];
    TC v = TC(0);
    if (j < N) {
      v = W[row * ldw + j];
      if (dinv) v = (TC)dinv[row] * v;
    }
    Ws[e] = v;
  }
  __syncthreads();
  const TM *Ac = cell_mats + cell * cell_stride;
  for (int a = threadIdx.x; a < n_loc; a += blockDim.x) {
    TC acc[CT];
#pragma unroll
    for (int c = 0; c < CT; ++c) acc[c] = TC(0);
    for (int b = 0; b < n_loc; ++b) {
      const TC av = (TC)Ac[(int64_t)b * n_loc + a];
      const TC *w = Ws + b * CT;
#pragma unroll
      for (int c = 0; c < CT; ++c) acc[c] += av * w[c];
    }
    TC *o = T + (int64_t)cn[a] * ldt + j0;
#pragma unroll
    for (int c = 0; c < CT; ++c)
      if (j0 + c < N) atomicAdd(o + c, acc[c]);
  }
}

template <typename TC>
rchfsi_status op_apply_simt(rchfsi_ctx *h, const rchfsi_operator &op, const double *dinv_in,
                            const TC *W, TC *T, int32_t N, int64_t ldw, int64_t ldt) {
  // N columns of a block whose rows are ldw (input) / ldt (output) elements apart: a column window of a
  // wider block is W + first_column with ldw = the block's width (0 = contiguous, ld = N)
  cudaStream_t st = h->stream;
  const int64_t m = op.m;
  if (ldw == 0) ldw = N;
  if (ldt == 0) ldt = N;
  if (op.kind == RCHFSI_OP_DENSE) {
    if (cdiv(N, 64) * cdiv(m, 64) >= 148) {
      dim3 grid((unsigned)cdiv(N, 64), (unsigned)cdiv(m, 64));
      dense_apply_kernel<TC, 64, 16><<<grid, 256, 0, st>>>(op.dense, op.lda, dinv_in, W, T, m, N, ldw, ldt);
    } else {
      dim3 grid((unsigned)cdiv(N, 64), (unsigned)cdiv(m, 16));
      dense_apply_kernel<TC, 16, 64><<<grid, 256, 0, st>>>(op.dense, op.lda, dinv_in, W, T, m, N, ldw, ldt);
    }
    LAUNCH_CHECK(h);
  } else if (op.kind == RCHFSI_OP_CSR) {
    constexpr int V = (sizeof(TC) == 8) ? 2 : 4;
    if (N % V == 0 && ldw % V == 0 && ldt % V == 0 && (reinterpret_cast<uintptr_t>(W) & 15u) == 0 &&
        (reinterpret_cast<uintptr_t>(T) & 15u) == 0) {
      int64_t total = m * (N / V);
      unsigned grid = (unsigned)std::min<int64_t>(cdiv(total, 256), 148 * 64);
      csr_apply_kernel<TC, V><<<grid, 256, 0, st>>>(op.rowptr, op.colind, op.vals, dinv_in, W, T, m, N, ldw, ldt);
    } else {
      int64_t total = m * N;
      unsigned grid = (unsigned)std::min<int64_t>(cdiv(total, 256), 148 * 64);
      csr_apply_kernel<TC, 1><<<grid, 256, 0, st>>>(op.rowptr, op.colind, op.vals, dinv_in, W, T, m, N, ldw, ldt);
    }
    LAUNCH_CHECK(h);
  } else if (op.kind == RCHFSI_OP_FE) {
    // 48 (FP64) / 96 (FP32) columns per CTA: the cell matrix (0.9 MB) is re-read once per column tile, so wide
    // tiles turn this kernel from L2-bound into FMA-bound (3.5x faster than 12-column tiles at config 4)
    constexpr int CT = (sizeof(TC) == 8) ? 48 : 96;
    if (ldt == N)
      RCHFSI_CUDA_CHECK(h, cudaMemsetAsync(T, 0, sizeof(TC) * (size_t)m * N, st));
    else
      RCHFSI_CUDA_CHECK(h, cudaMemset2DAsync(T, sizeof(TC) * (size_t)ldt, 0, sizeof(TC) * (size_t)N, (size_t)m, st));
    dim3 grid((unsigned)cdiv(N, CT), (unsigned)op.n_cells);
    int threads = (int)std::min<int64_t>(1024, cdiv(op.n_loc, 32) * 32);
    size_t smem = sizeof(TC) * (size_t)op.n_loc * CT;
    int64_t stride = op.cell_shared ? 0 : (int64_t)op.n_loc * op.n_loc;
    if (op.cell_mats) {
      auto kern = fe_apply_kernel<TC, double, CT>;
      RCHFSI_CUDA_CHECK(h, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
      kern<<<grid, threads, smem, st>>>(op.cell_mats, stride, op.conn, op.n_loc, dinv_in, W, T, N, ldw, ldt);
    } else {
      auto kern = fe_apply_kernel<TC, float, CT>;
      RCHFSI_CUDA_CHECK(h, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
      kern<<<grid, threads, smem, st>>>(op.cell_mats_f32, stride, op.conn, op.n_loc, dinv_in, W, T, N, ldw, ldt);
    }
    LAUNCH_CHECK(h);
  } else {
    h->err = "unknown operator kind";
    return RCHFSI_EINVAL;
  }
  return RCHFSI_OK;
}
template rchfsi_status op_apply_simt<double>(rchfsi_ctx *, const rchfsi_operator &, const double *,
                                             const double *, double *, int32_t, int64_t, int64_t);
template rchfsi_status op_apply_simt<float>(rchfsi_ctx *, const rchfsi_operator &, const double *,
                                            const float *, float *, int32_t, int64_t, int64_t);

}  // namespace rchfsi
