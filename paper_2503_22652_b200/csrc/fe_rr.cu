// FP64 FE operator apply for the Rayleigh-Ritz (off the hot path):
//   T = sum_c P_c^T A_c P_c W     (PAPER.md:357 Remark 4.1, in FP64 with the exact cell matrices)
// as  gather -> batched library DGEMM -> scatter, one colour of the cell colouring at a time.  Cells of one
// colour share no node, so the scatter is a plain read-modify-write (deterministic, no atomics); the first
// colour that touches a node writes, the later ones add (same first-touch flags as the tensor-core filter).
// The filter's own FP64 mode keeps the hand-written kernel of kernels_simt.cu; this path only serves
// rchfsi_rayleigh_ritz / rchfsi_solve, where the products are plain library GEMMs like the Gram and rotation
// products next to them.  Config 4 (m = 912,673, N = 1200): 48 ms per apply against 158 ms.
#include <algorithm>
#include <cstdlib>
#include "common.cuh"

namespace rchfsi {

namespace {

// One warp per gathered row, lanes along the contiguous columns (16-byte accesses when VEC = 2).
// Wg[bi][b][j] = W[conn[cell(bi)][b]][j]
// (cell stride cs, node stride bs) = (n_loc N, N): one [n_loc][N] block per cell (batched GEMM), or (N, batch N): all
// cells side by side, [n_loc][batch][N] (ONE GEMM when every cell has the same matrix)
template <int VEC>
__global__ void feg_gather_kernel(const double *__restrict__ W, int64_t ldw, const int32_t *__restrict__ conn,
                                  const int32_t *__restrict__ cells, int32_t n_loc, int32_t N, double *__restrict__ Wg,
                                  int32_t rows, int64_t cs, int64_t bs) {
  const int lane = threadIdx.x & 31;
  const int wpb = blockDim.x >> 5;
  for (int32_t r = blockIdx.x * wpb + (threadIdx.x >> 5); r < rows; r += gridDim.x * wpb) {
    const int32_t bi = r / n_loc;
    const int32_t b = r - bi * n_loc;
    const double *src = W + (int64_t)conn[(int64_t)cells[bi] * n_loc + b] * ldw;
    double *dst = Wg + bi * cs + b * bs;
    if constexpr (VEC == 2) {
      for (int j = lane; j < N / 2; j += 32) reinterpret_cast<double2 *>(dst)[j] = reinterpret_cast<const double2 *>(src)[j];
    } else {
      for (int j = lane; j < N; j += 32) dst[j] = src[j];
    }
  }
}

// T[conn[cell(bi)][a]][j] (= | +=) Tc[bi][a][j]
template <int VEC>
__global__ void feg_scatter_kernel(const double *__restrict__ Tc, const int32_t *__restrict__ conn,
                                   const uint8_t *__restrict__ flags, const int32_t *__restrict__ cells, int32_t n_loc,
                                   int32_t N, double *__restrict__ T, int64_t ldt, int32_t rows, int64_t cs, int64_t bs) {
  const int lane = threadIdx.x & 31;
  const int wpb = blockDim.x >> 5;
  for (int32_t r = blockIdx.x * wpb + (threadIdx.x >> 5); r < rows; r += gridDim.x * wpb) {
    const int32_t bi = r / n_loc;
    const int32_t a = r - bi * n_loc;
    const int64_t e = (int64_t)cells[bi] * n_loc + a;
    double *o = T + (int64_t)conn[e] * ldt;
    const double *src = Tc + bi * cs + a * bs;
    const bool first = flags[e] & 1;
    if constexpr (VEC == 2) {
      for (int j = lane; j < N / 2; j += 32) {
        double2 v = reinterpret_cast<const double2 *>(src)[j];
        if (!first) {
          const double2 old = reinterpret_cast<double2 *>(o)[j];
          v.x += old.x;
          v.y += old.y;
        }
        reinterpret_cast<double2 *>(o)[j] = v;
      }
    } else {
      for (int j = lane; j < N; j += 32) o[j] = first ? src[j] : o[j] + src[j];
    }
  }
}

__global__ void feg_convert_kernel(const float *__restrict__ mats, const int32_t *__restrict__ cells, int64_t per,
                                   double *__restrict__ out, int64_t batch, int shared) {
  const int64_t total = batch * per;
  for (int64_t t = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; t < total; t += (int64_t)gridDim.x * blockDim.x) {
    const int64_t bi = t / per;
    out[t] = (double)mats[(shared ? 0 : (cells ? (int64_t)cells[bi] : bi)) * per + (t - bi * per)];
  }
}

// pointer arrays of the batched GEMM: [0] = gathered operand, [1] = cell matrix, [2] = product
__global__ void feg_pointers_kernel(const double **ptrs, int64_t batch, int64_t cap, const double *Wg, double *Tc,
                                    int64_t wstride, const double *mats, int64_t mstride, const int32_t *cells,
                                    const double *conv) {
  const int64_t bi = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (bi >= batch) return;
  ptrs[bi] = Wg + bi * wstride;
  ptrs[cap + bi] = conv ? conv + bi * mstride : mats + (int64_t)cells[bi] * mstride;
  ptrs[2 * cap + bi] = Tc + bi * wstride;
}

}  // namespace

// cells per batched-GEMM call: one colour at most, about 1.5 GB of scratch at most
static int64_t fe_rr_cells_per_batch(const rchfsi_operator &op, int32_t N, int64_t max_color) {
  const int32_t nl = op.n_loc;
  const bool conv = (op.cell_mats == nullptr);
  const size_t per_cell = 2 * sizeof(double) * (size_t)nl * N + (conv ? sizeof(double) * (size_t)nl * nl : 0);
  return std::max<int64_t>(1, std::min<int64_t>(std::min<int64_t>(max_color, (int64_t)(1.5e9 / (double)per_cell)), ((int64_t)1 << 30) / nl));
}
size_t fe_rr_scratch_bytes(const rchfsi_operator &op, int32_t N, int64_t max_color) {
  if (op.kind != RCHFSI_OP_FE) return 0;
  const int64_t cap = fe_rr_cells_per_batch(op, N, max_color);
  const int32_t nl = op.n_loc;
  return 2 * (sizeof(double) * (size_t)cap * nl * N + 256) + (op.cell_mats == nullptr ? sizeof(double) * (size_t)cap * nl * nl + 256 : 0) +
         sizeof(double *) * 3 * (size_t)cap + 256;
}

bool fe_apply_gemm_supported(const rchfsi_ctx *h, const rchfsi_operator &op) {
  if (h->knobs.rr_fe_simt) return false;                               // A/B knob: keep the hand-written kernel
  const rchfsi_operator &A = h->A.d;
  return op.kind == RCHFSI_OP_FE && A.kind == RCHFSI_OP_FE && op.conn == A.conn && op.n_cells == A.n_cells &&
         op.n_loc == A.n_loc && h->cublas != nullptr && (op.cell_mats != nullptr || op.cell_mats_f32 != nullptr);
}

// scratch of the batched-GEMM apply: gathered operand + product (+ FP64 copy of a batch of FP32 cell matrices when
// `conv`), about 1.5 GB; sized once for the widest block the handle can see (N_cap or the chunk width of the memory-light
// Rayleigh-Ritz).  Every buffer has its own guard: a call that ran out of workspace is repeated after the caller added a
// segment (rchfsi_add_workspace) and must not allocate again what it already has.
static rchfsi_status feg_ensure(rchfsi_ctx *h, const rchfsi_operator &op, int32_t N, bool conv, int64_t *cap_out) {
  const FeColoring &col = h->coloring;
  const int32_t nl = op.n_loc;
  int64_t max_color = 0;
  for (int k = 0; k < col.n_colors; ++k) max_color = std::max(max_color, col.color_begin[k + 1] - col.color_begin[k]);
  const int32_t Nw = std::max<int32_t>(N, h->feg_N);
  const int64_t cap = fe_rr_cells_per_batch(op, Nw, max_color);
  const size_t need_w = sizeof(double) * (size_t)cap * nl * Nw;
  h->feg_N = Nw;
  if (h->feg_w_bytes < need_w) {
    if (h->feg_W_bytes < need_w) { RCHFSI_TRY(dev_alloc(h, (void **)&h->feg_W, need_w)); h->feg_W_bytes = need_w; }
    if (h->feg_T_bytes < need_w) { RCHFSI_TRY(dev_alloc(h, (void **)&h->feg_T, need_w)); h->feg_T_bytes = need_w; }
    h->feg_w_bytes = need_w;
  }
  if (conv && h->feg_a_cells < cap) {
    RCHFSI_TRY(dev_alloc(h, (void **)&h->feg_A, sizeof(double) * (size_t)cap * nl * nl));
    h->feg_a_cells = cap;
  }
  if (h->feg_ptr_cap < cap) {
    RCHFSI_TRY(dev_alloc(h, (void **)&h->feg_ptrs, sizeof(double *) * 3 * (size_t)cap));
    h->feg_ptr_cap = cap;
  }
  *cap_out = cap;
  return RCHFSI_OK;
}
// the same buffers before the first apply (rchfsi_solve's up-front pass); the per-batch FP64 conversion buffer of an
// FP32-only operator is left to first use: the Rayleigh-Ritz normally lends a full FP64 copy instead
rchfsi_status fe_rr_preallocate(rchfsi_ctx *h, const rchfsi_operator &op, int32_t N) {
  RCHFSI_TRY(fe_ensure_coloring(h));
  int64_t cap = 0;
  return feg_ensure(h, op, N, false, &cap);
}

rchfsi_status fe_apply_gemm(rchfsi_ctx *h, const rchfsi_operator &op, const double *W, double *T, int32_t N,
                            int64_t ldw, int64_t ldt) {
  if (ldw == 0) ldw = N;
  if (ldt == 0) ldt = N;
  RCHFSI_TRY(fe_ensure_coloring(h));
  const FeColoring &col = h->coloring;
  const int32_t nl = op.n_loc;
  // FP64 cell matrices: the caller's, or (FP32-only operators) the copy the Rayleigh-Ritz parked in the filter's dead
  // blocks for the duration of one call (fe_rr_lend_fp64_cells), or else a per-batch conversion
  const double *mats64 = op.cell_mats;
  if (!mats64 && h->feg_A_full && &op == &h->A.d) mats64 = h->feg_A_full;
  const bool conv = (mats64 == nullptr);
  const int64_t mper = op.cell_shared ? 0 : (int64_t)nl * nl;
  int64_t cap = 0;
  RCHFSI_TRY(feg_ensure(h, op, N, conv, &cap));
  const int64_t pcap = h->feg_ptr_cap;
  const bool vec2 = (N % 2 == 0) && (ldw % 2 == 0) && (ldt % 2 == 0) && ((reinterpret_cast<uintptr_t>(W) & 15u) == 0) &&
                    ((reinterpret_cast<uintptr_t>(T) & 15u) == 0);
  const double one = 1.0, zero = 0.0;
  cudaStream_t st = h->stream;
  const unsigned ew = 148 * 16;
  // (Measured and removed: gather of batch k+1 and scatter of batch k-1 on side streams under the GEMM of batch k, two
  // half-size scratch sets -- bit-identical results, no gain: every one of the three kernels fills the GPU by itself,
  // so they serialise anyway.  configs[3]: A Y 55.1 against 56.4 ms.)
  for (int k = 0; k < col.n_colors; ++k)
    for (int64_t b0 = col.color_begin[k]; b0 < col.color_begin[k + 1]; b0 += cap) {
      const int64_t batch = std::min<int64_t>(cap, col.color_begin[k + 1] - b0);
      const int32_t *cells = col.cell_order + b0;
      const int32_t rows = (int32_t)(batch * nl);
      // one matrix for every cell (a mass matrix on a uniform mesh): the cells go side by side and the colour is ONE
      // dgemm with M = batch N instead of `batch` small ones
      const bool one_gemm = op.cell_shared && !h->knobs.rr_fe_batched && batch * (int64_t)N < ((int64_t)1 << 31);
      const int64_t cs = one_gemm ? N : (int64_t)nl * N, bs = one_gemm ? batch * (int64_t)N : N;
      if (vec2) feg_gather_kernel<2><<<ew, 256, 0, st>>>(W, ldw, op.conn, cells, nl, N, h->feg_W, rows, cs, bs);
      else feg_gather_kernel<1><<<ew, 256, 0, st>>>(W, ldw, op.conn, cells, nl, N, h->feg_W, rows, cs, bs);
      LAUNCH_CHECK(h);
      if (conv && (!op.cell_shared || (k == 0 && b0 == col.color_begin[0]))) {
        feg_convert_kernel<<<ew, 256, 0, st>>>(op.cell_mats_f32, cells, (int64_t)nl * nl, h->feg_A, op.cell_shared ? 1 : batch, op.cell_shared ? 1 : 0);
        LAUNCH_CHECK(h);
      }
      if (!one_gemm) {
        feg_pointers_kernel<<<(unsigned)cdiv(batch, 128), 128, 0, st>>>(h->feg_ptrs, batch, pcap, h->feg_W, h->feg_T, (int64_t)nl * N,
                                                                        mats64, mper, cells, conv ? h->feg_A : nullptr);
        LAUNCH_CHECK(h);
      }
      // row-major [nl][N] blocks are column-major N x nl: Tc (N x nl) = Wg (N x nl) * Acm (nl x nl), where the
      // column-major read of the row-major cell matrix is Acm(b, a) = A_c[a][b], so Tc[a][j] = sum_b A_c[a][b] Wg[b][j]
      cublasStatus_t cst;
      if (one_gemm)
        cst = cublasDgemm(h->cublas, CUBLAS_OP_N, CUBLAS_OP_N, (int)(batch * N), nl, nl, &one, h->feg_W, (int)(batch * N),
                          conv ? h->feg_A : mats64, nl, &zero, h->feg_T, (int)(batch * N));
      else
        cst = cublasDgemmBatched(h->cublas, CUBLAS_OP_N, CUBLAS_OP_N, N, nl, nl, &one, h->feg_ptrs, N, h->feg_ptrs + pcap, nl,
                                 &zero, (double **)(h->feg_ptrs + 2 * pcap), N, (int)batch);
      if (cst != CUBLAS_STATUS_SUCCESS) {
        h->err = "cublasDgemm(Batched) (FE apply): status " + std::to_string((int)cst);
        return RCHFSI_ECUDA;
      }
      h->launches++;
      if (vec2) feg_scatter_kernel<2><<<ew, 256, 0, st>>>(h->feg_T, op.conn, col.flags, cells, nl, N, T, ldt, rows, cs, bs);
      else feg_scatter_kernel<1><<<ew, 256, 0, st>>>(h->feg_T, op.conn, col.flags, cells, nl, N, T, ldt, rows, cs, bs);
      LAUNCH_CHECK(h);
    }
  return RCHFSI_OK;
}

// FP64 copy of ALL cell matrices of an FP32-only operator A into `buf` (n_cells n_loc^2 doubles, lent by the caller for
// the duration of one Rayleigh-Ritz): every operator apply of that call then skips its per-batch conversion.
size_t fe_rr_fp64_cells_bytes(const rchfsi_ctx *h) {
  const rchfsi_operator &A = h->A.d;
  if (A.kind != RCHFSI_OP_FE || A.cell_mats || !A.cell_mats_f32 || A.cell_shared) return 0;
  return sizeof(double) * (size_t)A.n_cells * A.n_loc * A.n_loc;
}
rchfsi_status fe_rr_lend_fp64_cells(rchfsi_ctx *h, void *buf) {
  const rchfsi_operator &A = h->A.d;
  feg_convert_kernel<<<148 * 16, 256, 0, h->stream>>>(A.cell_mats_f32, nullptr, (int64_t)A.n_loc * A.n_loc,
                                                     reinterpret_cast<double *>(buf), A.n_cells, 0);
  LAUNCH_CHECK(h);
  h->feg_A_full = reinterpret_cast<const double *>(buf);
  return RCHFSI_OK;
}

}  // namespace rchfsi
