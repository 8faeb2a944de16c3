// rchfsi_estimate_bounds: estimates of the upper spectral bound the Chebyshev filter is parameterised by
// ("parameterised by estimates lam_min, lam_max, lam_T").  The recurrence applies
// D^-1 A (eq. (7), Alg. 3), so lam_max must bound lam(D^-1 A); for the convergence theory it should
// also bound lam(B^-1 A) (reading S7).  Three estimators, all on the device:
//   * k-step Lanczos (no reorthogonalisation) on S = D^-1/2 A D^-1/2 from a counter-based Gaussian start vector:
//     theta_max + beta_k |s_k| (Ritz value + its residual norm), the usual safeguarded estimate;
//   * ||D^-1 A||_inf = max_i d_i sum_j |a_ij| (Gershgorin): rigorous for lam(D^-1 A), loose;
//   * FE operators A and B on the same mesh: max_c lam_max(A_c, B_c) >= lam_max(A, B) (mediant inequality) over every
//     fe_cell_stride-th cell, each cell pencil by cuSOLVER dsygvd (rigorous when the stride is 1).
// Off the hot path: runs once per operator.
#include <algorithm>
#include <cmath>
#include <cstring>
#include <vector>
#include "common.cuh"
#include "rng.cuh"

namespace rchfsi {
namespace {

__global__ void gauss_fill_kernel(double *v, int64_t m, uint64_t base) {
  for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < m; i += (int64_t)gridDim.x * blockDim.x)
    v[i] = counter_gauss(base, (uint64_t)i);
}
// out = sqrt(dinv) .* in  (dinv == NULL: copy)
__global__ void scale_sqrt_kernel(double *out, const double *in, const double *dinv, int64_t m) {
  for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < m; i += (int64_t)gridDim.x * blockDim.x)
    out[i] = dinv ? sqrt(dinv[i]) * in[i] : in[i];
}
// w = sqrt(dinv) .* t - beta * v_prev ; dot[0] += w . v
__global__ void lanczos_a_kernel(double *w, const double *t, const double *dinv, const double *v_prev, double beta,
                                 const double *v, int64_t m, double *dot) {
  double acc = 0.0;
  for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < m; i += (int64_t)gridDim.x * blockDim.x) {
    const double x = (dinv ? sqrt(dinv[i]) * t[i] : t[i]) - beta * v_prev[i];
    w[i] = x;
    acc += x * v[i];
  }
  for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
  if ((threadIdx.x & 31) == 0) atomicAdd(dot, acc);
}
// w -= alpha v ; dot[1] += w . w
__global__ void lanczos_b_kernel(double *w, const double *v, double alpha, int64_t m, double *dot) {
  double acc = 0.0;
  for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < m; i += (int64_t)gridDim.x * blockDim.x) {
    const double x = w[i] - alpha * v[i];
    w[i] = x;
    acc += x * x;
  }
  for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
  if ((threadIdx.x & 31) == 0) atomicAdd(dot + 1, acc);
}
// v_prev = v ; v = w * s
__global__ void lanczos_c_kernel(double *v_prev, double *v, const double *w, double s, int64_t m) {
  for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < m; i += (int64_t)gridDim.x * blockDim.x) {
    v_prev[i] = v[i];
    v[i] = w[i] * s;
  }
}
__global__ void sumsq_kernel(const double *v, int64_t m, double *out) {
  double acc = 0.0;
  for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < m; i += (int64_t)gridDim.x * blockDim.x) acc += v[i] * v[i];
  for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
  if ((threadIdx.x & 31) == 0) atomicAdd(out, acc);
}

// absolute row sums r_i = sum_j |a_ij| (FE: assembled, r[conn_c[a]] += sum_b |A_c[a][b]|)
__global__ void abs_rowsum_dense_kernel(const double *A, int64_t lda, int64_t m, double *r) {
  const int64_t i = blockIdx.x;
  double acc = 0.0;
  for (int64_t j = threadIdx.x; j < m; j += blockDim.x) acc += fabs(A[i * lda + j]);
  for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
  if ((threadIdx.x & 31) == 0) atomicAdd(r + i, acc);
}
__global__ void abs_rowsum_csr_kernel(const int64_t *rowptr, const double *vals, int64_t m, double *r) {
  for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < m; i += (int64_t)gridDim.x * blockDim.x) {
    double acc = 0.0;
    for (int64_t t = rowptr[i]; t < rowptr[i + 1]; ++t) acc += fabs(vals[t]);
    r[i] = acc;
  }
}
template <typename TM>
__global__ void abs_rowsum_fe_kernel(const TM *mats, int64_t stride, const int32_t *conn, int32_t n_loc, double *r) {
  const int64_t c = blockIdx.x;
  const TM *Ac = mats + c * stride;
  for (int a = threadIdx.x; a < n_loc; a += blockDim.x) {
    double acc = 0.0;
    for (int b = 0; b < n_loc; ++b) acc += fabs((double)Ac[(int64_t)b * n_loc + a]);   // symmetric: column a = row a, coalesced
    atomicAdd(r + conn[c * n_loc + a], acc);
  }
}
// out[0] = max_i d_i r_i  (one block; non-negative values: integer ordering of the bit patterns)
__global__ void max_scaled_kernel(const double *r, const double *dinv, int64_t m, unsigned long long *out) {
  double best = 0.0;
  for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < m; i += (int64_t)gridDim.x * blockDim.x)
    best = fmax(best, (dinv ? fabs(dinv[i]) : 1.0) * r[i]);
  for (int o = 16; o > 0; o >>= 1) best = fmax(best, __shfl_xor_sync(0xffffffffu, best, o));
  if ((threadIdx.x & 31) == 0) atomicMax(out, (unsigned long long)__double_as_longlong(best));
}
template <typename TM>
__global__ void widen_cell_kernel(const TM *src, double *dst, int64_t n) {
  for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) dst[i] = (double)src[i];
}

// Eigenvalues of the symmetric tridiagonal (alpha_0..k-1, beta_0..k-2) by implicit QL, with the LAST row of the
// eigenvector matrix (z[j] = last component of eigenvector j), which is all the residual bound needs.
bool tridiag_ql(std::vector<double> d, std::vector<double> e, std::vector<double> &theta, std::vector<double> &zlast) {
  const int n = (int)d.size();
  e.resize(n, 0.0);
  std::vector<double> z(n, 0.0);
  z[n - 1] = 1.0;
  for (int l = 0; l < n; ++l) {
    int iter = 0, mm;
    do {
      for (mm = l; mm < n - 1; ++mm) {
        const double dd = std::fabs(d[mm]) + std::fabs(d[mm + 1]);
        if (std::fabs(e[mm]) <= 2.3e-16 * dd) break;
      }
      if (mm != l) {
        if (iter++ == 200) return false;
        double g = (d[l + 1] - d[l]) / (2.0 * e[l]);
        double r = std::hypot(g, 1.0);
        g = d[mm] - d[l] + e[l] / (g + (g >= 0 ? std::fabs(r) : -std::fabs(r)));
        double s = 1.0, c = 1.0, p = 0.0;
        int i;
        for (i = mm - 1; i >= l; --i) {
          double f = s * e[i], b = c * e[i];
          r = std::hypot(f, g);
          e[i + 1] = r;
          if (r == 0.0) {
            d[i + 1] -= p;
            e[mm] = 0.0;
            break;
          }
          s = f / r;
          c = g / r;
          g = d[i + 1] - p;
          r = (d[i] - g) * s + 2.0 * c * b;
          p = s * r;
          d[i + 1] = g + p;
          g = c * r - b;
          f = z[i + 1];                       // rotation applied to the last row of the eigenvector matrix
          z[i + 1] = s * z[i] + c * f;
          z[i] = c * z[i] - s * f;
        }
        if (r == 0.0 && i >= l) continue;
        d[l] -= p;
        e[l] = g;
        e[mm] = 0.0;
      }
    } while (mm != l);
  }
  theta = d;
  zlast = z;
  return true;
}

}  // namespace
}  // namespace rchfsi

using namespace rchfsi;

extern "C" rchfsi_status rchfsi_estimate_bounds(rchfsi_handle h, int32_t lanczos_steps, int32_t fe_cell_stride,
                                                uint64_t seed, rchfsi_bounds *out) {
  if (!h) return RCHFSI_EINVAL;
  if (!out || lanczos_steps < 2 || lanczos_steps > 512 || fe_cell_stride < 0) {
    h->err = "rchfsi_estimate_bounds: need out != NULL, 2 <= lanczos_steps <= 512, fe_cell_stride >= 0";
    return RCHFSI_EINVAL;
  }
  const int64_t m = h->m;
  const rchfsi_operator &A = h->A.d;
  cudaStream_t st = h->stream;
  const unsigned grid = (unsigned)std::min<int64_t>(cdiv(m, 256), 148 * 8);
  const double nan = std::nan("");
  rchfsi_bounds b{nan, nan, nan, nan, nan, nan, 0};

  if (!h->bnd_buf) RCHFSI_TRY(dev_alloc(h, (void **)&h->bnd_buf, sizeof(double) * (5 * (size_t)m + 4)));
  double *buf = h->bnd_buf;   // v_prev, v, w, t, u (each [m]) + 2 dot products + 1 max word
  double *v_prev = buf, *v = buf + m, *w = buf + 2 * m, *t = buf + 3 * m, *u = buf + 4 * m, *dots = buf + 5 * m;

  // ---- Lanczos on S = D^-1/2 A D^-1/2
  {
    const uint64_t base = splitmix64(seed);       // = workloads.noise.counter_gaussian(seed, apply_index = 0, m, 1)
    gauss_fill_kernel<<<grid, 256, 0, st>>>(v, m, base);
    LAUNCH_CHECK(h);
    RCHFSI_CUDA_CHECK(h, cudaMemsetAsync(dots, 0, sizeof(double) * 4, st));
    sumsq_kernel<<<grid, 256, 0, st>>>(v, m, dots);
    LAUNCH_CHECK(h);
    double nrm2 = 0.0;
    RCHFSI_CUDA_CHECK(h, cudaMemcpyAsync(&nrm2, dots, sizeof(double), cudaMemcpyDeviceToHost, st));
    RCHFSI_CUDA_CHECK(h, cudaStreamSynchronize(st));
    RCHFSI_CUDA_CHECK(h, cudaMemsetAsync(v_prev, 0, sizeof(double) * m, st));
    lanczos_c_kernel<<<grid, 256, 0, st>>>(w, v, v, 1.0 / std::sqrt(nrm2), m);      // v <- v / ||v|| (w is scratch)
    LAUNCH_CHECK(h);
    RCHFSI_CUDA_CHECK(h, cudaMemsetAsync(v_prev, 0, sizeof(double) * m, st));
    std::vector<double> alpha, beta;
    double bprev = 0.0;
    for (int j = 0; j < lanczos_steps; ++j) {
      scale_sqrt_kernel<<<grid, 256, 0, st>>>(u, v, h->dinv, m);
      LAUNCH_CHECK(h);
      RCHFSI_TRY(op_apply_simt<double>(h, A, nullptr, u, t, 1, 1, 1));
      RCHFSI_CUDA_CHECK(h, cudaMemsetAsync(dots, 0, sizeof(double) * 2, st));
      lanczos_a_kernel<<<grid, 256, 0, st>>>(w, t, h->dinv, v_prev, bprev, v, m, dots);
      LAUNCH_CHECK(h);
      double a = 0.0;
      RCHFSI_CUDA_CHECK(h, cudaMemcpyAsync(&a, dots, sizeof(double), cudaMemcpyDeviceToHost, st));
      RCHFSI_CUDA_CHECK(h, cudaStreamSynchronize(st));
      lanczos_b_kernel<<<grid, 256, 0, st>>>(w, v, a, m, dots);
      LAUNCH_CHECK(h);
      double b2 = 0.0;
      RCHFSI_CUDA_CHECK(h, cudaMemcpyAsync(&b2, dots + 1, sizeof(double), cudaMemcpyDeviceToHost, st));
      RCHFSI_CUDA_CHECK(h, cudaStreamSynchronize(st));
      const double bj = std::sqrt(b2);
      alpha.push_back(a);
      beta.push_back(bj);
      if (!(bj > 1e-300) || !std::isfinite(bj)) break;     // invariant subspace found (or breakdown)
      lanczos_c_kernel<<<grid, 256, 0, st>>>(v_prev, v, w, 1.0 / bj, m);
      LAUNCH_CHECK(h);
      bprev = bj;
    }
    std::vector<double> theta, zl;
    std::vector<double> off(beta.begin(), beta.end() - 1);
    if (!tridiag_ql(alpha, off, theta, zl)) { h->err = "rchfsi_estimate_bounds: tridiagonal QL did not converge"; return RCHFSI_EBREAKDOWN; }
    int imax = 0, imin = 0;
    for (int i = 1; i < (int)theta.size(); ++i) {
      if (theta[i] > theta[imax]) imax = i;
      if (theta[i] < theta[imin]) imin = i;
    }
    b.lanczos_theta_max = theta[imax];
    b.lanczos_theta_min = theta[imin];
    b.lanczos_max = theta[imax] + beta.back() * std::fabs(zl[imax]);
    b.lanczos_steps = (int32_t)alpha.size();
  }

  // ---- ||D^-1 A||_inf
  {
    double *r = w;
    RCHFSI_CUDA_CHECK(h, cudaMemsetAsync(r, 0, sizeof(double) * m, st));
    if (A.kind == RCHFSI_OP_DENSE) {
      abs_rowsum_dense_kernel<<<(unsigned)m, 128, 0, st>>>(A.dense, A.lda, m, r);
    } else if (A.kind == RCHFSI_OP_CSR) {
      abs_rowsum_csr_kernel<<<grid, 256, 0, st>>>(A.rowptr, A.vals, m, r);
    } else {
      const int64_t stride = A.cell_shared ? 0 : (int64_t)A.n_loc * A.n_loc;
      if (A.cell_mats) abs_rowsum_fe_kernel<double><<<(unsigned)A.n_cells, 128, 0, st>>>(A.cell_mats, stride, A.conn, A.n_loc, r);
      else abs_rowsum_fe_kernel<float><<<(unsigned)A.n_cells, 128, 0, st>>>(A.cell_mats_f32, stride, A.conn, A.n_loc, r);
    }
    LAUNCH_CHECK(h);
    unsigned long long *mx = reinterpret_cast<unsigned long long *>(dots + 2);
    RCHFSI_CUDA_CHECK(h, cudaMemsetAsync(mx, 0, sizeof(unsigned long long), st));
    max_scaled_kernel<<<grid, 256, 0, st>>>(r, h->dinv, m, mx);
    LAUNCH_CHECK(h);
    unsigned long long bits = 0;
    RCHFSI_CUDA_CHECK(h, cudaMemcpyAsync(&bits, mx, sizeof(bits), cudaMemcpyDeviceToHost, st));
    RCHFSI_CUDA_CHECK(h, cudaStreamSynchronize(st));
    double gv;
    static_assert(sizeof(gv) == sizeof(bits), "");
    memcpy(&gv, &bits, sizeof(gv));
    b.gershgorin_max = gv;
  }

  // ---- FE pencil on one mesh: max_c lam_max(A_c, B_c) over every fe_cell_stride-th cell
  const rchfsi_operator &B = h->B.d;
  if (fe_cell_stride > 0 && A.kind == RCHFSI_OP_FE && h->B.present && B.kind == RCHFSI_OP_FE && B.n_loc == A.n_loc &&
      B.n_cells == A.n_cells && !A.cell_shared) {
    const int n = A.n_loc;
    const size_t nn = (size_t)n * n;
    if (!h->cusolver) {
      if (cusolverDnCreate(&h->cusolver) != CUSOLVER_STATUS_SUCCESS || cusolverDnSetStream(h->cusolver, st) != CUSOLVER_STATUS_SUCCESS) {
        h->err = "cusolverDnCreate failed";
        return RCHFSI_ECUDA;
      }
    }
    if (!h->bnd_cell) RCHFSI_TRY(dev_alloc(h, (void **)&h->bnd_cell, sizeof(double) * (2 * nn + n + 2)));
    double *Ac = h->bnd_cell, *Bc = Ac + nn, *ev = Bc + nn, *work = nullptr;
    int *info = reinterpret_cast<int *>(ev + n);
    int lwork = 0;
    if (cusolverDnDsygvd_bufferSize(h->cusolver, CUSOLVER_EIG_TYPE_1, CUSOLVER_EIG_MODE_NOVECTOR, CUBLAS_FILL_MODE_LOWER, n,
                                    Ac, n, Bc, n, ev, &lwork) != CUSOLVER_STATUS_SUCCESS) {
      h->err = "cusolverDnDsygvd_bufferSize failed";
      return RCHFSI_ECUDA;
    }
    if (!h->bnd_work) RCHFSI_TRY(dev_alloc(h, (void **)&h->bnd_work, sizeof(double) * (size_t)std::max(lwork, 1)));
    work = h->bnd_work;
    double best = -INFINITY;
    const unsigned g2 = (unsigned)std::min<int64_t>(cdiv((int64_t)nn, 256), 148 * 4);
    for (int64_t c = 0; c < A.n_cells; c += fe_cell_stride) {
      if (A.cell_mats) widen_cell_kernel<double><<<g2, 256, 0, st>>>(A.cell_mats + c * nn, Ac, (int64_t)nn);
      else widen_cell_kernel<float><<<g2, 256, 0, st>>>(A.cell_mats_f32 + c * nn, Ac, (int64_t)nn);
      const int64_t cb = B.cell_shared ? 0 : c;
      if (B.cell_mats) widen_cell_kernel<double><<<g2, 256, 0, st>>>(B.cell_mats + cb * nn, Bc, (int64_t)nn);
      else widen_cell_kernel<float><<<g2, 256, 0, st>>>(B.cell_mats_f32 + cb * nn, Bc, (int64_t)nn);
      h->launches += 2;
      if (cusolverDnDsygvd(h->cusolver, CUSOLVER_EIG_TYPE_1, CUSOLVER_EIG_MODE_NOVECTOR, CUBLAS_FILL_MODE_LOWER, n, Ac, n, Bc, n,
                           ev, work, lwork, info) != CUSOLVER_STATUS_SUCCESS) {
        h->err = "cusolverDnDsygvd (cell pencil) failed";
        return RCHFSI_ECUDA;
      }
      double top = 0.0;
      int hinfo = 0;
      RCHFSI_CUDA_CHECK(h, cudaMemcpyAsync(&top, ev + n - 1, sizeof(double), cudaMemcpyDeviceToHost, st));
      RCHFSI_CUDA_CHECK(h, cudaMemcpyAsync(&hinfo, info, sizeof(int), cudaMemcpyDeviceToHost, st));
      RCHFSI_CUDA_CHECK(h, cudaStreamSynchronize(st));
      if (hinfo != 0) { h->err = "rchfsi_estimate_bounds: cell mass matrix not positive definite"; return RCHFSI_EBREAKDOWN; }
      best = std::max(best, top);
    }
    b.fe_cellwise_max = best;
  }

  // recommended bound: the Lanczos estimate with a 1 % margin, raised to the cell-wise pencil bound when one exists
  // (it also covers lam(B^-1 A)), never above the rigorous infinity-norm bound unless the pencil bound demands it
  double rec = b.lanczos_max + 0.01 * std::fabs(b.lanczos_max);
  if (std::isfinite(b.gershgorin_max)) rec = std::min(rec, b.gershgorin_max);
  if (std::isfinite(b.fe_cellwise_max)) rec = std::max(rec, b.fe_cellwise_max * (fe_cell_stride > 1 ? 1.02 : 1.0));
  b.lam_max = rec;
  *out = b;
  return RCHFSI_OK;
}
