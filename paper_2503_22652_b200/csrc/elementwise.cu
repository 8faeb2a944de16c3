// Element-wise pieces of Algorithm 2 / Algorithm 3 for the unfused
// paths, plus the small reductions (column norms, residual norms) and the debug noise hook.
// Blocks are [m][N] row-major; storage precision is a run-time code (RCHFSI_FP64 / FP32 /
// BF16) handled by uniform branches: these kernels are HBM-bound.
#include <mutex>
#include "common.cuh"
#include "rng.cuh"

namespace rchfsi {

template <int VEC>
struct Vals {
  double v[VEC];
};

template <int VEC>
__device__ __forceinline__ Vals<VEC> ld_vec(const void *p, int64_t idx, int prec) {
  Vals<VEC> r;
  if (prec == RCHFSI_FP64) {
    const double *q = reinterpret_cast<const double *>(p) + idx;
    if constexpr (VEC == 4) {
      double2 a = *reinterpret_cast<const double2 *>(q);
      double2 b = *reinterpret_cast<const double2 *>(q + 2);
      r.v[0] = a.x; r.v[1] = a.y; r.v[2] = b.x; r.v[3] = b.y;
    } else {
      r.v[0] = q[0];
    }
  } else if (prec == RCHFSI_BF16) {
    const __nv_bfloat16 *q = reinterpret_cast<const __nv_bfloat16 *>(p) + idx;
    if constexpr (VEC == 4) {
      uint2 raw = *reinterpret_cast<const uint2 *>(q);
      __nv_bfloat162 a = *reinterpret_cast<__nv_bfloat162 *>(&raw.x);
      __nv_bfloat162 b = *reinterpret_cast<__nv_bfloat162 *>(&raw.y);
      r.v[0] = __bfloat162float(a.x); r.v[1] = __bfloat162float(a.y);
      r.v[2] = __bfloat162float(b.x); r.v[3] = __bfloat162float(b.y);
    } else {
      r.v[0] = __bfloat162float(q[0]);
    }
  } else {
    const float *q = reinterpret_cast<const float *>(p) + idx;
    if constexpr (VEC == 4) {
      float4 a = *reinterpret_cast<const float4 *>(q);
      r.v[0] = a.x; r.v[1] = a.y; r.v[2] = a.z; r.v[3] = a.w;
    } else {
      r.v[0] = q[0];
    }
  }
  return r;
}

template <int VEC>
__device__ __forceinline__ void st_vec(void *p, int64_t idx, int prec, const Vals<VEC> &r) {
  if (prec == RCHFSI_FP64) {
    double *q = reinterpret_cast<double *>(p) + idx;
    if constexpr (VEC == 4) {
      *reinterpret_cast<double2 *>(q) = make_double2(r.v[0], r.v[1]);
      *reinterpret_cast<double2 *>(q + 2) = make_double2(r.v[2], r.v[3]);
    } else {
      q[0] = r.v[0];
    }
  } else if (prec == RCHFSI_BF16) {
    __nv_bfloat16 *q = reinterpret_cast<__nv_bfloat16 *>(p) + idx;
    if constexpr (VEC == 4) {
      __nv_bfloat162 a = __floats2bfloat162_rn((float)r.v[0], (float)r.v[1]);
      __nv_bfloat162 b = __floats2bfloat162_rn((float)r.v[2], (float)r.v[3]);
      uint2 raw;
      raw.x = *reinterpret_cast<uint32_t *>(&a);
      raw.y = *reinterpret_cast<uint32_t *>(&b);
      *reinterpret_cast<uint2 *>(q) = raw;
    } else {
      q[0] = __float2bfloat16_rn((float)r.v[0]);
    }
  } else {
    float *q = reinterpret_cast<float *>(p) + idx;
    if constexpr (VEC == 4) {
      *reinterpret_cast<float4 *>(q) = make_float4((float)r.v[0], (float)r.v[1], (float)r.v[2], (float)r.v[3]);
    } else {
      q[0] = (float)r.v[0];
    }
  }
}

// R_X <- a T (dinv_out) + b R_Y + c' R_X + a G Lambda_Y   (Alg. 3 loop body, PAPER.md:263;
// without G it is the Alg. 2 loop body)
template <int VEC>
__global__ void __launch_bounds__(256) step_kernel(StepArgs a, int store_prec, int t_prec, int shadow_prec) {
  const int nv = a.N / VEC;
  const int64_t total = a.m * nv;
  for (int64_t t = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; t < total;
       t += (int64_t)gridDim.x * blockDim.x) {
    const int64_t row = t / nv;
    const int j = (int)(t - row * nv) * VEC;
    const int64_t idx = row * a.N + j;
    Vals<VEC> T = ld_vec<VEC>(a.T, idx, t_prec);
    Vals<VEC> ry = ld_vec<VEC>(a.RY, idx, store_prec);
    Vals<VEC> rx = ld_vec<VEC>(a.RX, idx, store_prec);
    const double ds = a.dinv_out ? a.dinv_out[row] : 1.0;
    Vals<VEC> out;
#pragma unroll
    for (int q = 0; q < VEC; ++q) out.v[q] = a.k.a * (ds * T.v[q]) + a.k.b * ry.v[q] + a.k.cp * rx.v[q];
    if (a.G) {
      Vals<VEC> g = ld_vec<VEC>(a.G, idx, store_prec);
#pragma unroll
      for (int q = 0; q < VEC; ++q) out.v[q] += a.k.a * (g.v[q] * a.LY[j + q]);
    }
    st_vec<VEC>(a.RX, idx, store_prec, out);
    if (a.Wnext) st_vec<VEC>(a.Wnext, idx, shadow_prec, out);
  }
}

static inline unsigned ew_grid(int64_t total) {
  return (unsigned)std::max<int64_t>(1, std::min<int64_t>(cdiv(total, 256), 148 * 16));
}

rchfsi_status step_elementwise(rchfsi_ctx *h, int store_prec, int t_prec, int shadow_prec,
                               const StepArgs &a) {
  if (a.N % 4 == 0)
    step_kernel<4><<<ew_grid(a.m * (a.N / 4)), 256, 0, h->stream>>>(a, store_prec, t_prec, shadow_prec);
  else
    step_kernel<1><<<ew_grid(a.m * a.N), 256, 0, h->stream>>>(a, store_prec, t_prec, shadow_prec);
  LAUNCH_CHECK(h);
  return RCHFSI_OK;
}

// mode 0: dst = alpha * src                                   (R_Y = (sigma_1/e) G; G copy)
// mode 1: dst = alpha * (dinv[row] * T - c * src)             (Alg. 2 first step)
// mode 2: X   = dinv[row] * RY + X * LY[j]                    (Alg. 3 last line)
// mode 3: X   = RY                                            (Alg. 2 result)
template <int VEC>
__global__ void __launch_bounds__(256) misc_kernel(int mode, double alpha, double c, const void *T, int t_prec,
                                                   const double *dinv, const double *LY, const void *src,
                                                   void *dst, int dst_prec, void *shadow, int shadow_prec,
                                                   int64_t m, int32_t N, int64_t pm, int src_prec) {
  // pm != 0: the library-owned blocks (R_X / R_Y / G copy / shadows) are stored in PANEL layout
  // [ceil(N/128)][m][128] (see fe_tc.cu); user blocks (X, G) are always row-major [m][N].
  const int nv = N / VEC;
  const int64_t total = m * nv;
  for (int64_t t = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; t < total;
       t += (int64_t)gridDim.x * blockDim.x) {
    const int64_t row = t / nv;
    const int j = (int)(t - row * nv) * VEC;
    const int64_t idx = row * N + j;
    const int64_t lidx = pm ? (((int64_t)(j >> 7) * pm + row) << 7) + (j & 127) : idx;
    Vals<VEC> out;
    if (mode == 0) {
      Vals<VEC> s = ld_vec<VEC>(src, idx, src_prec);
#pragma unroll
      for (int q = 0; q < VEC; ++q) out.v[q] = alpha * s.v[q];
    } else if (mode == 1) {
      Vals<VEC> s = ld_vec<VEC>(src, idx, RCHFSI_FP64);
      Vals<VEC> tt = ld_vec<VEC>(T, idx, t_prec);
      const double ds = dinv ? dinv[row] : 1.0;
#pragma unroll
      for (int q = 0; q < VEC; ++q) out.v[q] = alpha * (ds * tt.v[q] - c * s.v[q]);
    } else if (mode == 2) {
      Vals<VEC> x = ld_vec<VEC>(dst, idx, RCHFSI_FP64);
      Vals<VEC> ry = ld_vec<VEC>(T, lidx, t_prec);
      const double ds = dinv ? dinv[row] : 1.0;
#pragma unroll
      for (int q = 0; q < VEC; ++q) out.v[q] = ds * ry.v[q] + x.v[q] * LY[j + q];
    } else {
      out = ld_vec<VEC>(T, lidx, t_prec);
    }
    st_vec<VEC>(dst, mode == 0 ? lidx : idx, dst_prec, out);
    if (shadow) st_vec<VEC>(shadow, lidx, shadow_prec, out);
  }
}

static rchfsi_status launch_misc(rchfsi_ctx *h, int mode, double alpha, double c, const void *T, int t_prec,
                                 const double *dinv, const double *LY, const void *src, void *dst,
                                 int dst_prec, void *shadow, int shadow_prec, int64_t m, int32_t N, int64_t pm = 0,
                                 int src_prec = RCHFSI_FP64) {
  if (N % 4 == 0)
    misc_kernel<4><<<ew_grid(m * (N / 4)), 256, 0, h->stream>>>(mode, alpha, c, T, t_prec, dinv, LY, src, dst,
                                                                 dst_prec, shadow, shadow_prec, m, N, pm, src_prec);
  else
    misc_kernel<1><<<ew_grid(m * N), 256, 0, h->stream>>>(mode, alpha, c, T, t_prec, dinv, LY, src, dst,
                                                           dst_prec, shadow, shadow_prec, m, N, pm, src_prec);
  LAUNCH_CHECK(h);
  return RCHFSI_OK;
}

rchfsi_status scale_convert(rchfsi_ctx *h, int store_prec, int shadow_prec, double alpha,
                            const void *src, void *dst, void *shadow, int64_t m, int32_t N, int64_t pm,
                            int src_prec) {
  return launch_misc(h, 0, alpha, 0.0, nullptr, 0, nullptr, nullptr, src, dst, store_prec, shadow,
                     shadow_prec, m, N, pm, src_prec);
}
rchfsi_status chfsi_first(rchfsi_ctx *h, int store_prec, int t_prec, int shadow_prec, double alpha,
                          double c, const void *T, const double *dinv, const double *X, void *Y,
                          void *shadow, int64_t m, int32_t N) {
  return launch_misc(h, 1, alpha, c, T, t_prec, dinv, nullptr, X, Y, store_prec, shadow, shadow_prec, m, N);
}
rchfsi_status finish_block(rchfsi_ctx *h, int store_prec, const void *RY, const double *dinv,
                           const double *LY, double *X, int64_t m, int32_t N, int64_t pm) {
  return launch_misc(h, LY ? 2 : 3, 0.0, 0.0, RY, store_prec, dinv, LY, nullptr, X, RCHFSI_FP64, nullptr, 0, m, N, pm);
}

// Lambda_k = C_k(Lambda), eq. (12): one thread per column, k sequential.
__global__ void lambda_table_kernel(const double *__restrict__ ritz, int32_t N, int32_t p, double e,
                                    double c, double sigma1, double *__restrict__ table) {
  int j = blockIdx.x * blockDim.x + threadIdx.x;
  if (j >= N) return;
  const double lam = ritz[j];
  double lx = 1.0, ly = (sigma1 / e) * (lam - c);
  table[j] = lx;
  if (p >= 1) table[(int64_t)N + j] = ly;
  double sigma = sigma1;
  const double gamma = 2.0 / sigma1;
  for (int k = 2; k <= p; ++k) {
    const double sigma2 = 1.0 / (gamma - sigma);
    const double a = 2.0 * sigma2 / e;
    const double ln = a * ly * lam - a * c * ly - sigma * sigma2 * lx;
    lx = ly;
    ly = ln;
    sigma = sigma2;
    table[(int64_t)k * N + j] = ly;
  }
}

rchfsi_status lambda_table(rchfsi_ctx *h, const double *ritz, int32_t N, int32_t p, double e,
                           double c, double sigma1, double *table) {
  lambda_table_kernel<<<(unsigned)cdiv(N, 128), 128, 0, h->stream>>>(ritz, N, p, e, c, sigma1, table);
  LAUNCH_CHECK(h);
  return RCHFSI_OK;
}

// ---------------------------------------------------------------------------- reductions
// sumsq[j] += sum_i V[i][j]^2 : each CTA owns a slab of rows, threads own columns.
__global__ void __launch_bounds__(256) column_sumsq_kernel(const void *V, int prec, int64_t m, int32_t N,
                                                           int64_t rows_per_cta, double *sumsq) {
  const int64_t r0 = blockIdx.x * rows_per_cta;
  const int64_t r1 = min(m, r0 + rows_per_cta);
  for (int j = threadIdx.x; j < N; j += blockDim.x) {
    double s = 0.0;
    for (int64_t i = r0; i < r1; ++i) {
      double v = ld_vec<1>(V, i * N + j, prec).v[0];
      s += v * v;
    }
    atomicAdd(sumsq + j, s);
  }
}

rchfsi_status column_sumsq(rchfsi_ctx *h, int prec, const void *V, int64_t m, int32_t N, double *sumsq) {
  RCHFSI_CUDA_CHECK(h, cudaMemsetAsync(sumsq, 0, sizeof(double) * N, h->stream));
  int64_t ctas = std::min<int64_t>(m, 148 * 8);
  int64_t rows = cdiv(m, ctas);
  ctas = cdiv(m, rows);
  column_sumsq_kernel<<<(unsigned)ctas, 256, 0, h->stream>>>(V, prec, m, N, rows, sumsq);
  LAUNCH_CHECK(h);
  return RCHFSI_OK;
}

__global__ void __launch_bounds__(256) scale_columns_kernel(double *V, int64_t m, int32_t N, const double *sumsq) {
  const int64_t total = m * N;
  for (int64_t t = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; t < total;
       t += (int64_t)gridDim.x * blockDim.x) {
    const int j = (int)(t % N);
    V[t] = V[t] / sqrt(sumsq[j]);
  }
}

rchfsi_status scale_columns_inv_norm(rchfsi_ctx *h, double *V, int64_t m, int32_t N, const double *sumsq) {
  scale_columns_kernel<<<ew_grid(m * N), 256, 0, h->stream>>>(V, m, N, sumsq);
  LAUNCH_CHECK(h);
  return RCHFSI_OK;
}

// G = AX - BX diag(ritz); res2[j] += sum_i G[i][j]^2
__global__ void __launch_bounds__(256) residual_kernel(const double *AX, const double *BX, const double *ritz,
                                                       double *G, double *res2, int64_t m, int32_t N,
                                                       int64_t rows_per_cta) {
  const int64_t r0 = blockIdx.x * rows_per_cta;
  const int64_t r1 = min(m, r0 + rows_per_cta);
  for (int j = threadIdx.x; j < N; j += blockDim.x) {
    const double lam = ritz[j];
    double s = 0.0;
    for (int64_t i = r0; i < r1; ++i) {
      const double g = AX[i * N + j] - BX[i * N + j] * lam;
      if (G) G[i * N + j] = g;
      s += g * g;
    }
    if (res2) atomicAdd(res2 + j, s);
  }
}
// column-window variant for the chunked Rayleigh-Ritz: AX, BX, G have their own row pitches and G may be FP32
__global__ void __launch_bounds__(256) residual_window_kernel(const double *AX, int64_t lda, const double *BX, int64_t ldb,
                                                              const double *ritz, void *G, int64_t ldg, int g_prec,
                                                              double *res2, int64_t m, int32_t w, int64_t rows_per_cta) {
  const int64_t r0 = blockIdx.x * rows_per_cta;
  const int64_t r1 = min(m, r0 + rows_per_cta);
  for (int j = threadIdx.x; j < w; j += blockDim.x) {
    const double lam = ritz[j];
    double s = 0.0;
    for (int64_t i = r0; i < r1; ++i) {
      const double g = AX[i * lda + j] - BX[i * ldb + j] * lam;
      if (G) {
        if (g_prec == RCHFSI_FP32) reinterpret_cast<float *>(G)[i * ldg + j] = (float)g;
        else reinterpret_cast<double *>(G)[i * ldg + j] = g;
      }
      s += g * g;
    }
    if (res2) atomicAdd(res2 + j, s);
  }
}
rchfsi_status residual_window(rchfsi_ctx *h, const double *AX, int64_t lda, const double *BX, int64_t ldb,
                              const double *ritz, void *G, int64_t ldg, int g_prec, double *res2, int64_t m, int32_t w) {
  int64_t ctas = std::min<int64_t>(m, 148 * 8);
  int64_t rows = cdiv(m, ctas);
  ctas = cdiv(m, rows);
  residual_window_kernel<<<(unsigned)ctas, 256, 0, h->stream>>>(AX, lda, BX, ldb, ritz, G, ldg, g_prec, res2, m, w, rows);
  LAUNCH_CHECK(h);
  return RCHFSI_OK;
}
rchfsi_status sqrt_inplace(rchfsi_ctx *h, double *v, int32_t N);
__global__ void sqrt_kernel(double *v, int32_t N) {
  int j = blockIdx.x * blockDim.x + threadIdx.x;
  if (j < N) v[j] = sqrt(v[j]);
}

rchfsi_status residual_block(rchfsi_ctx *h, const double *AX, const double *BX, const double *ritz,
                             double *G, double *res, int64_t m, int32_t N) {
  if (res) RCHFSI_CUDA_CHECK(h, cudaMemsetAsync(res, 0, sizeof(double) * N, h->stream));
  int64_t ctas = std::min<int64_t>(m, 148 * 8);
  int64_t rows = cdiv(m, ctas);
  ctas = cdiv(m, rows);
  residual_kernel<<<(unsigned)ctas, 256, 0, h->stream>>>(AX, BX, ritz, G, res, m, N, rows);
  LAUNCH_CHECK(h);
  if (res) {
    sqrt_kernel<<<(unsigned)cdiv(N, 128), 128, 0, h->stream>>>(res, N);
    LAUNCH_CHECK(h);
  }
  return RCHFSI_OK;
}

rchfsi_status sqrt_inplace(rchfsi_ctx *h, double *v, int32_t N) {
  sqrt_kernel<<<(unsigned)cdiv(N, 128), 128, 0, h->stream>>>(v, N);
  LAUNCH_CHECK(h);
  return RCHFSI_OK;
}

__global__ void symmetrize_kernel(double *H, int32_t N) {
  int i = blockIdx.y * blockDim.y + threadIdx.y;
  int j = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < N && j < i) {
    double s = 0.5 * (H[(int64_t)i * N + j] + H[(int64_t)j * N + i]);
    H[(int64_t)i * N + j] = s;
    H[(int64_t)j * N + i] = s;
  }
}
rchfsi_status symmetrize(rchfsi_ctx *h, double *H, int32_t N) {
  dim3 b(16, 16), g((unsigned)cdiv(N, 16), (unsigned)cdiv(N, 16));
  symmetrize_kernel<<<g, b, 0, h->stream>>>(H, N);
  LAUNCH_CHECK(h);
  return RCHFSI_OK;
}

// ------------------------------------------------------------------------------ noise hook
// Counter-based N(0,1): splitmix64 of (seed, apply index, i*N + j), Box-Muller.  The same map
// is implemented by workloads/noise.py (the random numbers are an INPUT of the inexact
// operator, reading S11).
__global__ void __launch_bounds__(256) noise_norm_kernel(const void *T, int prec, int64_t m, int32_t N,
                                                         int64_t rows_per_cta, uint64_t base, double *tn2,
                                                         double *gn2) {
  const int64_t r0 = blockIdx.x * rows_per_cta;
  const int64_t r1 = min(m, r0 + rows_per_cta);
  for (int j = threadIdx.x; j < N; j += blockDim.x) {
    double st = 0.0, sg = 0.0;
    for (int64_t i = r0; i < r1; ++i) {
      const double v = ld_vec<1>(T, i * N + j, prec).v[0];
      const double g = counter_gauss(base, (uint64_t)(i * N + j));
      st += v * v;
      sg += g * g;
    }
    atomicAdd(tn2 + j, st);
    atomicAdd(gn2 + j, sg);
  }
}
__global__ void __launch_bounds__(256) noise_add_kernel(void *T, int prec, int64_t m, int32_t N, double eps,
                                                        uint64_t base, const double *tn2, const double *gn2) {
  const int64_t total = m * N;
  for (int64_t t = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; t < total;
       t += (int64_t)gridDim.x * blockDim.x) {
    const int j = (int)(t % N);
    Vals<1> v = ld_vec<1>(T, t, prec);
    v.v[0] += eps * sqrt(tn2[j] / gn2[j]) * counter_gauss(base, (uint64_t)t);
    st_vec<1>(T, t, prec, v);
  }
}

rchfsi_status add_column_noise(rchfsi_ctx *h, int t_prec, void *T, int64_t m, int32_t N, double eps,
                               uint64_t seed, uint64_t apply_index, double *scratch2N) {
  const uint64_t base = splitmix64(seed ^ (apply_index * 0xD1B54A32D192ED03ull));
  RCHFSI_CUDA_CHECK(h, cudaMemsetAsync(scratch2N, 0, sizeof(double) * 2 * N, h->stream));
  int64_t ctas = std::min<int64_t>(m, 148 * 8);
  int64_t rows = cdiv(m, ctas);
  ctas = cdiv(m, rows);
  noise_norm_kernel<<<(unsigned)ctas, 256, 0, h->stream>>>(T, t_prec, m, N, rows, base, scratch2N, scratch2N + N);
  LAUNCH_CHECK(h);
  noise_add_kernel<<<ew_grid(m * N), 256, 0, h->stream>>>(T, t_prec, m, N, eps, base, scratch2N, scratch2N + N);
  LAUNCH_CHECK(h);
  return RCHFSI_OK;
}

// ------------------------------------------------------------------- FE symmetry check
template <typename TM>
__global__ void fe_asym_kernel(const TM *mats, int64_t n_mats, int32_t n_loc, double *out) {
  const int64_t per = (int64_t)n_loc * n_loc;
  double worst = 0.0;
  for (int64_t t = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; t < n_mats * per;
       t += (int64_t)gridDim.x * blockDim.x) {
    const int64_t c = t / per;
    const int64_t r = t - c * per;
    const int a = (int)(r / n_loc), b = (int)(r % n_loc);
    if (b < a) {
      const double x = (double)mats[t], y = (double)mats[c * per + (int64_t)b * n_loc + a];
      const double d = fabs(x - y) / fmax(1e-300, fmax(fabs(x), fabs(y)) + 1e-12);
      worst = fmax(worst, d);
    }
  }
  // non-negative doubles order like their bit patterns
  atomicMax(reinterpret_cast<unsigned long long *>(out), (unsigned long long)__double_as_longlong(worst));
}

// result cell of the symmetry check: module-scope device memory (rchfsi_create runs before any workspace exists and
// the library never calls cudaMalloc); creates are serialised on it
__device__ double g_asym_cell;
static std::mutex g_asym_mutex;

rchfsi_status fe_check_symmetric(rchfsi_ctx *h, const rchfsi_operator &op, double *max_asym_host) {
  std::lock_guard<std::mutex> lock(g_asym_mutex);
  double *d = nullptr;
  RCHFSI_CUDA_CHECK(h, cudaGetSymbolAddress((void **)&d, g_asym_cell));
  cudaMemsetAsync(d, 0, sizeof(double), h->stream);
  const int64_t n_mats = op.cell_shared ? 1 : op.n_cells;
  if (op.cell_mats)
    fe_asym_kernel<double><<<148 * 8, 256, 0, h->stream>>>(op.cell_mats, n_mats, op.n_loc, d);
  else
    fe_asym_kernel<float><<<148 * 8, 256, 0, h->stream>>>(op.cell_mats_f32, n_mats, op.n_loc, d);
  h->launches++;
  cudaError_t e = cudaMemcpyAsync(max_asym_host, d, sizeof(double), cudaMemcpyDeviceToHost, h->stream);
  if (e == cudaSuccess) e = cudaStreamSynchronize(h->stream);
  if (e != cudaSuccess) {
    h->err = std::string("fe_check_symmetric: ") + cudaGetErrorString(e);
    return RCHFSI_ECUDA;
  }
  return RCHFSI_OK;
}

}  // namespace rchfsi
