// Fused CSR step: T_i = sum_t a_it W_{col_t} in FP32 on the ALUs with
// 128-bit coalesced loads along the N contiguous columns, and the Alg. 3 update
//   R_X <- a T + b R_Y + c' R_X + a G Lambda_Y
// as the epilogue of the same thread, so every block crosses HBM once per step: R_Y, R_X and G
// are read once, R_X is written once.  The operand W is R_Y itself (converted to FP32 on the
// fly when the recurrence is stored in FP64); D^-1 is folded into the FP32 copy of the values
// (a_it * dinv[col_t]), which is exact algebra for A D^-1 ("A D^-1 R_Y").
#include <cstdlib>
#include <type_traits>
#include "common.cuh"

namespace rchfsi {

namespace {

__global__ void fold_vals_kernel(const double *__restrict__ vals, const int32_t *__restrict__ colind,
                                 const double *__restrict__ dinv, float *__restrict__ out, int64_t nnz) {
  for (int64_t t = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; t < nnz; t += (int64_t)gridDim.x * blockDim.x) {
    double v = vals[t];
    if (dinv) v *= dinv[colind[t]];
    out[t] = (float)v;
  }
}

__device__ __forceinline__ float4 ld4_as_float(const double *p) {
  const double2 a = *reinterpret_cast<const double2 *>(p);
  const double2 b = *reinterpret_cast<const double2 *>(p + 2);
  return make_float4((float)a.x, (float)a.y, (float)b.x, (float)b.y);
}
__device__ __forceinline__ float4 ld4_as_float(const float *p) { return *reinterpret_cast<const float4 *>(p); }

__device__ __forceinline__ void ld4_as_double(const double *p, double (&o)[4]) {
  const double2 a = *reinterpret_cast<const double2 *>(p);
  const double2 b = *reinterpret_cast<const double2 *>(p + 2);
  o[0] = a.x; o[1] = a.y; o[2] = b.x; o[3] = b.y;
}
__device__ __forceinline__ void ld4_as_double(const float *p, double (&o)[4]) {
  const float4 a = *reinterpret_cast<const float4 *>(p);
  o[0] = a.x; o[1] = a.y; o[2] = a.z; o[3] = a.w;
}
// Raw 4-element vectors of the storage type (two 16-byte words for FP64, one for FP32) so the loads of
// R_X and G can be issued before the gather loop and converted after it.
template <typename S> struct Vec4;
template <> struct Vec4<double> { double2 lo, hi; };
template <> struct Vec4<float> { float4 v; };
__device__ __forceinline__ Vec4<double> ld4_stream(const double *p) {
  Vec4<double> r;
  r.lo = __ldcs(reinterpret_cast<const double2 *>(p));
  r.hi = __ldcs(reinterpret_cast<const double2 *>(p + 2));
  return r;
}
__device__ __forceinline__ Vec4<float> ld4_stream(const float *p) {
  Vec4<float> r;
  r.v = __ldcs(reinterpret_cast<const float4 *>(p));
  return r;
}
__device__ __forceinline__ void unpack(const Vec4<double> &x, double (&o)[4]) { o[0] = x.lo.x; o[1] = x.lo.y; o[2] = x.hi.x; o[3] = x.hi.y; }
__device__ __forceinline__ void unpack(const Vec4<float> &x, double (&o)[4]) { o[0] = x.v.x; o[1] = x.v.y; o[2] = x.v.z; o[3] = x.v.w; }
__device__ __forceinline__ void st4_stream(double *p, const double (&o)[4]) {
  __stcs(reinterpret_cast<double2 *>(p), make_double2(o[0], o[1]));
  __stcs(reinterpret_cast<double2 *>(p + 2), make_double2(o[2], o[3]));
}
__device__ __forceinline__ void st4_stream(float *p, const double (&o)[4]) {
  __stcs(reinterpret_cast<float4 *>(p), make_float4((float)o[0], (float)o[1], (float)o[2], (float)o[3]));
}

// S = storage type of R_X, R_Y, G (double or float).  Each CTA owns ROWS consecutive rows (and, with
// gridDim.y > 1, one strip of the 4-column vectors) so that the +-1 neighbour rows it re-reads are L1 hits.
// A thread owns one 4-column vector of one row.  Its streaming operands (R_X, G: touched once per
// step, evict-first) are requested BEFORE the gather loop so their DRAM latency runs under it, and the
// gather is unrolled UNR nonzeros deep: UNR column indices / values first, then UNR independent operand
// loads, then the FMAs -- (UNR + 2) 16/32-byte requests in flight per thread instead of one.
template <typename S, int ROWS, int UNR>
__global__ void __launch_bounds__(256) csr_fused_kernel(const int64_t *__restrict__ rowptr,
                                                        const int32_t *__restrict__ colind,
                                                        const float *__restrict__ valsf,
                                                        const double *__restrict__ dinv_out,
                                                        const S *__restrict__ RY, S *__restrict__ RX,
                                                        const S *__restrict__ G, const double *__restrict__ LY,
                                                        StepCoef k, int64_t m, int32_t N) {
  const int nvec_all = N >> 2;
  const int vper = (nvec_all + (int)gridDim.y - 1) / (int)gridDim.y;
  const int v0 = (int)blockIdx.y * vper;
  const int nvec = min(vper, nvec_all - v0);
  if (nvec <= 0) return;
  const int64_t r0 = (int64_t)blockIdx.x * ROWS;
  const int items = ROWS * nvec;
  for (int it = threadIdx.x; it < items; it += blockDim.x) {
    const int rl = it / nvec;
    const int v = v0 + (it - rl * nvec);
    const int64_t row = r0 + rl;
    if (row >= m) break;
    const int64_t idx = row * N + 4 * v;
    const Vec4<S> rxv = ld4_stream(RX + idx);
    Vec4<S> gv;
    if (G) gv = ld4_stream(G + idx);
    float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
    const int64_t t1 = rowptr[row + 1];
    for (int64_t t = rowptr[row]; t < t1; t += UNR) {
      int32_t col[UNR];
      float a[UNR];
#pragma unroll
      for (int u = 0; u < UNR; ++u) {
        const bool ok = t + u < t1;
        col[u] = ok ? colind[t + u] : (int32_t)row;
        a[u] = ok ? valsf[t + u] : 0.f;
      }
      float4 w[UNR];
#pragma unroll
      for (int u = 0; u < UNR; ++u) w[u] = ld4_as_float(RY + (int64_t)col[u] * N + 4 * v);
#pragma unroll
      for (int u = 0; u < UNR; ++u) {
        acc.x = fmaf(a[u], w[u].x, acc.x);
        acc.y = fmaf(a[u], w[u].y, acc.y);
        acc.z = fmaf(a[u], w[u].z, acc.z);
        acc.w = fmaf(a[u], w[u].w, acc.w);
      }
    }
    double ry[4], rx[4], out[4];
    ld4_as_double(RY + idx, ry);
    unpack(rxv, rx);
    const double ds = dinv_out ? dinv_out[row] : 1.0;
    const double T[4] = {(double)acc.x, (double)acc.y, (double)acc.z, (double)acc.w};
#pragma unroll
    for (int q = 0; q < 4; ++q) out[q] = k.a * (ds * T[q]) + k.b * ry[q] + k.cp * rx[q];
    if (G) {
      double g[4];
      unpack(gv, g);
      const double2 l0 = *reinterpret_cast<const double2 *>(LY + 4 * v);
      const double2 l1 = *reinterpret_cast<const double2 *>(LY + 4 * v + 2);
      out[0] += k.a * (g[0] * l0.x);
      out[1] += k.a * (g[1] * l0.y);
      out[2] += k.a * (g[2] * l1.x);
      out[3] += k.a * (g[3] * l1.y);
    }
    st4_stream(RX + idx, out);
  }
}

// ---- second-generation kernel ---------------------------------------------------------------------------------
// Same operation and thread <-> data map idea (a thread owns VEC consecutive columns of one row), but
//   * the CSR structure of the CTA's 64 rows (row pointers, column indices, folded FP32 values) is staged in shared
//     memory once per CTA, so the per-nonzero dependent chain is LDS -> gather instead of L2 -> gather;
//   * the gather is unrolled UNR nonzeros deep with all UNR operand loads issued before the first FMA;
//   * VEC = 2 halves the registers a thread needs for FP64 blocks (one 16-byte load per operand), which is what
//     lets MINB CTAs be resident per SM.
template <typename S, int VEC> struct RawVec;
template <> struct RawVec<double, 4> { double2 a, b; };
template <> struct RawVec<double, 2> { double2 a; };
template <> struct RawVec<float, 4> { float4 a; };
template <> struct RawVec<float, 2> { float2 a; };
__device__ __forceinline__ void ldraw(const double *p, RawVec<double, 4> &r) { r.a = *reinterpret_cast<const double2 *>(p); r.b = *reinterpret_cast<const double2 *>(p + 2); }
__device__ __forceinline__ void ldraw(const double *p, RawVec<double, 2> &r) { r.a = *reinterpret_cast<const double2 *>(p); }
__device__ __forceinline__ void ldraw(const float *p, RawVec<float, 4> &r) { r.a = *reinterpret_cast<const float4 *>(p); }
__device__ __forceinline__ void ldraw(const float *p, RawVec<float, 2> &r) { r.a = *reinterpret_cast<const float2 *>(p); }
__device__ __forceinline__ void ldraw_cs(const double *p, RawVec<double, 4> &r) { r.a = __ldcs(reinterpret_cast<const double2 *>(p)); r.b = __ldcs(reinterpret_cast<const double2 *>(p + 2)); }
__device__ __forceinline__ void ldraw_cs(const double *p, RawVec<double, 2> &r) { r.a = __ldcs(reinterpret_cast<const double2 *>(p)); }
__device__ __forceinline__ void ldraw_cs(const float *p, RawVec<float, 4> &r) { r.a = __ldcs(reinterpret_cast<const float4 *>(p)); }
__device__ __forceinline__ void ldraw_cs(const float *p, RawVec<float, 2> &r) { r.a = __ldcs(reinterpret_cast<const float2 *>(p)); }
__device__ __forceinline__ void unraw(const RawVec<double, 4> &r, double (&o)[4]) { o[0] = r.a.x; o[1] = r.a.y; o[2] = r.b.x; o[3] = r.b.y; }
__device__ __forceinline__ void unraw(const RawVec<double, 2> &r, double (&o)[2]) { o[0] = r.a.x; o[1] = r.a.y; }
__device__ __forceinline__ void unraw(const RawVec<float, 4> &r, float (&o)[4]) { o[0] = r.a.x; o[1] = r.a.y; o[2] = r.a.z; o[3] = r.a.w; }
__device__ __forceinline__ void unraw(const RawVec<float, 2> &r, float (&o)[2]) { o[0] = r.a.x; o[1] = r.a.y; }
__device__ __forceinline__ void straw_cs(double *p, const double (&o)[4]) { __stcs(reinterpret_cast<double2 *>(p), make_double2(o[0], o[1])); __stcs(reinterpret_cast<double2 *>(p + 2), make_double2(o[2], o[3])); }
__device__ __forceinline__ void straw_cs(double *p, const double (&o)[2]) { __stcs(reinterpret_cast<double2 *>(p), make_double2(o[0], o[1])); }
__device__ __forceinline__ void straw_cs(float *p, const float (&o)[4]) { __stcs(reinterpret_cast<float4 *>(p), make_float4(o[0], o[1], o[2], o[3])); }
__device__ __forceinline__ void straw_cs(float *p, const float (&o)[2]) { __stcs(reinterpret_cast<float2 *>(p), make_float2(o[0], o[1])); }

constexpr int CSR2_ROWS = 64;
constexpr int CSR2_CAP = 1024;      // staged nonzeros per CTA (16 per row on average); larger row blocks read the arrays directly

template <typename S, int VEC, int UNR, int MINB>
__global__ void __launch_bounds__(256, MINB) csr_fused_v2_kernel(const int64_t *__restrict__ rowptr,
                                                                 const int32_t *__restrict__ colind,
                                                                 const float *__restrict__ valsf,
                                                                 const double *__restrict__ dinv_out,
                                                                 const S *__restrict__ RY, S *__restrict__ RX,
                                                                 const S *__restrict__ G, const double *__restrict__ LY,
                                                                 StepCoef k, int64_t m, int32_t N) {
  __shared__ int32_t s_rp[CSR2_ROWS + 1];
  __shared__ int32_t s_col[CSR2_CAP];
  __shared__ float s_val[CSR2_CAP];
  const int64_t r0 = (int64_t)blockIdx.x * CSR2_ROWS;
  const int nrows = (int)min((int64_t)CSR2_ROWS, m - r0);
  const int64_t base = rowptr[r0];
  const int cnt = (int)min((int64_t)(CSR2_CAP + 1), rowptr[r0 + nrows] - base);
  const bool staged = cnt <= CSR2_CAP;
  for (int t = threadIdx.x; t <= nrows; t += blockDim.x) s_rp[t] = (int)(rowptr[r0 + t] - base);
  if (staged)
    for (int t = threadIdx.x; t < cnt; t += blockDim.x) {
      s_col[t] = colind[base + t];
      s_val[t] = valsf[base + t];
    }
  __syncthreads();
  const int nvec = N / VEC;
  const int items = nrows * nvec;
  const S ka = (S)k.a, kb = (S)k.b, kc = (S)k.cp;
  for (int it = threadIdx.x; it < items; it += blockDim.x) {
    const int rl = it / nvec;
    const int v = it - rl * nvec;
    const int64_t row = r0 + rl;
    const int64_t idx = row * N + VEC * v;
    RawVec<S, VEC> rxr, gr, ryr;
    ldraw_cs(RX + idx, rxr);
    if (G) ldraw_cs(G + idx, gr);
    float acc[VEC];
#pragma unroll
    for (int q = 0; q < VEC; ++q) acc[q] = 0.f;
    const int t1 = s_rp[rl + 1];
    for (int t = s_rp[rl]; t < t1; t += UNR) {
      int32_t col[UNR];
      float a[UNR];
#pragma unroll
      for (int u = 0; u < UNR; ++u) {
        const bool ok = t + u < t1;
        col[u] = ok ? (staged ? s_col[t + u] : colind[base + t + u]) : (int32_t)row;
        a[u] = ok ? (staged ? s_val[t + u] : valsf[base + t + u]) : 0.f;
      }
      RawVec<S, VEC> w[UNR];
#pragma unroll
      for (int u = 0; u < UNR; ++u) ldraw(RY + (int64_t)col[u] * N + VEC * v, w[u]);
#pragma unroll
      for (int u = 0; u < UNR; ++u) {
        S wv[VEC];
        unraw(w[u], wv);
#pragma unroll
        for (int q = 0; q < VEC; ++q) acc[q] = fmaf(a[u], (float)wv[q], acc[q]);
      }
    }
    ldraw(RY + idx, ryr);
    S ry[VEC], rx[VEC], out[VEC];
    unraw(ryr, ry);
    unraw(rxr, rx);
    const S ds = dinv_out ? (S)dinv_out[row] : (S)1;
#pragma unroll
    for (int q = 0; q < VEC; ++q) out[q] = ka * (ds * (S)acc[q]) + kb * ry[q] + kc * rx[q];
    if (G) {
      S g[VEC];
      unraw(gr, g);
#pragma unroll
      for (int q = 0; q < VEC; ++q) out[q] += ka * (g[q] * (S)LY[VEC * v + q]);
    }
    straw_cs(RX + idx, out);
  }
}

const LowpCopy *find_copy(const rchfsi_ctx *h, int prec, bool folded) {
  for (const LowpCopy &c : h->lowp)
    if (c.prec == prec && c.folded == folded) return &c;
  return nullptr;
}

}  // namespace

bool csr_fused_supported(const rchfsi_ctx *h) {
  return h->A.d.kind == RCHFSI_OP_CSR && (h->N % 4) == 0 && h->opt.apply_prec != RCHFSI_FP64 &&
         h->A.d.nnz < ((int64_t)1 << 31);
}

rchfsi_status csr_fused_step(rchfsi_ctx *h, const FusedStep &s) {
  const rchfsi_operator &op = h->A.d;
  const bool folded = !s.chfsi && h->dinv != nullptr;
  const LowpCopy *cp = find_copy(h, RCHFSI_FP32, folded);
  if (!cp) {
    LowpCopy c;
    c.prec = RCHFSI_FP32;
    c.folded = folded;
    c.bytes = sizeof(float) * (size_t)op.nnz;
    RCHFSI_TRY(dev_alloc(h, &c.data, c.bytes));
    fold_vals_kernel<<<(unsigned)std::max<int64_t>(1, std::min<int64_t>(cdiv(op.nnz, 256), 148 * 8)), 256, 0, h->stream>>>(
        op.vals, op.colind, folded ? h->dinv : nullptr, (float *)c.data, op.nnz);
    LAUNCH_CHECK(h);
    h->lowp.push_back(c);
    cp = &h->lowp.back();
  }
  const double *dinv_out = s.chfsi ? h->dinv : nullptr;
  const dim3 grid((unsigned)cdiv(h->m, CSR2_ROWS));
  const int variant = h->knobs.csr_variant;
#define CSR2_LAUNCH(STYPE, VEC, UNR, MINB)                                                                          \
  csr_fused_v2_kernel<STYPE, VEC, UNR, MINB><<<grid, 256, 0, h->stream>>>(                                          \
      op.rowptr, op.colind, (const float *)cp->data, dinv_out, (const STYPE *)s.RY, (STYPE *)s.RX, (const STYPE *)s.G, \
      s.LY, s.k, h->m, h->N)
  if (variant == 0) {
    if (s.store_prec == RCHFSI_FP64)
      csr_fused_kernel<double, 64, 1><<<grid, 256, 0, h->stream>>>(op.rowptr, op.colind, (const float *)cp->data, dinv_out,
                                                                    (const double *)s.RY, (double *)s.RX,
                                                                    (const double *)s.G, s.LY, s.k, h->m, h->N);
    else
      csr_fused_kernel<float, 64, 1><<<grid, 256, 0, h->stream>>>(op.rowptr, op.colind, (const float *)cp->data, dinv_out,
                                                                   (const float *)s.RY, (float *)s.RX, (const float *)s.G,
                                                                   s.LY, s.k, h->m, h->N);
  } else if (s.store_prec == RCHFSI_FP64) {
    switch (variant) {
      case 1: CSR2_LAUNCH(double, 4, 1, 4); break;
      case 2: CSR2_LAUNCH(double, 4, 2, 4); break;
      case 3: CSR2_LAUNCH(double, 4, 4, 3); break;
      case 4: CSR2_LAUNCH(double, 2, 1, 8); break;
      case 5: CSR2_LAUNCH(double, 2, 2, 8); break;
      case 6: CSR2_LAUNCH(double, 2, 4, 6); break;
      case 7: CSR2_LAUNCH(double, 2, 8, 5); break;
      default: CSR2_LAUNCH(double, 2, 4, 8); break;
    }
  } else {
    switch (variant) {
      case 1: CSR2_LAUNCH(float, 4, 1, 6); break;
      case 2: CSR2_LAUNCH(float, 4, 2, 6); break;
      case 3: CSR2_LAUNCH(float, 4, 4, 5); break;
      case 4: CSR2_LAUNCH(float, 2, 1, 8); break;
      case 5: CSR2_LAUNCH(float, 2, 2, 8); break;
      case 6: CSR2_LAUNCH(float, 2, 4, 8); break;
      case 7: CSR2_LAUNCH(float, 4, 8, 4); break;
      default: CSR2_LAUNCH(float, 4, 4, 6); break;
    }
  }
#undef CSR2_LAUNCH
  LAUNCH_CHECK(h);
  return RCHFSI_OK;
}

}  // namespace rchfsi
