// Fused CSR step: T_i = sum_t a_it W_{col_t} in FP32 on the ALUs with
// 128-bit coalesced loads along the N contiguous columns, and the Alg. 3 update
//   R_X <- a T + b R_Y + c' R_X + a G Lambda_Y
// as the epilogue of the same thread, so every block crosses HBM once per step: R_Y, R_X and G
// are read once, R_X is written once.  The operand W is R_Y itself (converted to FP32 on the
// fly when the recurrence is stored in FP64); D^-1 is folded into the FP32 copy of the values
// (a_it * dinv[col_t]), which is exact algebra for A D^-1 ("A D^-1 R_Y").
#include <algorithm>
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

// S = storage type of R_X, R_Y, G (double or float).  Each CTA owns CSR_ROWS consecutive rows so that the +-1
// neighbour rows it re-reads are L1 hits.  A thread owns one 4-column vector of one row.  Its streaming operands
// (R_X, G: touched once per step, evict-first) are requested BEFORE the gather loop so their DRAM latency runs under
// it.  64 registers x 256 threads = 4 CTAs per SM.  Measured and dropped: deeper gather unrolling, the
// CSR structure of the row block staged in shared memory, 2 columns per thread, 5-8 or 1-3 resident CTAs per SM,
// column strips, row interleaving -- every one of them slower than this plain form.
constexpr int CSR_ROWS = 64;
template <typename S>
__global__ void __launch_bounds__(256, 4) csr_fused_kernel(const int64_t *__restrict__ rowptr,
                                                           const int32_t *__restrict__ colind,
                                                           const float *__restrict__ valsf,
                                                           const double *__restrict__ dinv_out,
                                                           const S *__restrict__ RY, S *__restrict__ RX,
                                                           const S *__restrict__ G, const double *__restrict__ LY,
                                                           StepCoef k, int64_t m, int32_t N) {
  const int nvec = N >> 2;
  const int64_t r0 = (int64_t)blockIdx.x * CSR_ROWS;
  const int items = CSR_ROWS * nvec;
  for (int it = threadIdx.x; it < items; it += blockDim.x) {
    const int rl = it / nvec;
    const int v = it - rl * nvec;
    const int64_t row = r0 + rl;
    if (row >= m) break;
    const int64_t idx = row * N + 4 * v;
    const Vec4<S> rxv = ld4_stream(RX + idx);
    Vec4<S> gv;
    if (G) gv = ld4_stream(G + idx);
    float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
    const int64_t t1 = rowptr[row + 1];
    for (int64_t t = rowptr[row]; t < t1; ++t) {
      const float a = valsf[t];
      const float4 w = ld4_as_float(RY + (int64_t)colind[t] * N + 4 * v);
      acc.x = fmaf(a, w.x, acc.x);
      acc.y = fmaf(a, w.y, acc.y);
      acc.z = fmaf(a, w.z, acc.z);
      acc.w = fmaf(a, w.w, acc.w);
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

LowpCopy *find_copy(rchfsi_ctx *h, int prec, bool folded) {
  for (LowpCopy &c : h->lowp)
    if (c.prec == prec && c.folded == folded) return &c;
  return nullptr;
}

}  // namespace

bool csr_fused_supported(const rchfsi_operator &A, int32_t N, const rchfsi_options &opt) {
  return A.kind == RCHFSI_OP_CSR && (N % 4) == 0 && opt.apply_prec != RCHFSI_FP64 && A.nnz < ((int64_t)1 << 31);
}
size_t csr_lowp_bytes(const rchfsi_operator &A) { return sizeof(float) * (size_t)A.nnz; }

// the folded FP32 copy of the values: allocated (and built) on first use, or up front by rchfsi_solve
static rchfsi_status csr_copy(rchfsi_ctx *h, bool folded, LowpCopy **out) {
  const rchfsi_operator &op = h->A.d;
  LowpCopy *cp = find_copy(h, RCHFSI_FP32, folded);
  if (!cp) {
    LowpCopy c;
    c.prec = RCHFSI_FP32;
    c.folded = folded;
    c.stale = true;
    c.bytes = csr_lowp_bytes(op);
    RCHFSI_TRY(dev_alloc(h, &c.data, c.bytes));
    h->lowp.push_back(c);
    cp = &h->lowp.back();
  }
  if (cp->stale) {
    fold_vals_kernel<<<(unsigned)std::max<int64_t>(1, std::min<int64_t>(cdiv(op.nnz, 256), 148 * 8)), 256, 0, h->stream>>>(
        op.vals, op.colind, folded ? h->dinv : nullptr, (float *)cp->data, op.nnz);
    LAUNCH_CHECK(h);
    cp->stale = false;
  }
  *out = cp;
  return RCHFSI_OK;
}
rchfsi_status csr_fused_prepare(rchfsi_ctx *h, bool chfsi) {
  LowpCopy *cp = nullptr;
  return csr_copy(h, !chfsi && h->dinv != nullptr, &cp);
}

rchfsi_status csr_fused_step(rchfsi_ctx *h, const FusedStep &s) {
  const rchfsi_operator &op = h->A.d;
  LowpCopy *cp = nullptr;
  RCHFSI_TRY(csr_copy(h, !s.chfsi && h->dinv != nullptr, &cp));
  const double *dinv_out = s.chfsi ? h->dinv : nullptr;
  const dim3 grid((unsigned)cdiv(h->m, CSR_ROWS));
  if (s.store_prec == RCHFSI_FP64)
    csr_fused_kernel<double><<<grid, 256, 0, h->stream>>>(op.rowptr, op.colind, (const float *)cp->data, dinv_out,
                                                           (const double *)s.RY, (double *)s.RX, (const double *)s.G, s.LY,
                                                           s.k, h->m, h->N);
  else
    csr_fused_kernel<float><<<grid, 256, 0, h->stream>>>(op.rowptr, op.colind, (const float *)cp->data, dinv_out,
                                                          (const float *)s.RY, (float *)s.RX, (const float *)s.G, s.LY, s.k,
                                                          h->m, h->N);
  LAUNCH_CHECK(h);
  return RCHFSI_OK;
}

}  // namespace rchfsi
