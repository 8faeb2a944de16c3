// Interface exchange of a ROW-SHARDED R-ChFSI filter.  The paper distributes the FE
// operator over MPI ranks and exchanges only nearest-neighbour interface data inside each matvec, optionally "in BF16
// precision; we term this method TF32B", "reducing inter-node message sizes by a factor of 4"
// (PAPER.md:357).  B200 form: one process per GPU owns a slab of cells and ALL rows its cells touch; the rows on the
// plane between two slabs are replicated on both ranks.  A local step (rchfsi_filter_step) gives, on an interface
// row, only this rank's share of the product:
//     R_new^(r) = base + a T_r,     base = b R_Y + c' R_X + a G Lambda_Y  (identical on both ranks),
// and the assembled row is base + a T_r + a T_r'.  Per step and interface:
//   rchfsi_interface_save   before the step: keep the old R_X rows (the step overwrites them);
//   rchfsi_interface_pack   after the step: base (recomputed, FP64) and delta = R_new - base = a T_r, rounded to the
//                           WIRE precision (BF16 / FP32 / FP64) into the send buffer;
//   [the caller exchanges send buffers with the neighbour: NCCL send/recv over NVLink, torch.distributed]
//   rchfsi_interface_apply  R_new = base + (delta_own + delta_nbr) with BOTH deltas in wire precision, so the two
//                           replicas of the row stay bit-identical (the sum of two numbers is commutative), and the
//                           operand shadow of the row is refreshed.
// With a BF16 wire the interface rows carry an O(2^-9) relative error in their share of the product: an inexact
// matvec, which is exactly what the residual recurrence tolerates (Thm 3.4).
#include <algorithm>
#include <cuda_bf16.h>
#include "common.cuh"

namespace rchfsi {
namespace {

__device__ __forceinline__ double ld_prec(const void *p, int64_t i, int prec) {
  return prec == RCHFSI_FP64 ? reinterpret_cast<const double *>(p)[i] : (double)reinterpret_cast<const float *>(p)[i];
}
__device__ __forceinline__ void st_prec(void *p, int64_t i, int prec, double v) {
  if (prec == RCHFSI_FP64) reinterpret_cast<double *>(p)[i] = v;
  else reinterpret_cast<float *>(p)[i] = (float)v;
}
__device__ __forceinline__ void st_wire(void *p, int64_t i, int wire, double v) {
  if (wire == RCHFSI_BF16) reinterpret_cast<__nv_bfloat16 *>(p)[i] = __float2bfloat16_rn((float)v);
  else if (wire == RCHFSI_FP32) reinterpret_cast<float *>(p)[i] = (float)v;
  else reinterpret_cast<double *>(p)[i] = v;
}
__device__ __forceinline__ double ld_wire(const void *p, int64_t i, int wire) {
  if (wire == RCHFSI_BF16) return (double)__bfloat162float(reinterpret_cast<const __nv_bfloat16 *>(p)[i]);
  if (wire == RCHFSI_FP32) return (double)reinterpret_cast<const float *>(p)[i];
  return reinterpret_cast<const double *>(p)[i];
}
// element (row, j) of a library-owned block: panel layout [ceil(N/128)][m][128] when pm != 0, else row-major [m][N]
__device__ __forceinline__ int64_t lib_index(int64_t row, int j, int32_t N, int64_t pm) {
  return pm ? (((int64_t)(j >> 7) * pm + row) << 7) + (j & 127) : row * N + j;
}

struct IfArgs {
  const int32_t *rows;
  int32_t n_rows, N;
  int64_t pm;            // panel layout stride (m) of the library-owned blocks, 0 = row-major
  int store, wire, shadow_prec;
  StepCoef k;
  const double *LY;      // Lambda_Y row of the last step
  const void *prevY;     // R_Y of the last step (after the swap: run.RX)
  void *newR;            // result block of the last step (after the swap: run.RY)
  const void *G;
  int g_lib;             // G in the library layout (else caller's row-major [m][N])
  void *shadow;          // operand shadow of newR or NULL
  void *old_rows;        // [n_rows][N] storage precision: R_X rows before the step
  double *base;          // [n_rows][N]
};

__global__ void if_save_kernel(IfArgs a, const void *RX) {
  const int64_t total = (int64_t)a.n_rows * a.N;
  for (int64_t t = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; t < total; t += (int64_t)gridDim.x * blockDim.x) {
    const int64_t i = t / a.N;
    const int j = (int)(t - i * a.N);
    st_prec(a.old_rows, t, a.store, ld_prec(RX, lib_index(a.rows[i], j, a.N, a.pm), a.store));
  }
}

__global__ void if_pack_kernel(IfArgs a, void *send) {
  const int64_t total = (int64_t)a.n_rows * a.N;
  for (int64_t t = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; t < total; t += (int64_t)gridDim.x * blockDim.x) {
    const int64_t i = t / a.N;
    const int j = (int)(t - i * a.N);
    const int64_t row = a.rows[i];
    const int64_t li = lib_index(row, j, a.N, a.pm);
    double base = a.k.b * ld_prec(a.prevY, li, a.store) + a.k.cp * ld_prec(a.old_rows, t, a.store);
    if (a.G) base += a.k.a * (ld_prec(a.G, a.g_lib ? li : row * a.N + j, a.store) * a.LY[j]);
    a.base[t] = base;
    st_wire(send, t, a.wire, ld_prec(a.newR, li, a.store) - base);
  }
}

__global__ void if_apply_kernel(IfArgs a, const void *own, const void *nbr) {
  const int64_t total = (int64_t)a.n_rows * a.N;
  for (int64_t t = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; t < total; t += (int64_t)gridDim.x * blockDim.x) {
    const int64_t i = t / a.N;
    const int j = (int)(t - i * a.N);
    const int64_t li = lib_index(a.rows[i], j, a.N, a.pm);
    const double v = a.base[t] + (ld_wire(own, t, a.wire) + ld_wire(nbr, t, a.wire));
    st_prec(a.newR, li, a.store, v);
    if (a.shadow) {
      const double s = ld_prec(a.newR, li, a.store);        // the stored (storage-precision) value is what the shadow mirrors
      if (a.shadow_prec == RCHFSI_BF16) reinterpret_cast<__nv_bfloat16 *>(a.shadow)[li] = __float2bfloat16_rn((float)s);
      else if (a.shadow_prec == RCHFSI_FP64) reinterpret_cast<double *>(a.shadow)[li] = s;
      else {
        uint32_t u;                                          // TF32 operands are stored as rounded FP32 bit patterns
        asm("cvt.rna.tf32.f32 %0, %1;" : "=r"(u) : "f"((float)s));
        reinterpret_cast<uint32_t *>(a.shadow)[li] = u;
      }
    }
  }
}

rchfsi_status if_args(rchfsi_ctx *h, const int32_t *rows, int32_t n_rows, int32_t wire, IfArgs *out, const char *who) {
  const FilterRun &r = h->run;
  if (!r.active) { h->err = std::string(who) + ": no filter in progress (rchfsi_filter_begin)"; return RCHFSI_EINVAL; }
  if (r.chfsi) { h->err = std::string(who) + ": the row-sharded exchange supports METHOD_RCHFSI (Algorithm 3) only"; return RCHFSI_EINVAL; }
  if (!rows || n_rows < 1 || n_rows > h->m) { h->err = std::string(who) + ": bad row list"; return RCHFSI_EINVAL; }
  if (wire != RCHFSI_FP64 && wire != RCHFSI_FP32 && wire != RCHFSI_BF16) { h->err = std::string(who) + ": wire precision must be FP64, FP32 or BF16"; return RCHFSI_EINVAL; }
  const size_t need = (size_t)n_rows * h->N_cap;
  if (h->if_cap < need) {
    if (h->if_old_cap < need) { RCHFSI_TRY(dev_alloc(h, &h->if_old, need * 8)); h->if_old_cap = need; }
    if (h->if_base_cap < need) { RCHFSI_TRY(dev_alloc(h, &h->if_base, need * 8)); h->if_base_cap = need; }
    h->if_cap = need;
  }
  IfArgs a{};
  a.rows = rows;
  a.n_rows = n_rows;
  a.N = h->N;
  a.pm = r.pl.panel ? h->m : 0;
  a.store = r.pl.store;
  a.wire = wire;
  a.shadow_prec = r.pl.operand == RCHFSI_BF16 ? RCHFSI_BF16 : (r.pl.operand == RCHFSI_FP64 ? RCHFSI_FP64 : RCHFSI_TF32);
  a.k = r.last;
  a.LY = r.last_LY;
  a.prevY = r.RX;
  a.newR = r.RY;
  a.G = r.Gst;
  a.g_lib = r.g_lib ? 1 : 0;
  a.shadow = r.pl.shadow ? r.Wcur : nullptr;
  a.old_rows = h->if_old;
  a.base = reinterpret_cast<double *>(h->if_base);
  *out = a;
  return RCHFSI_OK;
}

inline unsigned if_grid(int64_t total) { return (unsigned)std::max<int64_t>(1, std::min<int64_t>(cdiv(total, 256), 148 * 8)); }

}  // namespace
}  // namespace rchfsi

using namespace rchfsi;

extern "C" {

rchfsi_status rchfsi_interface_save(rchfsi_handle h, const int32_t *rows, int32_t n_rows) {
  if (!h) return RCHFSI_EINVAL;
  IfArgs a;
  RCHFSI_TRY(if_args(h, rows, n_rows, RCHFSI_FP64, &a, "rchfsi_interface_save"));
  if_save_kernel<<<if_grid((int64_t)n_rows * a.N), 256, 0, h->stream>>>(a, h->run.RX);   // the block the next step overwrites
  LAUNCH_CHECK(h);
  return RCHFSI_OK;
}

rchfsi_status rchfsi_interface_pack(rchfsi_handle h, const int32_t *rows, int32_t n_rows, int32_t wire_prec, void *send_buf) {
  if (!h) return RCHFSI_EINVAL;
  if (!send_buf) { h->err = "rchfsi_interface_pack: null send buffer"; return RCHFSI_EINVAL; }
  IfArgs a;
  RCHFSI_TRY(if_args(h, rows, n_rows, wire_prec, &a, "rchfsi_interface_pack"));
  if (!a.LY) { h->err = "rchfsi_interface_pack: no step has run yet"; return RCHFSI_EINVAL; }
  if_pack_kernel<<<if_grid((int64_t)n_rows * a.N), 256, 0, h->stream>>>(a, send_buf);
  LAUNCH_CHECK(h);
  return RCHFSI_OK;
}

rchfsi_status rchfsi_interface_apply(rchfsi_handle h, const int32_t *rows, int32_t n_rows, int32_t wire_prec,
                                     const void *own_buf, const void *nbr_buf) {
  if (!h) return RCHFSI_EINVAL;
  if (!own_buf || !nbr_buf) { h->err = "rchfsi_interface_apply: null buffer"; return RCHFSI_EINVAL; }
  IfArgs a;
  RCHFSI_TRY(if_args(h, rows, n_rows, wire_prec, &a, "rchfsi_interface_apply"));
  if_apply_kernel<<<if_grid((int64_t)n_rows * a.N), 256, 0, h->stream>>>(a, own_buf, nbr_buf);
  LAUNCH_CHECK(h);
  return RCHFSI_OK;
}

}  // extern "C"
