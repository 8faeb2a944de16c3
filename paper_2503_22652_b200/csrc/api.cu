// C ABI of librchfsi.so (include/rchfsi.h): argument validation, workspace management and the
// host-side control flow of Algorithms 1-3.  All arithmetic on blocks
// runs in the CUDA kernels of this library; the host only computes the Chebyshev scalars.
#include <cmath>
#include <cstdlib>
#include <cstring>
#include "common.cuh"

using namespace rchfsi;

static thread_local std::string g_create_error;

namespace rchfsi {
rchfsi_status dev_alloc(rchfsi_ctx *h, void **p, size_t bytes) {
  void *q = nullptr;
  cudaError_t e = cudaMalloc(&q, bytes ? bytes : 16);
  if (e != cudaSuccess) {
    cudaGetLastError();
    h->err = "cudaMalloc(" + std::to_string(bytes) + " bytes): " + cudaGetErrorString(e);
    return e == cudaErrorMemoryAllocation ? RCHFSI_ENOMEM : RCHFSI_ECUDA;
  }
  h->owned.push_back(q);
  *p = q;
  return RCHFSI_OK;
}
}  // namespace rchfsi

extern "C" {

const char *rchfsi_version(void) { return "rchfsi 0.1 sm_100a"; }

void rchfsi_default_options(rchfsi_options *opt) {
  if (!opt) return;
  std::memset(opt, 0, sizeof(*opt));
  opt->apply_prec = RCHFSI_FP64;
  opt->store_prec = RCHFSI_FP64;
  opt->normalize_columns_before_rr = 1;
}

static bool operator_ok(const rchfsi_operator *op, std::string &why) {
  if (op->m <= 0) { why = "operator m <= 0"; return false; }
  if (op->m >= (int64_t)1 << 31) { why = "m must be < 2^31 (int32 indices)"; return false; }
  switch (op->kind) {
    case RCHFSI_OP_DENSE:
      if (!op->dense || op->lda < op->m) { why = "dense operator: null array or lda < m"; return false; }
      return true;
    case RCHFSI_OP_CSR:
      if (!op->rowptr || !op->colind || !op->vals || op->nnz < 0) { why = "CSR operator: null array"; return false; }
      return true;
    case RCHFSI_OP_FE:
      if (!op->conn || (!op->cell_mats && !op->cell_mats_f32) || op->n_cells <= 0 || op->n_loc <= 0) {
        why = "FE operator: null array or empty mesh";
        return false;
      }
      return true;
    default:
      why = "unknown operator kind";
      return false;
  }
}

// the environment is read here, once per handle, never on the per-step launch path
static Knobs read_knobs() {
  Knobs k;
  auto geti = [](const char *name, int dflt) {
    const char *e = getenv(name);
    return e ? atoi(e) : dflt;
  };
  k.fe_shadow_pair = getenv("RCHFSI_FE_SHADOW_PAIR") != nullptr;
  k.fe_legacy = geti("RCHFSI_FE_LEGACY", 0) != 0;
  k.dense_bn = geti("RCHFSI_DENSE_BN", 0);
  k.dense_ks = geti("RCHFSI_DENSE_KS", 0);
  k.dense_mc = geti("RCHFSI_DENSE_MC", -1);
  k.rr_chunked = geti("RCHFSI_RR_CHUNKED", -1);
  k.rr_fe_simt = getenv("RCHFSI_RR_FE_SIMT") != nullptr;
  k.rr_timing = getenv("RCHFSI_RR_TIMING") != nullptr;
  k.rr_split = geti("RCHFSI_RR_SPLIT", -1);
  k.host_chunk = geti("RCHFSI_HOST_CHUNK", 0);
  k.csr_variant = geti("RCHFSI_CSR_VARIANT", 0);
#ifdef RCHFSI_PROBES
  k.tc_debug = geti("RCHFSI_TC_DEBUG", 0);
#endif
  return k;
}

static bool aligned16(const void *p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

rchfsi_status rchfsi_create(rchfsi_handle *out, const rchfsi_operator *A, const rchfsi_operator *B,
                            const double *dinv_diag, int32_t block_N, const rchfsi_options *opt,
                            void *cuda_stream) {
  if (!out || !A) { g_create_error = "rchfsi_create: null argument"; return RCHFSI_EINVAL; }
  std::string why;
  if (!operator_ok(A, why)) { g_create_error = "A: " + why; return RCHFSI_EINVAL; }
  if (B && !operator_ok(B, why)) { g_create_error = "B: " + why; return RCHFSI_EINVAL; }
  if (B && B->m != A->m) { g_create_error = "A and B differ in size"; return RCHFSI_EINVAL; }
  if (block_N < 1 || block_N > A->m) { g_create_error = "block_N must satisfy 1 <= N <= m"; return RCHFSI_EINVAL; }
  rchfsi_options o;
  rchfsi_default_options(&o);
  if (opt) o = *opt;
  if (o.apply_prec < RCHFSI_FP64 || o.apply_prec > RCHFSI_BF16) { g_create_error = "unknown apply_prec"; return RCHFSI_EINVAL; }
  if (o.store_prec != RCHFSI_FP64 && o.store_prec != RCHFSI_FP32) { g_create_error = "store_prec must be FP64 or FP32"; return RCHFSI_EINVAL; }
  if (o.store_prec == RCHFSI_FP32 && o.apply_prec == RCHFSI_FP64) { g_create_error = "store FP32 needs a reduced apply_prec"; return RCHFSI_EINVAL; }
  if (o.g_input_f32 && o.store_prec != RCHFSI_FP32) { g_create_error = "g_input_f32 needs store_prec FP32"; return RCHFSI_EINVAL; }
  if (o.noise_eps < 0) { g_create_error = "noise_eps < 0"; return RCHFSI_EINVAL; }
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) {
    cudaGetLastError();
    g_create_error = "no CUDA device (this library has no CPU fallback)";
    return RCHFSI_ECUDA;
  }
  rchfsi_ctx *h = new (std::nothrow) rchfsi_ctx();
  if (!h) { g_create_error = "out of host memory"; return RCHFSI_ENOMEM; }
  h->A.d = *A; h->A.present = true;
  if (B) { h->B.d = *B; h->B.present = true; }
  h->dinv = dinv_diag;
  h->m = A->m;
  h->N = block_N;
  h->N_cap = block_N;
  h->opt = o;
  h->stream = reinterpret_cast<cudaStream_t>(cuda_stream);
  h->knobs = read_knobs();
  {
    int dev = 0;
    cudaGetDevice(&dev);
    if (cudaDeviceGetAttribute(&h->num_sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || h->num_sms <= 0) h->num_sms = 148;
  }
  for (const rchfsi_operator *op : {A, B}) {
    if (op && op->kind == RCHFSI_OP_FE) {
      double asym = 0.0;
      rchfsi_status s = fe_check_symmetric(h, *op, &asym);
      if (s != RCHFSI_OK) { g_create_error = h->err; delete h; return s; }
      if (asym > (op->cell_mats ? 1e-10 : 1e-5)) {
        g_create_error = "FE cell matrices are not symmetric (relative asymmetry " + std::to_string(asym) + ")";
        delete h;
        return RCHFSI_EINVAL;
      }
    }
  }
  if (A->kind == RCHFSI_OP_FE) {
    // colouring of the cell conflict graph; also validates conn (range, every row covered by a cell)
    rchfsi_status s = fe_ensure_coloring(h);
    if (s != RCHFSI_OK) { g_create_error = h->err; rchfsi_destroy(h); return s; }
  }
  if (cudaEventCreate(&h->ev_step0) != cudaSuccess || cudaEventCreate(&h->ev_step1) != cudaSuccess) {
    g_create_error = "cudaEventCreate failed";
    delete h;
    return RCHFSI_ECUDA;
  }
  *out = h;
  return RCHFSI_OK;
}

rchfsi_status rchfsi_destroy(rchfsi_handle h) {
  if (!h) return RCHFSI_EINVAL;
  cudaStreamSynchronize(h->stream);
  for (void *p : h->owned) cudaFree(p);
  if (h->cublas) cublasDestroy(h->cublas);
  if (h->cusolver) cusolverDnDestroy(h->cusolver);
  for (int i = 0; i < rchfsi_ctx::HOST_SETS; ++i)
    for (cudaEvent_t e : {h->ev_g[i], h->ev_xin[i], h->ev_done[i], h->ev_free[i]})
      if (e) cudaEventDestroy(e);
  if (h->in_stream) cudaStreamDestroy(h->in_stream);
  if (h->out_stream) cudaStreamDestroy(h->out_stream);
  if (h->ev_step0) cudaEventDestroy(h->ev_step0);
  if (h->ev_step1) cudaEventDestroy(h->ev_step1);
  delete h;
  return RCHFSI_OK;
}

rchfsi_status rchfsi_operator_changed(rchfsi_handle h) {
  if (!h) return RCHFSI_EINVAL;
  RCHFSI_CUDA_CHECK(h, cudaStreamSynchronize(h->stream));
  // the reduced-precision copies (with D^-1 folded in) and the TMA descriptors onto them are rebuilt on the next step
  for (rchfsi::LowpCopy &c : h->lowp) {
    for (size_t i = 0; i < h->owned.size(); ++i)
      if (h->owned[i] == c.data) { h->owned.erase(h->owned.begin() + i); break; }
    cudaFree(c.data);
  }
  h->lowp.clear();
  h->tmaps.clear();
  return RCHFSI_OK;
}

const char *rchfsi_last_error(rchfsi_handle h) { return h ? h->err.c_str() : g_create_error.c_str(); }

int64_t rchfsi_launch_count(rchfsi_handle h) { return h ? h->launches : -1; }

rchfsi_status rchfsi_last_filter_step_ms(rchfsi_handle h, float *ms_total_out, int32_t *steps_out) {
  if (!h || !ms_total_out || !steps_out) return RCHFSI_EINVAL;
  RCHFSI_CUDA_CHECK(h, cudaStreamSynchronize(h->stream));
  float ms = 0.f;
  if (h->last_steps > 0) RCHFSI_CUDA_CHECK(h, cudaEventElapsedTime(&ms, h->ev_step0, h->ev_step1));
  *ms_total_out = ms;
  *steps_out = h->last_steps;
  return RCHFSI_OK;
}

size_t rchfsi_workspace_bytes(const rchfsi_operator *A, const rchfsi_operator *B, int32_t block_N,
                              const rchfsi_options *opt) {
  if (!A || block_N < 1) return 0;
  rchfsi_options o;
  rchfsi_default_options(&o);
  if (opt) o = *opt;
  const size_t el = (size_t)A->m * block_N;
  const size_t s = prec_bytes(o.store_prec);
  size_t total = 2 * el * s;                              // R_X, R_Y
  if (o.store_prec != RCHFSI_FP64) total += el * s;       // storage-precision copy of G
  total += 2 * el * 4;                                    // operand shadows (worst case FP32)
  total += el * 8;                                        // unfused operator output / G scratch
  total += (B ? 3 : 2) * el * 8 + el * 8;                 // Rayleigh-Ritz temporaries + solve's G
  total += 2 * (size_t)block_N * block_N * 8 * 2;         // Gram matrices + dsygvd workspace (approx.)
  if (A->kind == RCHFSI_OP_DENSE && o.apply_prec != RCHFSI_FP64) total += (size_t)A->m * A->m * 4;
  if (A->kind == RCHFSI_OP_FE && o.apply_prec != RCHFSI_FP64)
    total += (size_t)A->n_cells * 352 * 352 * (o.apply_prec == RCHFSI_BF16 ? 2 : 4);
  if (A->kind == RCHFSI_OP_FE) total += (size_t)1600 << 20;   // gather / product / FP64 cell-batch scratch of the Rayleigh-Ritz applies
  return total;
}

rchfsi_status rchfsi_apply(rchfsi_handle h, int32_t which, const double *V, double *out) {
  if (!h) return RCHFSI_EINVAL;
  if (!V || !out || V == out || (which != 0 && which != 1)) { h->err = "rchfsi_apply: bad argument"; return RCHFSI_EINVAL; }
  if (which == 1 && !h->B.present) {
    RCHFSI_CUDA_CHECK(h, cudaMemcpyAsync(out, V, sizeof(double) * (size_t)h->m * h->N, cudaMemcpyDeviceToDevice, h->stream));
    return RCHFSI_OK;
  }
  return op_apply_simt<double>(h, which == 0 ? h->A.d : h->B.d, nullptr, V, out, h->N);
}

rchfsi_status rchfsi_rayleigh_ritz(rchfsi_handle h, double *Y_in_X_out, double *ritz_out, double *G_out,
                                   double *resnorm_out) {
  if (!h) return RCHFSI_EINVAL;
  if (!Y_in_X_out || !ritz_out || !aligned16(Y_in_X_out) || (G_out && !aligned16(G_out))) {
    h->err = "rchfsi_rayleigh_ritz: null or misaligned pointer";
    return RCHFSI_EINVAL;
  }
  if (rr_wants_chunked(h)) return rayleigh_ritz_chunked(h, Y_in_X_out, ritz_out, G_out, RCHFSI_FP64, resnorm_out);
  return rayleigh_ritz_impl(h, Y_in_X_out, ritz_out, G_out, resnorm_out);
}

}  // extern "C"
