// C ABI of librchfsi.so (include/rchfsi.h): argument validation, workspace management and the
// host-side control flow of Algorithms 1-3.  All arithmetic on blocks
// runs in the CUDA kernels of this library; the host only computes the Chebyshev scalars.
#include <algorithm>
#include <cmath>
#include <cstdlib>
#include <cstring>
#include "common.cuh"

using namespace rchfsi;

static thread_local std::string g_create_error;

namespace rchfsi {
// Every device buffer of a handle is carved from the caller's workspace segments (rchfsi_add_workspace): first fit,
// 256-byte aligned, never returned (buffers live as long as the handle).  The library itself never calls cudaMalloc.
constexpr size_t WS_ALIGN = 256;
rchfsi_status dev_alloc(rchfsi_ctx *h, void **p, size_t bytes) {
  const size_t need = (std::max<size_t>(bytes, 16) + WS_ALIGN - 1) / WS_ALIGN * WS_ALIGN;
  for (WorkspaceSegment &sg : h->segments) {
    const size_t pad = (WS_ALIGN - (reinterpret_cast<uintptr_t>(sg.base) + sg.used) % WS_ALIGN) % WS_ALIGN;
    if (sg.used + pad + need <= sg.size) {
      *p = sg.base + sg.used + pad;
      sg.used += pad + need;
      h->ws_used += need;
      h->shortfall = 0;
      return RCHFSI_OK;
    }
  }
  h->shortfall = need + WS_ALIGN;
  h->err = "workspace exhausted: a buffer of " + std::to_string(need) + " bytes does not fit (" + std::to_string(h->ws_used) +
           " bytes in use); add a segment of rchfsi_workspace_shortfall() bytes with rchfsi_add_workspace and call again";
  return RCHFSI_ENOMEM;
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
  k.rr_fe_batched = getenv("RCHFSI_RR_FE_BATCHED") != nullptr;
  k.rr_split = geti("RCHFSI_RR_SPLIT", -1);
  k.rr_i8_rows = geti("RCHFSI_RR_I8_ROWS", 0);
  k.rr_gram_i8 = geti("RCHFSI_RR_GRAM_I8", -1);
  k.rr_i8_bn = geti("RCHFSI_RR_I8_BN", 128);
  k.host_chunk = geti("RCHFSI_HOST_CHUNK", 0);
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
    rchfsi_status s = fe_build_coloring(h);
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
  // the reduced-precision copies (with D^-1 folded in) keep their buffers; their contents are rebuilt on the next step
  for (rchfsi::LowpCopy &c : h->lowp) c.stale = true;
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

rchfsi_status rchfsi_add_workspace(rchfsi_handle h, void *device_buffer, size_t bytes) {
  if (!h) return RCHFSI_EINVAL;
  if (!device_buffer || bytes < 2 * WS_ALIGN) { h->err = "rchfsi_add_workspace: null buffer or fewer than 512 bytes"; return RCHFSI_EINVAL; }
  h->segments.push_back(rchfsi::WorkspaceSegment{static_cast<char *>(device_buffer), bytes, 0});
  h->shortfall = 0;
  return RCHFSI_OK;
}

size_t rchfsi_workspace_shortfall(rchfsi_handle h) { return h ? h->shortfall : 0; }
size_t rchfsi_workspace_used(rchfsi_handle h) { return h ? h->ws_used : 0; }

// Planner: the same buffers, by the same rules, as the allocation sites (ensure_filter_workspace, ensure_rr_workspace,
// rchfsi_solve, rchfsi_filter_host, rchfsi_estimate_bounds, the reduced-precision operator copies), each rounded up
// to the allocator's granule.  An upper bound that a single segment of this size satisfies; tests check both.
size_t rchfsi_workspace_bytes(const rchfsi_operator *A, const rchfsi_operator *B, int32_t block_N,
                              const rchfsi_options *opt, int32_t uses, int32_t max_degree) {
  if (!A || block_N < 1) return 0;
  rchfsi_options o;
  rchfsi_default_options(&o);
  if (opt) o = *opt;
  const Knobs kn = read_knobs();
  const Plan pl = make_plan(*A, block_N, o, kn);
  const size_t m = (size_t)A->m, N = (size_t)block_N;
  auto al = [](size_t b) { return (std::max<size_t>(b, 16) + WS_ALIGN - 1) / WS_ALIGN * WS_ALIGN + WS_ALIGN; };
  size_t total = 0;
  const size_t el = m * N, el_lib = m * (pl.panel ? (size_t)cdiv(block_N, 128) * 128 : N);
  const bool fe = A->kind == RCHFSI_OP_FE;
  if (fe) total += al(4 * (size_t)A->n_cells) + al((size_t)A->n_cells * A->n_loc);            // colouring: cell order + flags
  const bool want_filter = uses & (RCHFSI_USE_FILTER | RCHFSI_USE_SOLVE | RCHFSI_USE_FILTER_HOST);
  if (want_filter) {
    total += 2 * al(el_lib * prec_bytes(pl.store));                                           // R_X, R_Y
    if (pl.shadow) total += (pl.shadow_inplace ? 1 : 2) * al(el_lib * (pl.operand == RCHFSI_BF16 ? 2 : 4));
    if (pl.fused == 0) total += al(el_lib * prec_bytes(pl.tprec));                            // unfused operator output
    if (!o.g_input_f32 && (pl.store != RCHFSI_FP64 || pl.panel)) total += al(el_lib * prec_bytes(pl.store));   // G in storage layout
    total += al(8 * (size_t)(std::max(max_degree, 1) + 1) * N) + al(16 * N);                  // Lambda_k table, column norms
    if (uses & RCHFSI_USE_FILTER_NULL_G) total += 2 * al(el * 8);                             // G = NULL: A X and G in FP64
    // reduced-precision operator copies: with and without D^-1 folded in (R-ChFSI / ChFSI)
    size_t lp = 0;
    if (pl.fused == 1) lp = al(csr_lowp_bytes(*A));
    if (pl.fused == 2) lp = al(dense_lowp_bytes(*A, o.apply_prec));
    if (pl.fused == 3) lp = al(fe_lowp_bytes(*A, o.apply_prec));
    total += 2 * lp;
  }
  if (uses & (RCHFSI_USE_RAYLEIGH_RITZ | RCHFSI_USE_SOLVE)) {
    total += (B ? 3 : 2) * al(el * 8);                                                        // A Y, (B Y), rotation target
    total += 2 * al(8 * N * N) + 2 * al(8 * N) + al(16 * N) + al(4);                          // Gram matrices, Ritz values, residuals
    total += al(8 * (3 * N * N + 16 * N + 64) + ((size_t)8 << 20));                              // dsygvd workspace (cuSOLVER query at run time)
    if (fe) total += fe_rr_scratch_bytes(*A, block_N, A->n_cells);
    total += rr_i8_plan_bytes((int64_t)m, block_N) + al(std::min<size_t>(el * 8, (size_t)3e9 + 8 * N));   // INT8 products (rr_i8.cu), row panel of rchfsi_rotate
  }
  if (uses & RCHFSI_USE_SOLVE) total += al(el * 8);                                           // residual block of the solve
  if (uses & RCHFSI_USE_FILTER_HOST) {
    const size_t gb = o.g_input_f32 ? 4 : 8;
    total += 3 * (al(el * 8) + al(el * gb)) + al(8 * N);                                      // at most the whole block per staging set
  }
  if (uses & RCHFSI_USE_BOUNDS) {
    total += al(8 * (5 * m + 4));
    if (fe) total += al(8 * (2 * (size_t)A->n_loc * A->n_loc + A->n_loc + 2)) + al(8 * (3 * (size_t)A->n_loc * A->n_loc + 64 * (size_t)A->n_loc) + ((size_t)1 << 20));
  }
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

rchfsi_status rchfsi_rotate(rchfsi_handle h, double *Y_in_X_out, const double *E_colmajor) {
  if (!h) return RCHFSI_EINVAL;
  if (!Y_in_X_out || !E_colmajor || !aligned16(Y_in_X_out) || !aligned16(E_colmajor)) {
    h->err = "rchfsi_rotate: null or misaligned argument";
    return RCHFSI_EINVAL;
  }
  if (h->run.active) { h->err = "rchfsi_rotate: a step-wise filter is in progress"; return RCHFSI_EINVAL; }
  return rotate_in_place(h, Y_in_X_out, E_colmajor);
}

rchfsi_status rchfsi_rayleigh_ritz(rchfsi_handle h, double *Y_in_X_out, double *ritz_out, double *G_out,
                                   double *resnorm_out) {
  if (!h) return RCHFSI_EINVAL;
  if (!Y_in_X_out || !ritz_out || !aligned16(Y_in_X_out) || (G_out && !aligned16(G_out))) {
    h->err = "rchfsi_rayleigh_ritz: null or misaligned pointer";
    return RCHFSI_EINVAL;
  }
  const bool chunked = rr_wants_chunked(h);
  RCHFSI_TRY(rr_preallocate(h, chunked));      // ENOMEM, if any, before the block is touched
  if (chunked) return rayleigh_ritz_chunked(h, Y_in_X_out, ritz_out, G_out, RCHFSI_FP64, resnorm_out);
  return rayleigh_ritz_impl(h, Y_in_X_out, ritz_out, G_out, resnorm_out);
}

}  // extern "C"
