// rchfsi_filter / rchfsi_filter_host / rchfsi_solve: host control flow of Algorithm 2
// (PAPER.md:78-86), Algorithm 3 and Algorithm 1.
#include <algorithm>
#include <cmath>
#include <cstdlib>
#include "common.cuh"

using namespace rchfsi;

namespace rchfsi {

Plan make_plan(const rchfsi_operator &A, int32_t N, const rchfsi_options &opt, const Knobs &kn) {
  Plan p{};
  p.store = opt.store_prec;
  const int ap = opt.apply_prec;
  p.fused = 0;
  if (ap == RCHFSI_FP64) {
    p.operand = RCHFSI_FP64;
  } else {
    p.operand = RCHFSI_FP32;
    if (opt.noise_eps <= 0) {
      if (A.kind == RCHFSI_OP_CSR && csr_fused_supported(A, N, opt)) p.fused = 1;
      if (A.kind == RCHFSI_OP_DENSE && ap != RCHFSI_FP32 && dense_tc_supported(A, N, opt)) p.fused = 2;
      if (A.kind == RCHFSI_OP_FE && ap != RCHFSI_FP32 && fe_tc_supported(A, N, opt)) p.fused = 3;
    }
    if (p.fused >= 2 && ap == RCHFSI_BF16) p.operand = RCHFSI_BF16;
    if (p.fused == 1) p.operand = p.store;   // the CSR kernel reads R_Y itself, converting on the fly
  }
  p.tprec = (ap == RCHFSI_FP64) ? RCHFSI_FP64 : RCHFSI_FP32;
  p.shadow = (p.operand != p.store);
  p.panel = (p.fused == 3);
  // FE step: the (cell, column tile) CTA that is the LAST toucher of a node writes the shadow row of the finished
  // R_X value.  Every CTA that gathers that row for the same column tile belongs to a cell containing the node,
  // i.e. to an earlier colour launch (complete, stream order) or to the writing CTA itself, whose gather ends
  // before its epilogue starts: the new shadow may overwrite the old one, one buffer instead of two
  // (14.8 GB instead of 29.6 GB of BF16 shadows at config 5).  The dense step cannot: its row tiles read all rows.
  // RCHFSI_FE_SHADOW_PAIR=1 keeps the two-buffer scheme (the tests compare the two bit for bit).
  p.shadow_inplace = p.shadow && p.fused == 3 && !kn.fe_shadow_pair;
  return p;
}

}  // namespace rchfsi

namespace {

Plan make_plan(const rchfsi_ctx *h) { return rchfsi::make_plan(h->A.d, h->N, h->opt, h->knobs); }

rchfsi_status ensure_filter_workspace(rchfsi_ctx *h, const Plan &pl, int32_t degree, bool need_gs) {
  // sized for the block width of rchfsi_create (N_cap), whatever the active width of this call
  const size_t el = (size_t)h->m * (pl.panel ? (size_t)cdiv(h->N_cap, 128) * 128 : (size_t)h->N_cap);
  if (!h->RX) { RCHFSI_TRY(dev_alloc(h, &h->RX, el * prec_bytes(pl.store))); h->RX_bytes = el * prec_bytes(pl.store); }
  if (!h->RY) { RCHFSI_TRY(dev_alloc(h, &h->RY, el * prec_bytes(pl.store))); h->RY_bytes = el * prec_bytes(pl.store); }
  if (pl.shadow) {
    const size_t wb = el * (pl.operand == RCHFSI_BF16 ? 2 : 4);
    if (!h->Wa) { RCHFSI_TRY(dev_alloc(h, &h->Wa, wb)); h->Wa_bytes = wb; }
    if (!pl.shadow_inplace && !h->Wb) RCHFSI_TRY(dev_alloc(h, &h->Wb, wb));
  }
  if (pl.fused == 0 && !h->T) RCHFSI_TRY(dev_alloc(h, &h->T, el * prec_bytes(pl.tprec)));
  if (need_gs && !h->Gs) RCHFSI_TRY(dev_alloc(h, &h->Gs, el * prec_bytes(pl.store)));
  if (!h->lam_table || h->lam_table_p < degree) {
    RCHFSI_TRY(dev_alloc(h, (void **)&h->lam_table, sizeof(double) * (size_t)(degree + 1) * h->N_cap));
    h->lam_table_p = degree;
  }
  if (!h->colnorm) RCHFSI_TRY(dev_alloc(h, (void **)&h->colnorm, sizeof(double) * 2 * h->N_cap));
  return RCHFSI_OK;
}

// One operator apply + recurrence update, fused when a fused kernel exists for this plan.
rchfsi_status do_step(rchfsi_ctx *h, const Plan &pl, bool chfsi, const StepCoef &k, const void *W,
                      const void *RY, void *RX, const void *G, const double *LY, void *Wnext,
                      uint64_t apply_index, bool g_rowmajor = false) {
  if (pl.fused) {
    FusedStep s{k, W, RY, RX, G, LY, Wnext, h->opt.apply_prec, pl.store, chfsi,
                /*g_rowmajor=*/pl.panel && g_rowmajor && G != nullptr};
    if (pl.fused == 1) return csr_fused_step(h, s);
    if (pl.fused == 2) return dense_tc_step(h, s);
    return fe_tc_step(h, s);
  }
  const double *dinv_in = chfsi ? nullptr : h->dinv;
  if (pl.tprec == RCHFSI_FP64)
    RCHFSI_TRY(op_apply_simt<double>(h, h->A.d, dinv_in, (const double *)W, (double *)h->T, h->N));
  else
    RCHFSI_TRY(op_apply_simt<float>(h, h->A.d, dinv_in, (const float *)W, (float *)h->T, h->N));
  if (h->opt.noise_eps > 0)
    RCHFSI_TRY(add_column_noise(h, pl.tprec, h->T, h->m, h->N, h->opt.noise_eps, h->opt.noise_seed,
                                apply_index, h->colnorm));
  StepArgs a{k, h->T, RY, RX, G, LY, chfsi ? h->dinv : nullptr, Wnext, h->m, h->N};
  return step_elementwise(h, pl.store, pl.tprec, pl.operand, a);
}

}  // namespace

// G_arg points to FP64 values, or to FP32 values when g_is_f32 (caller's g_input_f32 option, or the FP32
// residual block rchfsi_solve keeps in its memory-light mode).  Validation, workspace, scalars, Lambda table and the
// initial blocks: everything of Alg. 2 / Alg. 3 before the loop.
static rchfsi_status filter_begin(rchfsi_handle h, int32_t method, double *X, const double *ritz, const void *G_arg,
                                  bool g_is_f32, int32_t degree, double lam_min, double lam_T, double lam_max) {
  const double *G = reinterpret_cast<const double *>(G_arg);
  if (!h) return RCHFSI_EINVAL;
  h->run.active = false;
  if (!X || (reinterpret_cast<uintptr_t>(X) & 15u)) { h->err = "rchfsi_filter: X null or misaligned"; return RCHFSI_EINVAL; }
  if (method != RCHFSI_METHOD_CHFSI && method != RCHFSI_METHOD_RCHFSI) { h->err = "rchfsi_filter: unknown method"; return RCHFSI_EINVAL; }
  if (method == RCHFSI_METHOD_RCHFSI && !ritz) { h->err = "rchfsi_filter: ritz is required for R-ChFSI"; return RCHFSI_EINVAL; }
  if (G && (reinterpret_cast<uintptr_t>(G) & 15u)) { h->err = "rchfsi_filter: G misaligned"; return RCHFSI_EINVAL; }
  if (degree < 1) { h->err = "rchfsi_filter: degree < 1"; return RCHFSI_EINVAL; }
  if (degree >= 100 && h->opt.apply_prec != RCHFSI_FP64 && !h->opt.allow_high_degree) {
    // PAPER.md:347-359 and footnote 5: FP32 / TF32 R-ChFSI matches FP64 for p <= 80, not for p = 100, 120
    h->err = "rchfsi_filter: degree >= 100 with a reduced-precision apply is unstable (PAPER.md:347-359); set allow_high_degree to force it";
    return RCHFSI_EINVAL;
  }
  if (!(lam_min < lam_T) || !(lam_T < lam_max) || !std::isfinite(lam_min) || !std::isfinite(lam_max)) {
    h->err = "rchfsi_filter: need lam_min < lam_T < lam_max";
    return RCHFSI_EINVAL;
  }
  FilterRun &r = h->run;
  r = FilterRun{};
  r.chfsi = (method == RCHFSI_METHOD_CHFSI);
  r.pl = make_plan(h);
  const Plan &pl = r.pl;
  const int64_t m = h->m;
  const int32_t N = h->N;
  const size_t el = (size_t)m * N;
  cudaStream_t st = h->stream;
  // FP32 residual block from the caller (g_input_f32): used in place, never copied (config 5 memory plan)
  r.gf32 = !r.chfsi && g_is_f32;
  if (r.gf32 && (!G || pl.store != RCHFSI_FP32)) {
    h->err = "rchfsi_filter: g_input_f32 needs a non-NULL G and store_prec FP32";
    return RCHFSI_EINVAL;
  }
  const bool need_gs = !r.chfsi && !r.gf32 && (pl.store != RCHFSI_FP64 || pl.panel);
  const int64_t pm = pl.panel ? m : 0;
  const size_t el_lib = pl.panel ? (size_t)m * (size_t)cdiv(N, 128) * 128 : el;
  RCHFSI_TRY(ensure_filter_workspace(h, pl, degree, need_gs));

  // first line of Alg. 2 / Alg. 3
  r.e = (lam_max - lam_T) / 2.0;
  r.c = (lam_max + lam_T) / 2.0;
  r.sigma1 = r.e / (lam_min - r.c);
  r.gamma = 2.0 / r.sigma1;
  r.sigma = r.sigma1;
  r.X = X;
  r.degree = degree;
  r.RX = h->RX;
  r.RY = h->RY;
  r.Wcur = pl.shadow ? h->Wa : nullptr;
  r.Wnext = pl.shadow ? (pl.shadow_inplace ? h->Wa : h->Wb) : nullptr;
  const double e = r.e, c = r.c, sigma1 = r.sigma1;

  if (!r.chfsi) {
    // G = A X - B X Lambda with the exact operators (reading S5) when the caller has none
    if (!G) {
      const size_t el_cap = (size_t)m * h->N_cap;
      if (!h->Gtmp) RCHFSI_TRY(dev_alloc(h, (void **)&h->Gtmp, el_cap * 8));
      if (!h->rr1) RCHFSI_TRY(dev_alloc(h, (void **)&h->rr1, el_cap * 8));
      RCHFSI_TRY(op_apply_simt<double>(h, h->A.d, nullptr, X, h->rr1, N));
      const double *BX = X;
      if (h->B.present) {
        RCHFSI_TRY(op_apply_simt<double>(h, h->B.d, nullptr, X, h->Gtmp, N));
        BX = h->Gtmp;
      }
      RCHFSI_TRY(residual_block(h, h->rr1, BX, ritz, h->Gtmp, nullptr, m, N));
      G = h->Gtmp;
    }
    RCHFSI_TRY(lambda_table(h, ritz, N, degree, e, c, sigma1, h->lam_table));
    RCHFSI_CUDA_CHECK(h, cudaMemsetAsync(r.RX, 0, el_lib * prec_bytes(pl.store), st));     // R_X <- 0
    RCHFSI_TRY(scale_convert(h, pl.store, pl.operand, sigma1 / e, G, r.RY, r.Wcur, m, N, pm,
                             r.gf32 ? RCHFSI_FP32 : RCHFSI_FP64));                        // R_Y <- (sigma_1/e) G
    if (need_gs) {
      RCHFSI_TRY(scale_convert(h, pl.store, 0, 1.0, G, h->Gs, nullptr, m, N, pm));
      r.Gst = h->Gs;
      r.g_lib = true;
    } else {
      r.Gst = G;
    }
  } else {
    // Alg. 2: X_k = X, Y = (sigma_1/e)(D^-1 A (x) X - c X)
    RCHFSI_TRY(scale_convert(h, pl.store, pl.operand, 1.0, X, r.RX, r.Wcur, m, N, pm));
    const void *W0 = pl.shadow ? r.Wcur : r.RX;
    if (pl.fused) {
      // first step through the fused kernels: RY <- a T + b X with a = sigma_1/e, b = -a c, c' = 0
      RCHFSI_CUDA_CHECK(h, cudaMemsetAsync(r.RY, 0, el_lib * prec_bytes(pl.store), st));
      StepCoef k0{sigma1 / e, -(sigma1 / e) * c, 0.0};
      RCHFSI_TRY(do_step(h, pl, true, k0, W0, r.RX, r.RY, nullptr, nullptr, r.Wnext, r.apply_index++));
    } else {
      if (pl.tprec == RCHFSI_FP64)
        RCHFSI_TRY(op_apply_simt<double>(h, h->A.d, nullptr, (const double *)W0, (double *)h->T, N));
      else
        RCHFSI_TRY(op_apply_simt<float>(h, h->A.d, nullptr, (const float *)W0, (float *)h->T, N));
      if (h->opt.noise_eps > 0)
        RCHFSI_TRY(add_column_noise(h, pl.tprec, h->T, m, N, h->opt.noise_eps, h->opt.noise_seed, r.apply_index, h->colnorm));
      r.apply_index++;
      RCHFSI_TRY(chfsi_first(h, pl.store, pl.tprec, pl.operand, sigma1 / e, c, h->T, h->dinv, X, r.RY, r.Wnext, m, N));
    }
    if (pl.shadow) std::swap(r.Wcur, r.Wnext);
  }
  r.k = 2;
  r.active = true;
  return RCHFSI_OK;
}

// One pass of the loop body of Alg. 2 / Alg. 3: the fused operator + recurrence step k, then swap(R_X, R_Y).
static rchfsi_status filter_step(rchfsi_handle h) {
  FilterRun &r = h->run;
  if (!r.active || r.k > r.degree) { h->err = "rchfsi_filter_step: no step left (call rchfsi_filter_begin first)"; return RCHFSI_EINVAL; }
  const int32_t N = h->N;
  const double sigma2 = 1.0 / (r.gamma - r.sigma);
  StepCoef kc{2.0 * sigma2 / r.e, -2.0 * sigma2 * r.c / r.e, -r.sigma * sigma2};
  const double *LY = r.chfsi ? nullptr : h->lam_table + (size_t)(r.k - 1) * N;
  const void *W = r.pl.shadow ? r.Wcur : r.RY;
  RCHFSI_TRY(do_step(h, r.pl, r.chfsi, kc, W, r.RY, r.RX, r.chfsi ? nullptr : r.Gst, LY, r.Wnext, r.apply_index++, r.gf32));
  std::swap(r.RX, r.RY);                       // swap(R_X, R_Y)
  if (r.pl.shadow) std::swap(r.Wcur, r.Wnext);
  r.sigma = sigma2;
  r.last = kc;
  r.last_LY = LY;
  r.k++;
  return RCHFSI_OK;
}

// Last line of Alg. 3, Y_p = D^-1 R_Y + X Lambda_Y; Alg. 2: the block itself.
static rchfsi_status filter_end(rchfsi_handle h) {
  FilterRun &r = h->run;
  if (!r.active || r.k <= r.degree) { h->err = "rchfsi_filter_end: steps are left (or no filter was begun)"; return RCHFSI_EINVAL; }
  const int64_t m = h->m;
  const int32_t N = h->N;
  const int64_t pm = r.pl.panel ? m : 0;
  r.active = false;
  if (h->x_pending) {   // rchfsi_filter_host: X is still arriving on the copy stream
    h->x_pending = false;
    RCHFSI_CUDA_CHECK(h, cudaStreamWaitEvent(h->stream, h->ev_x, 0));
  }
  if (!r.chfsi)
    return finish_block(h, r.pl.store, r.RY, h->dinv, h->lam_table + (size_t)r.degree * N, r.X, m, N, pm);
  return finish_block(h, r.pl.store, r.RY, nullptr, nullptr, r.X, m, N, pm);
}

static rchfsi_status filter_impl(rchfsi_handle h, int32_t method, double *X, const double *ritz, const void *G_arg,
                                 bool g_is_f32, int32_t degree, double lam_min, double lam_T, double lam_max) {
  RCHFSI_TRY(filter_begin(h, method, X, ritz, G_arg, g_is_f32, degree, lam_min, lam_T, lam_max));
  RCHFSI_CUDA_CHECK(h, cudaEventRecord(h->ev_step0, h->stream));
  for (int32_t k = 2; k <= degree; ++k) RCHFSI_TRY(filter_step(h));
  RCHFSI_CUDA_CHECK(h, cudaEventRecord(h->ev_step1, h->stream));
  h->last_steps = degree - 1;
  return filter_end(h);
}

extern "C" {

rchfsi_status rchfsi_filter(rchfsi_handle h, int32_t method, double *X, const double *ritz, const double *G,
                            int32_t degree, double lam_min, double lam_T, double lam_max) {
  if (!h) return RCHFSI_EINVAL;
  return filter_impl(h, method, X, ritz, G, h->opt.g_input_f32 != 0, degree, lam_min, lam_T, lam_max);
}

rchfsi_status rchfsi_filter_begin(rchfsi_handle h, int32_t method, double *X, const double *ritz, const double *G,
                                  int32_t degree, double lam_min, double lam_T, double lam_max) {
  if (!h) return RCHFSI_EINVAL;
  return filter_begin(h, method, X, ritz, G, h->opt.g_input_f32 != 0, degree, lam_min, lam_T, lam_max);
}
rchfsi_status rchfsi_filter_step(rchfsi_handle h) { return h ? filter_step(h) : RCHFSI_EINVAL; }
rchfsi_status rchfsi_filter_end(rchfsi_handle h) { return h ? filter_end(h) : RCHFSI_EINVAL; }
int32_t rchfsi_filter_steps_left(rchfsi_handle h) { return (h && h->run.active) ? h->run.degree - h->run.k + 1 : 0; }

// Column-chunked host pipeline.  The columns of the block are independent through the whole filter (Alg. 3 touches
// column j only through eps_j and Lambda_k[j]), so the block is cut into column chunks and chunk
// i+1 is uploaded while chunk i is filtered and chunk i-1 is downloaded: three streams, three staging sets.
static int32_t host_chunk_width(const rchfsi_ctx *h) {
  const int32_t N = h->N_cap;
  if (h->knobs.host_chunk >= 128) return std::min<int32_t>((int32_t)cdiv(h->knobs.host_chunk, 128) * 128, N);   // test knob
  const double blk = 8.0 * (double)h->m * N;
  if (blk < 256e6 || N < 256) return N;               // small blocks: one chunk (the X upload still overlaps the steps)
  int32_t w = (int32_t)cdiv(cdiv(N, 6), 128) * 128;   // about six chunks, whole 128-column tiles
  return std::min(w, N);
}

rchfsi_status rchfsi_filter_host(rchfsi_handle h, int32_t method, double *X_host, const double *ritz_host,
                                 const double *G_host, int32_t degree, double lam_min, double lam_T,
                                 double lam_max) {
  if (!h) return RCHFSI_EINVAL;
  if (!X_host || (method == RCHFSI_METHOD_RCHFSI && !ritz_host)) { h->err = "rchfsi_filter_host: null argument"; return RCHFSI_EINVAL; }
  if (h->N != h->N_cap) { h->err = "rchfsi_filter_host: handle is inside another call"; return RCHFSI_EINVAL; }
  const int64_t m = h->m;
  const int32_t N = h->N_cap;
  const bool gf32 = h->opt.g_input_f32 != 0;
  const size_t gb = gf32 ? 4 : 8;                       // bytes per element of G_host (FP32 with g_input_f32)
  cudaStream_t st = h->stream;
  const int32_t w = host_chunk_width(h);
  const int nchunks = (int)cdiv(N, w);
  const int nsets = std::min<int>(rchfsi_ctx::HOST_SETS, nchunks);
  // (each buffer, event and stream has its own guard: the call may be repeated after the caller added workspace)
  for (int i = 0; i < nsets; ++i) {
    if (!h->hX[i]) RCHFSI_TRY(dev_alloc(h, (void **)&h->hX[i], sizeof(double) * (size_t)m * w));
    if (!h->ev_g[i]) RCHFSI_CUDA_CHECK(h, cudaEventCreateWithFlags(&h->ev_g[i], cudaEventDisableTiming));
    if (!h->ev_xin[i]) RCHFSI_CUDA_CHECK(h, cudaEventCreateWithFlags(&h->ev_xin[i], cudaEventDisableTiming));
    if (!h->ev_done[i]) RCHFSI_CUDA_CHECK(h, cudaEventCreateWithFlags(&h->ev_done[i], cudaEventDisableTiming));
    if (!h->ev_free[i]) RCHFSI_CUDA_CHECK(h, cudaEventCreateWithFlags(&h->ev_free[i], cudaEventDisableTiming));
  }
  if (!h->hritz) RCHFSI_TRY(dev_alloc(h, (void **)&h->hritz, sizeof(double) * N));
  if (!h->in_stream) RCHFSI_CUDA_CHECK(h, cudaStreamCreateWithFlags(&h->in_stream, cudaStreamNonBlocking));
  if (!h->out_stream) RCHFSI_CUDA_CHECK(h, cudaStreamCreateWithFlags(&h->out_stream, cudaStreamNonBlocking));
  h->host_chunk = w;
  if (G_host)
    for (int i = 0; i < nsets; ++i)
      if (!h->hG[i]) RCHFSI_TRY(dev_alloc(h, &h->hG[i], gb * (size_t)m * w));
  if (ritz_host) RCHFSI_CUDA_CHECK(h, cudaMemcpyAsync(h->hritz, ritz_host, sizeof(double) * N, cudaMemcpyHostToDevice, st));
  // everything enqueued earlier on the main stream (previous calls reading the staging sets) is ordered first
  RCHFSI_CUDA_CHECK(h, cudaEventRecord(h->ev_free[0], st));
  RCHFSI_CUDA_CHECK(h, cudaStreamWaitEvent(h->in_stream, h->ev_free[0], 0));
  RCHFSI_CUDA_CHECK(h, cudaStreamWaitEvent(h->out_stream, h->ev_free[0], 0));
  rchfsi_status result = RCHFSI_OK;
  for (int c = 0; c < nchunks && result == RCHFSI_OK; ++c) {
    const int b = c % nsets;
    const int32_t j0 = c * w, wc = std::min<int32_t>(w, N - j0);
    // ---- upload (in_stream): G first, it is what the recurrence needs; X is read only by the last line
    if (c >= nsets) RCHFSI_CUDA_CHECK(h, cudaStreamWaitEvent(h->in_stream, h->ev_free[b], 0));
    if (G_host)
      RCHFSI_CUDA_CHECK(h, cudaMemcpy2DAsync(h->hG[b], gb * wc, reinterpret_cast<const char *>(G_host) + gb * j0, gb * N,
                                             gb * wc, (size_t)m, cudaMemcpyHostToDevice, h->in_stream));
    RCHFSI_CUDA_CHECK(h, cudaEventRecord(h->ev_g[b], h->in_stream));
    RCHFSI_CUDA_CHECK(h, cudaMemcpy2DAsync(h->hX[b], sizeof(double) * wc, X_host + j0, sizeof(double) * N,
                                           sizeof(double) * wc, (size_t)m, cudaMemcpyHostToDevice, h->in_stream));
    RCHFSI_CUDA_CHECK(h, cudaEventRecord(h->ev_xin[b], h->in_stream));
    // ---- filter the chunk (main stream) as a block of width wc
    RCHFSI_CUDA_CHECK(h, cudaStreamWaitEvent(st, h->ev_g[b], 0));
    const bool late_x = (method == RCHFSI_METHOD_RCHFSI) && G_host != nullptr;
    if (late_x) {
      h->ev_x = h->ev_xin[b];
      h->x_pending = true;
    } else {
      RCHFSI_CUDA_CHECK(h, cudaStreamWaitEvent(st, h->ev_xin[b], 0));
    }
    h->N = wc;
    result = filter_impl(h, method, h->hX[b], ritz_host ? h->hritz + j0 : nullptr, G_host ? h->hG[b] : nullptr, gf32,
                         degree, lam_min, lam_T, lam_max);
    h->N = N;
    if (h->x_pending) {   // the filter returned before its last line (invalid arguments)
      h->x_pending = false;
      cudaStreamSynchronize(h->in_stream);
    }
    if (result != RCHFSI_OK) break;
    RCHFSI_CUDA_CHECK(h, cudaEventRecord(h->ev_done[b], st));
    // ---- download (out_stream)
    RCHFSI_CUDA_CHECK(h, cudaStreamWaitEvent(h->out_stream, h->ev_done[b], 0));
    RCHFSI_CUDA_CHECK(h, cudaMemcpy2DAsync(X_host + j0, sizeof(double) * N, h->hX[b], sizeof(double) * wc,
                                           sizeof(double) * wc, (size_t)m, cudaMemcpyDeviceToHost, h->out_stream));
    RCHFSI_CUDA_CHECK(h, cudaEventRecord(h->ev_free[b], h->out_stream));
  }
  cudaStreamSynchronize(h->in_stream);
  cudaStreamSynchronize(h->out_stream);
  RCHFSI_CUDA_CHECK(h, cudaStreamSynchronize(st));
  return result;
}

rchfsi_status rchfsi_solve(rchfsi_handle h, int32_t method, double *X, int32_t n_wanted, int32_t degree,
                           double lam_min, double lam_T, double lam_max, double tol, int32_t max_iter,
                           double *evals_out, double *resnorm_out, int32_t *iters_out, double *history_out) {
  if (!h) return RCHFSI_EINVAL;
  if (!X || !evals_out || !resnorm_out || !iters_out) { h->err = "rchfsi_solve: null argument"; return RCHFSI_EINVAL; }
  if (n_wanted < 1 || n_wanted > h->N || max_iter < 1 || degree < 1 || !(tol > 0)) { h->err = "rchfsi_solve: bad n_wanted / max_iter / degree / tol"; return RCHFSI_EINVAL; }
  if (!(lam_min < lam_T) || !(lam_T < lam_max)) { h->err = "rchfsi_solve: need lam_min < lam_T < lam_max"; return RCHFSI_EINVAL; }
  const int32_t N = h->N;
  const size_t el = (size_t)h->m * N;
  cudaStream_t st = h->stream;
  const bool rch = (method == RCHFSI_METHOD_RCHFSI);
  // Memory-light mode when three more FP64 blocks do not fit (config 5): chunked Rayleigh-Ritz, and with FP32
  // recurrence storage the residual block G is kept in FP32 (SURVEY 8(d) memory plan) and read in place.
  const bool chunked = rr_wants_chunked(h);
  const bool g32 = chunked && rch && h->opt.store_prec == RCHFSI_FP32;
  void *Gbuf = nullptr;
  if (rch) {
    if (g32) {
      if (!h->Gsolve32) RCHFSI_TRY(dev_alloc(h, (void **)&h->Gsolve32, el * 4));
      Gbuf = h->Gsolve32;
    } else {
      if (!h->Gtmp) RCHFSI_TRY(dev_alloc(h, (void **)&h->Gtmp, el * 8));
      Gbuf = h->Gtmp;
    }
  }
  {
    // the filter's workspace first: the chunked Rayleigh-Ritz sizes its chunks from the memory that is left
    const Plan pl = make_plan(h);
    const bool chf = (method == RCHFSI_METHOD_CHFSI);
    RCHFSI_TRY(ensure_filter_workspace(h, pl, degree, !chf && !g32 && (pl.store != RCHFSI_FP64 || pl.panel)));
    // ... and everything else a filter or a Rayleigh-Ritz of this solve will allocate (reduced-precision operator
    // copies, chunk buffers, FE apply scratch, the INT8 products' buffers): nothing is computed on X before the
    // workspace is known to suffice, so an ENOMEM call can be repeated with X untouched
    if (pl.fused == 1) RCHFSI_TRY(csr_fused_prepare(h, chf));
    if (pl.fused == 2) RCHFSI_TRY(dense_tc_prepare(h, h->opt.apply_prec, chf));
    if (pl.fused == 3) RCHFSI_TRY(fe_tc_prepare(h, h->opt.apply_prec, chf));
    RCHFSI_TRY(rr_preallocate(h, chunked));
  }
  auto do_rr = [&]() -> rchfsi_status {
    if (chunked) return rayleigh_ritz_chunked(h, X, h->ritz_dev, Gbuf, g32 ? RCHFSI_FP32 : RCHFSI_FP64, h->res_dev);
    return rayleigh_ritz_impl(h, X, h->ritz_dev, (double *)Gbuf, h->res_dev);
  };
  std::vector<double> ritz(N), res(N);
  // reading S2: one Rayleigh-Ritz on the initial guess gives B-orthonormal X, Lambda and G
  RCHFSI_TRY(do_rr());
  rchfsi_status result = RCHFSI_ENOTCONVERGED;
  int32_t it = 0;
  for (it = 1; it <= max_iter; ++it) {
    if (h->opt.adaptive_bounds) {             // reading S7
      RCHFSI_CUDA_CHECK(h, cudaMemcpyAsync(ritz.data(), h->ritz_dev, sizeof(double) * N, cudaMemcpyDeviceToHost, st));
      RCHFSI_CUDA_CHECK(h, cudaStreamSynchronize(st));
      if (ritz[0] < ritz[N - 1] && ritz[N - 1] < lam_max) { lam_min = ritz[0]; lam_T = ritz[N - 1]; }
    }
    RCHFSI_TRY(filter_impl(h, method, X, h->ritz_dev, Gbuf, g32, degree, lam_min, lam_T, lam_max));
    RCHFSI_TRY(do_rr());
    RCHFSI_CUDA_CHECK(h, cudaMemcpyAsync(res.data(), h->res_dev, sizeof(double) * N, cudaMemcpyDeviceToHost, st));
    RCHFSI_CUDA_CHECK(h, cudaStreamSynchronize(st));
    double worst = 0.0;
    for (int j = 0; j < n_wanted; ++j) worst = std::fmax(worst, res[j]);
    if (history_out) history_out[it - 1] = worst;
    if (!(worst == worst)) { h->err = "rchfsi_solve: residual is NaN"; result = RCHFSI_EBREAKDOWN; break; }
    if (worst < tol) { result = RCHFSI_OK; break; }
  }
  if (it > max_iter) it = max_iter;
  RCHFSI_CUDA_CHECK(h, cudaMemcpyAsync(ritz.data(), h->ritz_dev, sizeof(double) * N, cudaMemcpyDeviceToHost, st));
  RCHFSI_CUDA_CHECK(h, cudaMemcpyAsync(res.data(), h->res_dev, sizeof(double) * N, cudaMemcpyDeviceToHost, st));
  RCHFSI_CUDA_CHECK(h, cudaStreamSynchronize(st));
  for (int j = 0; j < N; ++j) { evals_out[j] = ritz[j]; resnorm_out[j] = res[j]; }
  *iters_out = it;
  if (result == RCHFSI_ENOTCONVERGED) h->err = "rchfsi_solve: max_iter reached";
  return result;
}

}  // extern "C"
