// Dense tensor-core step: one kernel per recurrence step computing
//   T = A_lp (x) W   on tcgen05 (kind::tf32 or kind::f16 with BF16 operands, FP32 accumulate in TMEM)
// with the Alg. 3 update  R_X <- a T + b R_Y + c' R_X + a G Lambda_Y fused as the
// epilogue, so the recurrence blocks cross HBM once per step.
//
// Tile orientation: the accumulator tile is D[128 block columns j][BN matrix rows i]:
//   MMA "A" operand = W^T tile, M = j (contiguous in memory)  -> MN-major, SWIZZLE_128B
//   MMA "B" operand = operator rows i, K contiguous           -> K-major,  SWIZZLE_128B
// so a TMEM lane is a block column and a TMEM column is a matrix row: a warp reading TMEM
// lane-wise touches 32 consecutive j of one row i, i.e. the epilogue's global loads and stores
// of R_Y, R_X, G are fully coalesced without staging through shared memory, and Lambda_Y[j] is
// a per-thread constant.
//
// Warp roles (256 threads): warp 0 = TMA producer, warp 1 = MMA issuer (one elected lane),
// warp 2 = TMEM allocator, warps 4-7 = epilogue (TMEM lane quarter = warp % 4).
#include "common.cuh"
#include "tc_common.cuh"

namespace rchfsi {

bool make_tmap_2d(CUtensorMap *out, const void *base, int elem_bytes, bool bf16, uint64_t rows, uint64_t cols,
                  uint64_t pitch_bytes, uint32_t box_cols, uint32_t box_rows, bool atom32) {
  typedef CUresult (*EncodeFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                               const cuuint64_t *, const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave,
                               CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
  static EncodeFn encode = nullptr;
  if (!encode) {
    void *fn = nullptr;
    cudaDriverEntryPointQueryResult qres;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres) != cudaSuccess || !fn) return false;
    encode = reinterpret_cast<EncodeFn>(fn);
  }
  cuuint64_t dims[2] = {cols, rows};
  cuuint64_t strides[1] = {pitch_bytes};
  cuuint32_t box[2] = {box_cols, box_rows};
  cuuint32_t estr[2] = {1, 1};
  CUtensorMapDataType dt = bf16 ? CU_TENSOR_MAP_DATA_TYPE_BFLOAT16
                                : (elem_bytes == 4 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT32 : CU_TENSOR_MAP_DATA_TYPE_UINT8);
  CUresult r = encode(out, dt, 2, const_cast<void *>(base), dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                      atom32 ? CU_TENSOR_MAP_SWIZZLE_128B_ATOM_32B : CU_TENSOR_MAP_SWIZZLE_128B,
                      CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  return r == CUDA_SUCCESS;
}

namespace {

using namespace tc;

struct DenseTcParams {
  StepCoef k;
  const void *RY;
  void *RX;
  const void *G;
  const double *LY;
  const double *dinv_out;
  void *Wnext;
  int64_t m;
  int32_t N;
  int32_t num_k_blocks;
};

template <int BN>
struct DenseCfg {
  static constexpr int W_BYTES = 16384;                 // 128 block columns x 128 B of K per stage
  static constexpr int A_BYTES = BN * 128;              // BN operator rows x 128 B of K per stage
  static constexpr int STAGE_BYTES = W_BYTES + A_BYTES;
  static constexpr int STAGES = (BN >= 256) ? 4 : (BN >= 128 ? 6 : 8);
  static constexpr int SMEM_BYTES = STAGES * STAGE_BYTES + 1024 /*align slack*/ + 256 /*barriers*/;
  static constexpr int TMEM_COLS = BN < 32 ? 32 : BN;
};

template <typename S>
__device__ __forceinline__ double ld_s(const S *p) { return (double)*p; }

// KIND 0: TF32 (FP32 bit patterns; W may be R_Y itself), KIND 1: BF16 operands.
template <int KIND, int BN, typename S>
__global__ void __launch_bounds__(256, 1) dense_tc_kernel(const __grid_constant__ CUtensorMap tmW,
                                                          const __grid_constant__ CUtensorMap tmA, DenseTcParams p) {
  using Cfg = DenseCfg<BN>;
  constexpr int KR = KIND == 0 ? 32 : 64;       // K extent of one stage (128 B per operator row)
  extern __shared__ uint8_t smem_raw[];
  uint8_t *smem = reinterpret_cast<uint8_t *>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  uint64_t *full_bar = reinterpret_cast<uint64_t *>(smem + Cfg::STAGES * Cfg::STAGE_BYTES);
  uint64_t *empty_bar = full_bar + Cfg::STAGES;
  uint64_t *accum_bar = empty_bar + Cfg::STAGES;
  uint32_t *tmem_slot = reinterpret_cast<uint32_t *>(accum_bar + 1);

  const int warp = threadIdx.x >> 5;
  const int lane = threadIdx.x & 31;
  const int j0 = blockIdx.x * 128;
  const int64_t i0 = (int64_t)blockIdx.y * BN;
  const int nkb = p.num_k_blocks;

  if (warp == 0 && lane == 0) {
    tma_prefetch_desc(&tmW);
    tma_prefetch_desc(&tmA);
    for (int s = 0; s < Cfg::STAGES; ++s) {
      mbar_init(full_bar + s, 1);
      mbar_init(empty_bar + s, 1);
    }
    mbar_init(accum_bar, 1);
    fence_barrier_init();
  }
  if (warp == 2) tmem_alloc(tmem_slot, Cfg::TMEM_COLS);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = *tmem_slot;

  if (warp == 0) {
    if (lane == 0) {
      for (int kb = 0; kb < nkb; ++kb) {
        const int s = kb % Cfg::STAGES;
        const uint32_t ph = (kb / Cfg::STAGES) & 1;
        mbar_wait(empty_bar + s, ph ^ 1);
        uint8_t *ws = smem + s * Cfg::STAGE_BYTES;
        uint8_t *as = ws + Cfg::W_BYTES;
        mbar_expect_tx(full_bar + s, Cfg::STAGE_BYTES);
        if constexpr (KIND == 0) {
#pragma unroll
          for (int a = 0; a < 4; ++a) tma_load_2d(ws + a * 4096, &tmW, full_bar + s, j0 + 32 * a, kb * KR);
        } else {
#pragma unroll
          for (int a = 0; a < 2; ++a) tma_load_2d(ws + a * 8192, &tmW, full_bar + s, j0 + 64 * a, kb * KR);
        }
        tma_load_2d(as, &tmA, full_bar + s, kb * KR, (int32_t)i0);
      }
    }
  } else if (warp == 1) {
    if (lane == 0) {
      constexpr uint32_t idesc = make_idesc(KIND == 0 ? 2 : 1, /*A MN-major*/ 1, /*B K-major*/ 0, 128, BN);
      for (int kb = 0; kb < nkb; ++kb) {
        const int s = kb % Cfg::STAGES;
        const uint32_t ph = (kb / Cfg::STAGES) & 1;
        mbar_wait(full_bar + s, ph);
        tc_fence_after();
        const uint32_t ws = smem_u32(smem + s * Cfg::STAGE_BYTES);
        const uint32_t as = ws + Cfg::W_BYTES;
#pragma unroll
        for (int q = 0; q < 4; ++q) {
          // W^T tile, MN-major.  TF32: SWIZZLE_128B_BASE32B, 8 k rows per MMA = two 4-row groups
          // (SBO 512 B), M atoms (32 columns) 4096 B apart.  BF16: SWIZZLE_128B, 16 k rows per MMA =
          // two 8-row groups (SBO 1024 B), M atoms (64 columns) 8192 B apart.
          const uint64_t da = (KIND == 0) ? make_smem_desc(ws + q * 1024, 4096, 512, 1)
                                          : make_smem_desc(ws + q * 2048, 8192, 1024, 2);
          // operator rows, K-major: 32 B of K per MMA inside the 128 B swizzled row, 8-row groups 1024 B apart
          const uint64_t db = make_smem_desc(as + q * 32, 16, 1024);
          umma<KIND>(tmem_base, da, db, idesc, (kb > 0 || q > 0) ? 1u : 0u);
        }
        umma_commit(empty_bar + s);
      }
      umma_commit(accum_bar);
    }
  } else if (warp >= 4) {
    const int q = warp & 3;
    const int j = j0 + 32 * q + lane;
    const bool jok = j < p.N;
    const S *RY = reinterpret_cast<const S *>(p.RY);
    S *RX = reinterpret_cast<S *>(p.RX);
    const S *G = reinterpret_cast<const S *>(p.G);
    const double ly = (G != nullptr && jok) ? p.LY[j] : 0.0;
    const double ka = p.k.a, kb_ = p.k.b, kc = p.k.cp;
    mbar_wait(accum_bar, 0);
    tc_fence_after();
#pragma unroll 1
    for (int c0 = 0; c0 < BN; c0 += 32) {
      uint32_t r[32];
      tmem_ld_32x32(tmem_base + ((uint32_t)(32 * q) << 16) + (uint32_t)c0, r);
      tmem_ld_wait();
      if (!jok) continue;
#pragma unroll
      for (int t = 0; t < 32; ++t) {
        const int64_t i = i0 + c0 + t;
        if (i < p.m) {
          const int64_t idx = i * p.N + j;
          double T = (double)__uint_as_float(r[t]);
          if (p.dinv_out) T *= p.dinv_out[i];
          double out = ka * T + kb_ * ld_s(RY + idx) + kc * ld_s(RX + idx);
          if (G) out += ka * (ld_s(G + idx) * ly);
          RX[idx] = (S)out;
          if (p.Wnext) {
            if constexpr (KIND == 0) {   // round to nearest TF32 here: the MMA itself truncates
              uint32_t u;
              asm("cvt.rna.tf32.f32 %0, %1;" : "=r"(u) : "f"((float)out));
              reinterpret_cast<uint32_t *>(p.Wnext)[idx] = u;
            }
            else
              reinterpret_cast<__nv_bfloat16 *>(p.Wnext)[idx] = __float2bfloat16_rn((float)out);
          }
        }
      }
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 2) {
    tc_fence_after();
    tmem_dealloc(tmem_base, Cfg::TMEM_COLS);
  }
}

// lowp[i][k] = round(A[i][k] * dinv[k]) in TF32 (RN, stored as FP32) or BF16; zero padding to ld
template <int KIND>
__global__ void dense_lowp_kernel(const double *__restrict__ A, int64_t lda, const double *__restrict__ dinv, void *out,
                                  int64_t m, int64_t ld) {
  const int64_t total = m * ld;
  for (int64_t t = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; t < total; t += (int64_t)gridDim.x * blockDim.x) {
    const int64_t i = t / ld, k = t - i * ld;
    double v = 0.0;
    if (k < m) {
      v = A[i * lda + k];
      if (dinv) v *= dinv[k];
    }
    if constexpr (KIND == 0) {
      float f = (float)v;
      uint32_t u;
      asm("cvt.rna.tf32.f32 %0, %1;" : "=r"(u) : "f"(f));
      reinterpret_cast<uint32_t *>(out)[t] = u;
    } else {
      reinterpret_cast<__nv_bfloat16 *>(out)[t] = __float2bfloat16_rn((float)v);
    }
  }
}

const LowpCopy *get_dense_copy(rchfsi_ctx *h, int prec, bool folded, rchfsi_status *st) {
  *st = RCHFSI_OK;
  for (const LowpCopy &c : h->lowp)
    if (c.prec == prec && c.folded == folded) return &c;
  LowpCopy c;
  c.prec = prec;
  c.folded = folded;
  c.ld = cdiv(h->m, 64) * 64;
  c.rows_pad = h->m;
  c.bytes = (size_t)h->m * c.ld * (prec == RCHFSI_BF16 ? 2 : 4);
  *st = dev_alloc(h, &c.data, c.bytes);
  if (*st != RCHFSI_OK) return nullptr;
  const unsigned grid = (unsigned)std::min<int64_t>(cdiv(h->m * c.ld, 256), 148 * 16);
  if (prec == RCHFSI_BF16)
    dense_lowp_kernel<1><<<grid, 256, 0, h->stream>>>(h->A.d.dense, h->A.d.lda, folded ? h->dinv : nullptr, c.data, h->m, c.ld);
  else
    dense_lowp_kernel<0><<<grid, 256, 0, h->stream>>>(h->A.d.dense, h->A.d.lda, folded ? h->dinv : nullptr, c.data, h->m, c.ld);
  h->launches++;
  h->lowp.push_back(c);
  return &h->lowp.back();
}

template <int KIND, int BN, typename S>
rchfsi_status launch_dense(rchfsi_ctx *h, const CUtensorMap &tmW, const CUtensorMap &tmA, const DenseTcParams &p) {
  using Cfg = DenseCfg<BN>;
  auto kern = dense_tc_kernel<KIND, BN, S>;
  RCHFSI_CUDA_CHECK(h, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, Cfg::SMEM_BYTES));
  dim3 grid((unsigned)cdiv(p.N, 128), (unsigned)cdiv(p.m, BN));
  kern<<<grid, 256, Cfg::SMEM_BYTES, h->stream>>>(tmW, tmA, p);
  LAUNCH_CHECK(h);
  return RCHFSI_OK;
}

template <int KIND, typename S>
rchfsi_status launch_dense_bn(rchfsi_ctx *h, int bn, const CUtensorMap &tmW, const CUtensorMap &tmA, const DenseTcParams &p) {
  if (bn == 256) return launch_dense<KIND, 256, S>(h, tmW, tmA, p);
  if (bn == 128) return launch_dense<KIND, 128, S>(h, tmW, tmA, p);
  return launch_dense<KIND, 64, S>(h, tmW, tmA, p);
}

}  // namespace

bool dense_tc_supported(const rchfsi_ctx *h) {
  if (h->A.d.kind != RCHFSI_OP_DENSE) return false;
  if (h->opt.apply_prec == RCHFSI_TF32) return h->N % 4 == 0;
  if (h->opt.apply_prec == RCHFSI_BF16) return h->N % 8 == 0;
  return false;
}

int dense_tc_pick_bn(int64_t m, int32_t N) {
  const int64_t tj = cdiv(N, 128);
  if (tj * cdiv(m, 256) >= 120) return 256;
  if (tj * cdiv(m, 128) >= 120) return 128;
  return 64;
}

rchfsi_status dense_tc_step(rchfsi_ctx *h, const FusedStep &s) {
  const bool bf16 = (s.apply_prec == RCHFSI_BF16);
  const bool folded = !s.chfsi && h->dinv != nullptr;
  rchfsi_status st;
  const LowpCopy *cp = get_dense_copy(h, bf16 ? RCHFSI_BF16 : RCHFSI_TF32, folded, &st);
  if (!cp) return st;
  const int eb = bf16 ? 2 : 4;
  const int bn = dense_tc_pick_bn(h->m, h->N);
  CUtensorMap tmW, tmA;
  // W [m][N]: box = 128 B of block columns x (32 | 64) k rows
  if (!make_tmap_2d(&tmW, s.W, eb, bf16, (uint64_t)h->m, (uint64_t)h->N, (uint64_t)h->N * eb, bf16 ? 64 : 32, bf16 ? 64 : 32, !bf16) ||
      !make_tmap_2d(&tmA, cp->data, eb, bf16, (uint64_t)h->m, (uint64_t)cp->ld, (uint64_t)cp->ld * eb, bf16 ? 64 : 32, (uint32_t)bn)) {
    h->err = "cuTensorMapEncodeTiled failed";
    return RCHFSI_ECUDA;
  }
  DenseTcParams p{s.k, s.RY, s.RX, s.G, s.LY, s.chfsi ? h->dinv : nullptr, s.Wnext, h->m, h->N,
                  (int32_t)cdiv(h->m, bf16 ? 64 : 32)};
  if (s.store_prec == RCHFSI_FP64)
    return bf16 ? launch_dense_bn<1, double>(h, bn, tmW, tmA, p) : launch_dense_bn<0, double>(h, bn, tmW, tmA, p);
  return bf16 ? launch_dense_bn<1, float>(h, bn, tmW, tmA, p) : launch_dense_bn<0, float>(h, bn, tmW, tmA, p);
}

}  // namespace rchfsi
