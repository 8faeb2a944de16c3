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
#include <cstdlib>
#include "common.cuh"
#include "tc_common.cuh"

namespace rchfsi {

bool make_tmap_2d(CUtensorMap *out, const void *base, int elem_bytes, bool bf16, uint64_t rows, uint64_t cols,
                  uint64_t pitch_bytes, uint32_t box_cols, uint32_t box_rows, int atom32) {
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
                                : (elem_bytes == 4 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT32
                                                   : (elem_bytes == 8 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT64 : CU_TENSOR_MAP_DATA_TYPE_UINT8));
  CUresult r = encode(out, dt, 2, const_cast<void *>(base), dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                      atom32 == 2 ? CU_TENSOR_MAP_SWIZZLE_NONE
                                  : (atom32 == 1 ? CU_TENSOR_MAP_SWIZZLE_128B_ATOM_32B : CU_TENSOR_MAP_SWIZZLE_128B),
                      CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  return r == CUDA_SUCCESS;
}

bool get_tmap_2d(rchfsi_ctx *h, CUtensorMap *out, const void *base, int elem_bytes, bool bf16, uint64_t rows, uint64_t cols,
                 uint64_t pitch_bytes, uint32_t box_cols, uint32_t box_rows, int atom32) {
  for (const TmapEntry &e : h->tmaps)
    if (e.base == base && e.rows == rows && e.cols == cols && e.pitch == pitch_bytes && e.box_cols == box_cols &&
        e.box_rows == box_rows && e.elem_bytes == elem_bytes && e.bf16 == (int)bf16 && e.atom32 == (int)atom32) {
      *out = e.map;
      return true;
    }
  TmapEntry e{base, rows, cols, pitch_bytes, box_cols, box_rows, elem_bytes, (int)bf16, (int)atom32, {}};
  if (!make_tmap_2d(&e.map, base, elem_bytes, bf16, rows, cols, pitch_bytes, box_cols, box_rows, atom32)) return false;
  if (h->tmaps.size() >= 64) h->tmaps.erase(h->tmaps.begin());   // callers hold copies, never pointers into the cache
  h->tmaps.push_back(e);
  *out = e.map;
  return true;
}

rchfsi_status ensure_func_smem(rchfsi_ctx *h, const void *func, int bytes) {
  auto it = h->func_smem.find(func);
  if (it != h->func_smem.end() && it->second >= bytes) return RCHFSI_OK;
  RCHFSI_CUDA_CHECK(h, cudaFuncSetAttribute(func, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes));
  h->func_smem[func] = bytes;
  return RCHFSI_OK;
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
  int32_t ksplit;       // K splits = cluster size along z (1, 2, 4 or 8)
  int32_t mcast;        // 1: the two column tiles of a cluster (cluster x = 2) share the operator tile by TMA multicast
  int32_t debug_mode;   // 0 normal; 1 = no MMA (TMA throughput); 2 = no TMA (MMA throughput): timing probes only
};

template <int BN>
struct DenseCfg {
  static constexpr int KP = 2;                          // 128-byte K panels per pipeline stage
  static constexpr int W_BYTES = 16384;                 // 128 block columns x 128 B of K per panel
  static constexpr int A_BYTES = BN * 128;              // BN operator rows x 128 B of K per panel
  static constexpr int PANEL_BYTES = W_BYTES + A_BYTES;
  static constexpr int STAGE_BYTES = KP * PANEL_BYTES;
  static constexpr int STAGES = (200 * 1024) / STAGE_BYTES < 8 ? (200 * 1024) / STAGE_BYTES : 8;
  static constexpr int SMEM_BYTES = STAGES * STAGE_BYTES + 1024 /*align slack*/ + 256 /*barriers*/;
  static constexpr int TMEM_COLS = BN;
};

template <typename S>
__device__ __forceinline__ double ld_s(const S *p) { return (double)*p; }

// KIND 0: TF32 (FP32 bit patterns; W may be R_Y itself), KIND 1: BF16 operands.
template <int KIND, int BN, typename S>
__global__ void __launch_bounds__(256, 1) dense_tc_kernel(const __grid_constant__ CUtensorMap tmW,
                                                          const __grid_constant__ CUtensorMap tmA,
                                                          const __grid_constant__ CUtensorMap tmAh, DenseTcParams p) {
  using Cfg = DenseCfg<BN>;
  constexpr int KR = KIND == 0 ? 32 : 64;       // K extent of one stage (128 B per operator row)
  extern __shared__ uint8_t smem_raw[];
  // (the offset form smem_raw + pad, which keeps the shared address space and pays off in fe_tc.cu, measures 4 %
  // slower here: 32.6 against 31.2 us per C2 step)
  uint8_t *smem = reinterpret_cast<uint8_t *>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  uint64_t *full_bar = reinterpret_cast<uint64_t *>(smem + Cfg::STAGES * Cfg::STAGE_BYTES);
  uint64_t *empty_bar = full_bar + Cfg::STAGES;
  uint64_t *accum_bar = empty_bar + Cfg::STAGES;
  uint32_t *tmem_slot = reinterpret_cast<uint32_t *>(accum_bar + 1);

  const int warp = threadIdx.x >> 5;
  const int lane = threadIdx.x & 31;
  const int j0 = blockIdx.x * 128;
  const int64_t i0 = (int64_t)blockIdx.y * BN;
  // split-K: the gridDim.z CTAs of a cluster share one output tile; CTA z accumulates its K slice
  const int ks = gridDim.z;
  const int kb_begin = (int)((int64_t)p.num_k_blocks * blockIdx.z / ks);
  const int nkb = (int)((int64_t)p.num_k_blocks * (blockIdx.z + 1) / ks) - kb_begin;

  // multicast (p.mcast): cluster = (2 column tiles, 1, ks K-splits); the pair with the same z loads half of the
  // operator tile each and delivers it to both, so a stage is free only when BOTH consumers have released it
  const bool mc = p.mcast != 0;
  const uint32_t cx = mc ? (blockIdx.x & 1u) : 0u;
  const uint16_t pair_mask = mc ? (uint16_t)(3u << (2u * blockIdx.z)) : (uint16_t)0;
  if (warp == 0 && lane == 0) {
    tma_prefetch_desc(&tmW);
    tma_prefetch_desc(&tmA);
    tma_prefetch_desc(&tmAh);
    for (int s = 0; s < Cfg::STAGES; ++s) {
      mbar_init(full_bar + s, 1);
      mbar_init(empty_bar + s, mc ? 2 : 1);
    }
    mbar_init(accum_bar, 1);
    fence_barrier_init();
  }
  if (warp == 2) tmem_alloc(tmem_slot, Cfg::TMEM_COLS);
  tc_fence_before();
  __syncthreads();
  if (mc) cluster_sync_all();     // every barrier of the cluster exists before the first remote arrival
  tc_fence_after();
  const uint32_t tmem_base = *tmem_slot;

  if (warp == 0) {
    // ===== TMA producer: the whole warp walks the ring, one elected lane issues =====
    for (int kb = 0; kb < nkb; ++kb) {
      const int s = kb % Cfg::STAGES;
      const uint32_t ph = (kb / Cfg::STAGES) & 1;
      mbar_wait(empty_bar + s, ph ^ 1);
      if (elect_one()) {
        if (PROBE(p.debug_mode, 2)) {
          mbar_arrive(full_bar + s);
        } else {
          mbar_expect_tx(full_bar + s, Cfg::STAGE_BYTES);
#pragma unroll
          for (int pn = 0; pn < Cfg::KP; ++pn) {
            uint8_t *ws = smem + s * Cfg::STAGE_BYTES + pn * Cfg::PANEL_BYTES;
            uint8_t *as = ws + Cfg::W_BYTES;
            const int k0 = ((kb_begin + kb) * Cfg::KP + pn) * KR;
            if constexpr (KIND == 0) {
#pragma unroll
              for (int a = 0; a < 4; ++a) tma_load_2d(ws + a * 4096, &tmW, full_bar + s, j0 + 32 * a, k0);
            } else {
#pragma unroll
              for (int a = 0; a < 2; ++a) tma_load_2d(ws + a * 8192, &tmW, full_bar + s, j0 + 64 * a, k0);
            }
            if (mc)
              tma_load_2d_mc(as + cx * (BN / 2) * 128, &tmAh, full_bar + s, k0, (int32_t)(i0 + cx * (BN / 2)), pair_mask);
            else
              tma_load_2d(as, &tmA, full_bar + s, k0, (int32_t)i0);
          }
        }
      }
      __syncwarp();
    }
  } else if (warp == 1) {
    // ===== MMA issuer =====
    constexpr uint32_t idesc = make_idesc(KIND == 0 ? 2 : 1, /*A MN-major*/ 1, /*B K-major*/ 0, 128, BN);
    // W^T tile, MN-major.  TF32: SWIZZLE_128B_BASE32B, 8 k rows per MMA = two 4-row groups (SBO 512 B),
    // M atoms (32 columns) 4096 B apart.  BF16: SWIZZLE_128B, 16 k rows per MMA = two 8-row groups
    // (SBO 1024 B), M atoms (64 columns) 8192 B apart.  Operator rows, K-major SWIZZLE_128B: 32 B of K
    // per MMA inside the 128 B row, 8-row groups 1024 B apart.
    const uint64_t da0 = (KIND == 0) ? make_smem_desc(smem_u32(smem), 4096, 512, 1) : make_smem_desc(smem_u32(smem), 8192, 1024, 2);
    const uint64_t db0 = make_smem_desc(smem_u32(smem) + Cfg::W_BYTES, 16, 1024, 2);
    for (int kb = 0; kb < nkb; ++kb) {
      const int s = kb % Cfg::STAGES;
      const uint32_t ph = (kb / Cfg::STAGES) & 1;
      mbar_wait(full_bar + s, ph);
      tc_fence_after();
      if (elect_one()) {
        if (PROBE(p.debug_mode, 1)) {
          mbar_arrive(empty_bar + s);
        } else {
#pragma unroll
          for (int pn = 0; pn < Cfg::KP; ++pn) {
            const uint32_t off = (uint32_t)(s * Cfg::STAGE_BYTES + pn * Cfg::PANEL_BYTES) >> 4;   // 16-byte units
#pragma unroll
            for (int q = 0; q < 4; ++q) {
              const uint64_t da = da0 + off + (uint32_t)(q * (KIND == 0 ? 1024 : 2048) >> 4);
              const uint64_t db = db0 + off + (uint32_t)(q * 32 >> 4);
              umma<KIND>(tmem_base, da, db, idesc, (kb > 0 || pn > 0 || q > 0) ? 1u : 0u);
            }
          }
          if (mc) umma_commit_mc(empty_bar + s, pair_mask);
          else umma_commit(empty_bar + s);
        }
      }
      __syncwarp();
    }
    if (elect_one()) {
      if (PROBE(p.debug_mode, 1)) mbar_arrive(accum_bar); else umma_commit(accum_bar);
    }
  }
  __syncwarp();
  // ---- epilogue: all 8 warps.  Warp w reads TMEM lanes 32 (w % 4) .. +31 (its lane quarter) and the
  // column half w / 4 of the tile; loads of R_Y, R_X, G for 8 rows are issued before any use.
  {
    const int q = warp & 3;
    const int half = warp >> 2;
    const int j = j0 + 32 * q + lane;
    const bool jok = j < p.N;
    const S *__restrict__ RY = reinterpret_cast<const S *>(p.RY);
    S *__restrict__ RX = reinterpret_cast<S *>(p.RX);
    const S *__restrict__ G = reinterpret_cast<const S *>(p.G);
    const S ly = (S)((G != nullptr && jok) ? p.LY[j] : 0.0);
    const S ka = (S)p.k.a, kb_ = (S)p.k.b, kc = (S)p.k.cp;
    mbar_wait(accum_bar, 0);
    tc_fence_after();
    constexpr int HALF_COLS = BN / 2;
    if (ks > 1) {
      // ---- split-K fix-up over distributed shared memory: every CTA of the cluster parks its partial
      // tile in its own shared memory ([matrix row][128 columns] FP32, over the dead operand stages),
      // then CTA z sums the BN / ks matrix rows it owns over the ranks in fixed order (deterministic)
      // and applies the update to them.
      float *part = reinterpret_cast<float *>(smem);
      const int jl = threadIdx.x & 127;
      const int jj = j0 + jl;
      const bool jjok = jj < p.N && !PROBE(p.debug_mode, 4);
      const S ly2 = (S)((G != nullptr && jjok) ? p.LY[jj] : 0.0);
      const int cpr = BN / ks;                                  // matrix rows owned by this CTA
      const int cbase = blockIdx.z * cpr + (threadIdx.x >> 7);  // this thread: every second owned row
      const int nrow = cpr / 2;
      // R_Y, R_X, G of RB rows at a time; the first batch is requested before the partial tiles are exchanged and
      // every later one while the current batch is summed, so only the first latency is exposed
      constexpr int RB = 16;
      S ry[RB], rx[RB], g[RB];
      auto gload = [&](S (&a)[RB], S (&b)[RB], S (&c)[RB], int u0) {
#pragma unroll
        for (int t = 0; t < RB; ++t) {
          const int64_t i = i0 + cbase + 2 * (u0 + t);
          const int64_t idx = i * p.N + jj;
          const bool ok = jjok && (u0 + t) < nrow && i < p.m;
          a[t] = ok ? __ldg(RY + idx) : S(0);
          b[t] = ok ? RX[idx] : S(0);
          c[t] = (ok && G) ? __ldg(G + idx) : S(0);
        }
      };
      gload(ry, rx, g, 0);
#pragma unroll 1
      for (int c0 = half * HALF_COLS; c0 < (half + 1) * HALF_COLS; c0 += 32) {
        uint32_t r[32];
        tmem_ld_32x32(tmem_base + ((uint32_t)(32 * q) << 16) + (uint32_t)c0, r);
        tmem_ld_wait();
#pragma unroll
        for (int t = 0; t < 32; ++t) part[(c0 + t) * 128 + 32 * q + lane] = __uint_as_float(r[t]);
      }
      cluster_sync_all();
      const uint32_t part_s = smem_u32(part);
#pragma unroll 1
      for (int u0 = 0; u0 < nrow; u0 += RB) {
        if (u0 > 0) gload(ry, rx, g, u0);
        float T[RB];
#pragma unroll
        for (int t = 0; t < RB; ++t) T[t] = 0.f;
        // all the partial sums of the batch are requested before the first is used (fixed rank order: deterministic)
        for (int rr = 0; rr < ks; ++rr) {
          const uint32_t base = dsmem_map(part_s, (PROBE(p.debug_mode, 64) ? blockIdx.z : (uint32_t)rr) * (mc ? 2u : 1u) + cx);   // bit 6: local reads only (timing probe)
          float pv[RB];
#pragma unroll
          for (int t = 0; t < RB; ++t) {
            const int c = cbase + 2 * (u0 + t);
            const bool ok = jjok && (u0 + t) < nrow && i0 + c < p.m;
            pv[t] = ok ? dsmem_ld_f32(base + (uint32_t)(c * 128 + jl) * 4u) : 0.f;
          }
#pragma unroll
          for (int t = 0; t < RB; ++t) T[t] += pv[t];
        }
#pragma unroll
        for (int t = 0; t < RB; ++t) {
          const int c = cbase + 2 * (u0 + t);
          const int64_t i = i0 + c;
          if (jjok && (u0 + t) < nrow && i < p.m) {
            const int64_t idx = i * p.N + jj;
            S Tt = (S)T[t];
            if (p.dinv_out) Tt *= (S)p.dinv_out[i];
            const S out = ka * Tt + kb_ * ry[t] + kc * rx[t] + ka * (g[t] * ly2);
            RX[idx] = out;
            if (p.Wnext) {
              if constexpr (KIND == 0) {
                uint32_t uu;
                asm("cvt.rna.tf32.f32 %0, %1;" : "=r"(uu) : "f"((float)out));
                reinterpret_cast<uint32_t *>(p.Wnext)[idx] = uu;
              } else {
                reinterpret_cast<__nv_bfloat16 *>(p.Wnext)[idx] = __float2bfloat16_rn((float)out);
              }
            }
          }
        }
      }
      cluster_sync_all();     // nobody leaves while its shared memory may still be read
    } else
#pragma unroll 1
    for (int c0 = half * HALF_COLS; c0 < (half + 1) * HALF_COLS; c0 += 32) {
      uint32_t r[32];
      tmem_ld_32x32(tmem_base + ((uint32_t)(32 * q) << 16) + (uint32_t)c0, r);
      tmem_ld_wait();
      if (!jok || PROBE(p.debug_mode, 4)) continue;
#pragma unroll
      for (int t0 = 0; t0 < 32; t0 += 8) {
        S ry[8], rx[8], g[8];
#pragma unroll
        for (int t = 0; t < 8; ++t) {
          const int64_t i = i0 + c0 + t0 + t;
          const int64_t idx = i * p.N + j;
          const bool ok = i < p.m;
          ry[t] = ok ? __ldg(RY + idx) : S(0);
          rx[t] = ok ? RX[idx] : S(0);
          g[t] = (ok && G) ? __ldg(G + idx) : S(0);
        }
#pragma unroll
        for (int t = 0; t < 8; ++t) {
          const int64_t i = i0 + c0 + t0 + t;
          if (i < p.m) {
            const int64_t idx = i * p.N + j;
            S T = (S)__uint_as_float(r[t0 + t]);
            if (p.dinv_out) T *= (S)p.dinv_out[i];
            const S out = ka * T + kb_ * ry[t] + kc * rx[t] + ka * (g[t] * ly);
            RX[idx] = out;
            if (p.Wnext) {
              if constexpr (KIND == 0) {   // round to nearest TF32 here: the MMA itself truncates
                uint32_t u;
                asm("cvt.rna.tf32.f32 %0, %1;" : "=r"(u) : "f"((float)out));
                reinterpret_cast<uint32_t *>(p.Wnext)[idx] = u;
              } else {
                reinterpret_cast<__nv_bfloat16 *>(p.Wnext)[idx] = __float2bfloat16_rn((float)out);
              }
            }
          }
        }
      }
    }
  }
  tc_fence_before();
  __syncthreads();
  if (mc && ks == 1) cluster_sync_all();   // the peer's last release still arrives on this CTA's barriers
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
  LowpCopy *cp = nullptr;
  for (LowpCopy &c : h->lowp)
    if (c.prec == prec && c.folded == folded) cp = &c;
  if (!cp) {
    LowpCopy c;
    c.prec = prec;
    c.folded = folded;
    c.stale = true;
    c.ld = cdiv(h->m, 64) * 64;
    c.rows_pad = h->m;
    c.bytes = dense_lowp_bytes(h->A.d, prec);
    *st = dev_alloc(h, &c.data, c.bytes);
    if (*st != RCHFSI_OK) return nullptr;
    h->lowp.push_back(c);
    cp = &h->lowp.back();
  }
  if (cp->stale) {
    const unsigned grid = (unsigned)std::min<int64_t>(cdiv(h->m * cp->ld, 256), 148 * 16);
    if (prec == RCHFSI_BF16)
      dense_lowp_kernel<1><<<grid, 256, 0, h->stream>>>(h->A.d.dense, h->A.d.lda, folded ? h->dinv : nullptr, cp->data, h->m, cp->ld);
    else
      dense_lowp_kernel<0><<<grid, 256, 0, h->stream>>>(h->A.d.dense, h->A.d.lda, folded ? h->dinv : nullptr, cp->data, h->m, cp->ld);
    h->launches++;
    cp->stale = false;
  }
  return cp;
}

template <int KIND, int BN, typename S>
rchfsi_status launch_dense(rchfsi_ctx *h, const CUtensorMap &tmW, const CUtensorMap &tmA, const CUtensorMap &tmAh,
                           const DenseTcParams &p) {
  using Cfg = DenseCfg<BN>;
  auto kern = dense_tc_kernel<KIND, BN, S>;
  RCHFSI_TRY(ensure_func_smem(h, reinterpret_cast<const void *>(kern), Cfg::SMEM_BYTES));
  cudaLaunchConfig_t cfg{};
  cfg.gridDim = dim3((unsigned)cdiv(p.N, 128), (unsigned)cdiv(p.m, BN), (unsigned)p.ksplit);
  cfg.blockDim = dim3(256);
  cfg.dynamicSmemBytes = Cfg::SMEM_BYTES;
  cfg.stream = h->stream;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeClusterDimension;     // the K splits of a tile form one cluster
  attr[0].val.clusterDim.x = p.mcast ? 2 : 1;
  attr[0].val.clusterDim.y = 1;
  attr[0].val.clusterDim.z = (unsigned)p.ksplit;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  RCHFSI_CUDA_CHECK(h, cudaLaunchKernelEx(&cfg, kern, tmW, tmA, tmAh, p));
  LAUNCH_CHECK(h);
  return RCHFSI_OK;
}

template <int KIND, typename S>
rchfsi_status launch_dense_bn(rchfsi_ctx *h, int bn, const CUtensorMap &tmW, const CUtensorMap &tmA, const CUtensorMap &tmAh,
                              const DenseTcParams &p) {
  if (bn == 256) return launch_dense<KIND, 256, S>(h, tmW, tmA, tmAh, p);
  if (bn == 128) return launch_dense<KIND, 128, S>(h, tmW, tmA, tmAh, p);
  return launch_dense<KIND, 64, S>(h, tmW, tmA, tmAh, p);
}

}  // namespace

bool dense_tc_supported(const rchfsi_operator &A, int32_t N, const rchfsi_options &opt) {
  if (A.kind != RCHFSI_OP_DENSE) return false;
  if (opt.apply_prec == RCHFSI_TF32) return N % 4 == 0;
  if (opt.apply_prec == RCHFSI_BF16) return N % 8 == 0;
  return false;
}
size_t dense_lowp_bytes(const rchfsi_operator &A, int prec) {
  return (size_t)A.m * (size_t)(cdiv(A.m, 64) * 64) * (prec == RCHFSI_BF16 ? 2 : 4);
}

// Tile height BN (operator rows per CTA) and K splits.  Large problems: the widest tile that still gives a full
// wave.  Mid-size problems (config 2: 2 x 32 tiles of 128 rows for 148 SMs): 128-row tiles with the K range split
// over a 2-CTA cluster and the partial tiles summed through distributed shared memory -- 128 CTAs with an N = 128
// MMA (96 cycles for twice the work of the 80-cycle N = 64 one) and 2/3 of the operand traffic of 64-row tiles;
// measured 33.1 against 35.2 us per step.  Small problems: 64-row tiles.
void dense_tc_pick(const Knobs &kn, int64_t m, int32_t N, int nkb128, int *bn_out, int *ks_out) {
  int bn = 0, ks = 1;
  if (kn.dense_bn == 64 || kn.dense_bn == 128 || kn.dense_bn == 256) bn = kn.dense_bn;   // tuning knob
  const int64_t tj = cdiv(N, 128);
  if (bn == 0) {
    const int64_t t128 = tj * cdiv(m, 128);
    if (tj * cdiv(m, 256) >= 120) bn = 256;
    else if (t128 >= 120) bn = 128;
    else if (2 * t128 >= 100 && 2 * t128 <= 148 && nkb128 >= 8) { bn = 128; ks = 2; }
    else bn = 64;
  }
  if (kn.dense_ks == 1 || kn.dense_ks == 2 || kn.dense_ks == 4 || kn.dense_ks == 8) ks = kn.dense_ks;
  *bn_out = bn;
  *ks_out = ks;
}

rchfsi_status dense_tc_prepare(rchfsi_ctx *h, int apply_prec, bool chfsi) {
  rchfsi_status st;
  get_dense_copy(h, apply_prec == RCHFSI_BF16 ? RCHFSI_BF16 : RCHFSI_TF32, !chfsi && h->dinv != nullptr, &st);
  return st;
}

rchfsi_status dense_tc_step(rchfsi_ctx *h, const FusedStep &s) {
  const bool bf16 = (s.apply_prec == RCHFSI_BF16);
  const bool folded = !s.chfsi && h->dinv != nullptr;
  rchfsi_status st;
  const LowpCopy *cp = get_dense_copy(h, bf16 ? RCHFSI_BF16 : RCHFSI_TF32, folded, &st);
  if (!cp) return st;
  const int eb = bf16 ? 2 : 4;
  const int32_t nkb = (int32_t)cdiv(h->m, (bf16 ? 64 : 32) * 2);
  int bn = 64, ks = 1;
  dense_tc_pick(h->knobs, h->m, h->N, nkb, &bn, &ks);
  while (ks > 1 && (nkb < 2 * ks || bn % (2 * ks) != 0)) ks /= 2;
  // W [m][N]: box = 128 B of block columns x (32 | 64) k rows
  CUtensorMap tmW, tmA, tmAh;
  // tmAh: half-height operator tile for the multicast pair (each CTA fetches one half for both)
  if (!get_tmap_2d(h, &tmW, s.W, eb, bf16, (uint64_t)h->m, (uint64_t)h->N, (uint64_t)h->N * eb, bf16 ? 64 : 32,
                   bf16 ? 64 : 32, !bf16) ||
      !get_tmap_2d(h, &tmA, cp->data, eb, bf16, (uint64_t)h->m, (uint64_t)cp->ld, (uint64_t)cp->ld * eb, bf16 ? 64 : 32,
                   (uint32_t)bn) ||
      !get_tmap_2d(h, &tmAh, cp->data, eb, bf16, (uint64_t)h->m, (uint64_t)cp->ld, (uint64_t)cp->ld * eb, bf16 ? 64 : 32,
                   (uint32_t)bn / 2)) {
    h->err = "cuTensorMapEncodeTiled failed";
    return RCHFSI_ECUDA;
  }
  int mcast = (cdiv(h->N, 128) % 2 == 0 && 2 * ks <= 8) ? 1 : 0;
  if (h->knobs.dense_mc == 0) mcast = 0;                                           // tuning knob
  const int dbg = h->knobs.tc_debug;
  if (PROBE(dbg, 3)) mcast = 0;                                                    // the timing probes assume one consumer per stage
  DenseTcParams p{s.k, s.RY, s.RX, s.G, s.LY, s.chfsi ? h->dinv : nullptr, s.Wnext, h->m, h->N,
                  nkb, ks, mcast, dbg};
  if (s.store_prec == RCHFSI_FP64)
    return bf16 ? launch_dense_bn<1, double>(h, bn, tmW, tmA, tmAh, p) : launch_dense_bn<0, double>(h, bn, tmW, tmA, tmAh, p);
  return bf16 ? launch_dense_bn<1, float>(h, bn, tmW, tmA, tmAh, p) : launch_dense_bn<0, float>(h, bn, tmW, tmA, tmAh, p);
}

}  // namespace rchfsi
