// FE cell-batched tensor-core step (PAPER.md:357 Remark 4.1 "sequence of
// element-level dense matrix-matrix multiplications"): per (cell c, tile of 128 block columns)
//   T_c[a][j] = sum_b A_c[a][b] W[conn_c[b]][j]
// on tcgen05 (kind::tf32 / kind::f16 BF16, FP32 accumulate in TMEM) with
//   * the GATHER fused into the prologue: the rows conn_c[b] of the operand block W are fetched by
//     TMA tile::gather4 straight into the swizzled MN-major operand layout (no gathered copy);
//   * an ATOMIC-FREE scatter-add fused with the Alg. 3 update: the cells are
//     coloured so that cells of one colour share no node; colours run as stream-ordered launches.
//     The update is linear in T, so the first cell touching a node writes
//         R_X <- a T_c + b R_Y + c' R_X + a G Lambda_Y
//     and every later cell adds  R_X += a T_c  with a plain read-modify-write; the last toucher also
//     writes the operand-precision shadow of the finished row.  Deterministic, no atomics.
// Orientation as in dense_tc.cu: accumulator D[128 columns j][local nodes a], so TMEM lane = block
// column (coalesced global access in the epilogue) and TMEM column = local node.
// D^-1 is folded into the columns of the low-precision cell matrices (A_c diag(dinv[conn_c])), an
// exact identity A D^-1 = sum_c P_c^T (A_c D_c^-1) P_c.
#include <algorithm>
#include <cstdlib>
#include "common.cuh"
#include "tc_common.cuh"

namespace rchfsi {

namespace {

using namespace tc;

struct FeTcParams {
  StepCoef k;
  const void *RY;
  void *RX;
  const void *G;
  const double *LY;
  const double *dinv_out;
  void *Wnext;
  const int32_t *conn;        // [n_cells][n_loc]
  const uint8_t *flags;       // [n_cells][n_loc] bit0 first toucher, bit1 last toucher
  const int32_t *cell_order;  // cells of this colour
  int64_t m;
  int32_t N;
  int32_t n_loc;
  int32_t nh;                 // accumulator halves (1 or 2)
  int32_t nhalf;              // local nodes per half (multiple of 16, <= 256)
  int32_t np;                 // padded local-node extent of the low-precision copy (= nh * nhalf)
  int32_t ksteps;             // MMA K steps: ceil(n_loc / (8 | 16))
  int32_t stages;
  int32_t debug_mode;
};

constexpr int FE_W_BYTES = 16384;
constexpr int FE_THREADS = 512;   // 16 warps: the epilogue needs memory-level parallelism

// KIND 0: TF32, KIND 1: BF16.  S: storage type of R_X, R_Y, G.
template <int KIND, typename S>
__global__ void __launch_bounds__(FE_THREADS, 1) fe_tc_kernel(const __grid_constant__ CUtensorMap tmW,
                                                       const __grid_constant__ CUtensorMap tmA, FeTcParams p) {
  constexpr int KR = KIND == 0 ? 32 : 64;     // k rows per 128-byte panel
  constexpr int KSTEP = KIND == 0 ? 8 : 16;   // k per MMA
  extern __shared__ uint8_t smem_raw[];
  uint8_t *smem = reinterpret_cast<uint8_t *>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  const int a_bytes = p.np * 128;
  const int stage_bytes = FE_W_BYTES + a_bytes;
  uint64_t *full_bar = reinterpret_cast<uint64_t *>(smem + p.stages * stage_bytes);
  uint64_t *empty_bar = full_bar + 8;
  uint64_t *accum_bar = empty_bar + 8;
  uint32_t *tmem_slot = reinterpret_cast<uint32_t *>(accum_bar + 1);
  int32_t *conn_s = reinterpret_cast<int32_t *>(tmem_slot + 2);          // [n_loc]
  uint8_t *flag_s = reinterpret_cast<uint8_t *>(conn_s + p.n_loc);       // [n_loc]

  const int warp = threadIdx.x >> 5;
  const int lane = threadIdx.x & 31;
  const int j0 = blockIdx.x * 128;
  const int64_t cell = p.cell_order[blockIdx.y];
  const int npanels = (p.ksteps * KSTEP + KR - 1) / KR;
  const uint32_t tmem_cols = (p.np <= 32) ? 32u : (p.np <= 64 ? 64u : (p.np <= 128 ? 128u : (p.np <= 256 ? 256u : 512u)));

  for (int t = threadIdx.x; t < p.n_loc; t += blockDim.x) {
    conn_s[t] = p.conn[cell * p.n_loc + t];
    flag_s[t] = p.flags[cell * p.n_loc + t];
  }
  if (warp == 0 && lane == 0) {
    tma_prefetch_desc(&tmW);
    tma_prefetch_desc(&tmA);
    for (int s = 0; s < p.stages; ++s) {
      mbar_init(full_bar + s, 1);
      mbar_init(empty_bar + s, 1);
    }
    mbar_init(accum_bar, 1);
    fence_barrier_init();
  }
  if (warp == 2) tmem_alloc(tmem_slot, tmem_cols);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = *tmem_slot;

  if (warp == 0) {
    // ===== producer: 32 lanes issue the 32 gather4 loads of a panel in parallel =====
    for (int pn = 0; pn < npanels; ++pn) {
      const int s = pn % p.stages;
      const uint32_t ph = (pn / p.stages) & 1;
      mbar_wait(empty_bar + s, ph ^ 1);
      uint8_t *ws = smem + s * stage_bytes;
      if (lane == 0) mbar_expect_tx(full_bar + s, stage_bytes);
      __syncwarp();
      // lane -> (group of 4 k rows, 128-byte column chunk)
      const int g = (KIND == 0) ? (lane >> 2) : (lane >> 1);
      const int a = (KIND == 0) ? (lane & 3) : (lane & 1);
      const int kbase = pn * KR + 4 * g;
      int32_t r[4];
#pragma unroll
      for (int t = 0; t < 4; ++t) r[t] = (kbase + t < p.n_loc) ? conn_s[kbase + t] : (int32_t)p.m;   // row m is out of bounds: zeros
      tma_gather4(ws + a * (KIND == 0 ? 4096 : 8192) + g * 512, &tmW, full_bar + s, j0 + a * (KIND == 0 ? 32 : 64), r[0], r[1],
                  r[2], r[3]);
      if (lane < p.nh)
        tma_load_2d(ws + FE_W_BYTES + lane * p.nhalf * 128, &tmA, full_bar + s, pn * KR, (int32_t)(cell * p.np + lane * p.nhalf));
      __syncwarp();
    }
  } else if (warp == 1) {
    // ===== MMA issuer =====
    const uint32_t idesc = make_idesc(KIND == 0 ? 2 : 1, /*A MN-major*/ 1, /*B K-major*/ 0, 128, p.nhalf);
    const uint64_t da0 = (KIND == 0) ? make_smem_desc(smem_u32(smem), 4096, 512, 1) : make_smem_desc(smem_u32(smem), 8192, 1024, 2);
    const uint64_t db0 = make_smem_desc(smem_u32(smem) + FE_W_BYTES, 16, 1024, 2);
    for (int pn = 0; pn < npanels; ++pn) {
      const int s = pn % p.stages;
      const uint32_t ph = (pn / p.stages) & 1;
      mbar_wait(full_bar + s, ph);
      tc_fence_after();
      if (elect_one()) {
        const uint32_t off = (uint32_t)(s * stage_bytes) >> 4;
        const int nq = min(4, p.ksteps - 4 * pn);
        for (int q = 0; q < nq; ++q) {
          const uint64_t da = da0 + off + (uint32_t)(q * (KIND == 0 ? 1024 : 2048) >> 4);
          for (int hh = 0; hh < p.nh; ++hh) {
            const uint64_t db = db0 + off + (uint32_t)((hh * p.nhalf * 128 + q * 32) >> 4);
            umma<KIND>(tmem_base + hh * p.nhalf, da, db, idesc, (pn > 0 || q > 0) ? 1u : 0u);
          }
        }
        umma_commit(empty_bar + s);
      }
      __syncwarp();
    }
    if (elect_one()) umma_commit(accum_bar);
  }
  __syncwarp();

  // ===== epilogue: all 16 warps; lane quarter = warp % 4, 16-row chunks interleaved over warp / 4.
  // All loads of a batch (R_X always; R_Y and G on first-touch rows) are issued before any use:
  // this phase is HBM-bound and lives on bytes in flight.
  {
    constexpr int BATCH = sizeof(S) == 8 ? 8 : 16;
    const int q4 = warp & 3;
    const int par = warp >> 2;
    const int j = j0 + 32 * q4 + lane;
    const bool jok = j < p.N;
    const S *__restrict__ RY = reinterpret_cast<const S *>(p.RY);
    S *__restrict__ RX = reinterpret_cast<S *>(p.RX);
    const S *__restrict__ G = reinterpret_cast<const S *>(p.G);
    // the update runs in the storage precision (FP32 storage: FP32 arithmetic)
    const S ly = (S)((G != nullptr && jok) ? p.LY[j] : 0.0);
    const S ka = (S)p.k.a, kb_ = (S)p.k.b, kc = (S)p.k.cp;
    mbar_wait(accum_bar, 0);
    tc_fence_after();
    const int nchunks = (p.n_loc + 15) >> 4;
#pragma unroll 1
    for (int ch = par; ch < nchunks; ch += FE_THREADS / 128) {
      uint32_t r[16];
      tmem_ld_32x16(tmem_base + ((uint32_t)(32 * q4) << 16) + (uint32_t)(ch * 16), r);
      tmem_ld_wait();
      if (!jok || (p.debug_mode & 4)) continue;
#pragma unroll
      for (int t0 = 0; t0 < 16; t0 += BATCH) {
        S rx[BATCH], ry[BATCH], g[BATCH];
#pragma unroll
        for (int t = 0; t < BATCH; ++t) {
          const int a = ch * 16 + t0 + t;
          const bool ok = a < p.n_loc;
          const int aa = ok ? a : 0;
          const bool first = ok && (flag_s[aa] & 1u);
          const int64_t idx = (int64_t)conn_s[aa] * p.N + j;
          rx[t] = ok ? RX[idx] : S(0);
          ry[t] = first ? __ldg(RY + idx) : S(0);
          g[t] = (first && G) ? __ldg(G + idx) : S(0);
        }
#pragma unroll
        for (int t = 0; t < BATCH; ++t) {
          const int a = ch * 16 + t0 + t;
          if (a < p.n_loc) {
            const uint32_t flt = flag_s[a];
            const int32_t rowt = conn_s[a];
            const int64_t idx = (int64_t)rowt * p.N + j;
            S T = (S)__uint_as_float(r[t0 + t]);
            if (p.dinv_out) T *= (S)p.dinv_out[rowt];
            S out;
            if (flt & 1u)
              out = ka * T + kb_ * ry[t] + kc * rx[t] + ka * (g[t] * ly);
            else
              out = rx[t] + ka * T;
            RX[idx] = out;
            if (p.Wnext && (flt & 2u)) {
              if constexpr (KIND == 0) {
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
  if (warp == 2) {
    tc_fence_after();
    tmem_dealloc(tmem_base, tmem_cols);
  }
}

}  // namespace
}  // namespace rchfsi

#include "fe_tc_host.inc"
