// FE cell-batched tensor-core step (PAPER.md:357 Remark 4.1 "sequence of
// element-level dense matrix-matrix multiplications"): per (cell c, tile of 128 block columns)
//   T_c[a][j] = sum_b A_c[a][b] W[conn_c[b]][j]
// on tcgen05 (kind::tf32 / kind::f16 BF16, FP32 accumulate in TMEM) with
//   * the GATHER fused into the prologue: the rows conn_c[b] of the operand block W are fetched by
//     16-byte cp.async straight into the swizzled MN-major operand layout (no gathered copy; TMA
//     tile::gather4 does the same but retires only ~1 op per 100 cycles per SM, see below);
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
  const void *W;              // operand block (FP32 bits for TF32, BF16): R_Y itself or its shadow
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
  int32_t g_rowmajor;         // G is the caller's row-major [m][N] block (FP32, used in place)
  int32_t debug_mode;
};

constexpr int FE_W_BYTES = 16384;
constexpr int FE_WORK_WARPS = 16;                        // gather producers in the main loop, then epilogue
constexpr int FE_THREADS = (FE_WORK_WARPS + 2) * 32;     // + TMA warp (cell-matrix panels) + MMA warp
constexpr int FE_DEPTH = 4;                              // epilogue staging slots per warp
constexpr int FE_SLOT_BYTES = 3072;                      // R_X, R_Y, G: RW rows x 32 columns each
constexpr int FE_STAGES = 3;

// KIND 0: TF32, KIND 1: BF16.  S: storage type of R_X, R_Y, G.
//
// Warp roles (18 warps):
//   warps 0-15  main loop: GATHER producers -- the rows conn_c[b] of the operand block go global -> shared
//               with 16-byte cp.async, each piece written at its place in the swizzled MN-major UMMA
//               operand layout (measured: TMA tile::gather4 retires only ~1 op per 100 cycles per SM,
//               5 B/clk, so the gather is done by the otherwise idle epilogue warps instead);
//               epilogue: each warp stages the R_X / R_Y / G rows it needs in a private ring of
//               FE_DEPTH shared-memory slots with cp.async (bytes in flight independent of registers),
//               reads its TMEM lane quarter, applies the update and stores coalesced 128-byte runs.
//   warp 16     TMA producer of the cell-matrix panels (two 176-row boxes per 128-byte K panel)
//   warp 17     TMEM allocator and MMA issuer (one elected lane)
template <int KIND, typename S>
__global__ void __launch_bounds__(FE_THREADS, 1) fe_tc_kernel(const __grid_constant__ CUtensorMap tmA, FeTcParams p) {
  constexpr int KR = KIND == 0 ? 32 : 64;     // k rows per 128-byte panel
  constexpr int KSTEP = KIND == 0 ? 8 : 16;   // k per MMA
  constexpr int RW = 128 / (4 * (int)sizeof(S)) * 1;   // rows per warp and chunk: 8 (FP32) / 4 (FP64)
  constexpr int R = 4 * RW;                            // rows per chunk over the 4 row-quarters
  constexpr int SEG = 32 * (int)sizeof(S);             // bytes of one row segment (32 columns)
  extern __shared__ uint8_t smem_raw[];
  uint8_t *smem = reinterpret_cast<uint8_t *>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  const int stage_bytes = FE_W_BYTES + p.np * 128;
  const int main_bytes = max(FE_STAGES * stage_bytes, FE_WORK_WARPS * FE_DEPTH * FE_SLOT_BYTES);
  uint64_t *full_bar = reinterpret_cast<uint64_t *>(smem + main_bytes);
  uint64_t *empty_bar = full_bar + 4;
  uint64_t *accum_bar = empty_bar + 4;
  uint32_t *tmem_slot = reinterpret_cast<uint32_t *>(accum_bar + 1);
  // rw_s[a] = (column tile * m + global row of local node a) | first-touch << 30 | last-touch << 31:
  // the row's index in the panel layout [column tile][m][128] and its colouring flags in one word
  uint32_t *rw_s = reinterpret_cast<uint32_t *>(tmem_slot + 2);          // [n_loc]

  const int warp = threadIdx.x >> 5;
  const int lane = threadIdx.x & 31;
  const int j0 = blockIdx.x * 128;
  const int64_t cell = p.cell_order[blockIdx.y];
  const int npanels = (p.debug_mode & 512) ? 0 : (p.ksteps * KSTEP + KR - 1) / KR;   // bit 9: fixed-cost probe
  const uint32_t tmem_cols = (p.np <= 32) ? 32u : (p.np <= 64 ? 64u : (p.np <= 128 ? 128u : (p.np <= 256 ? 256u : 512u)));

  for (int t = threadIdx.x; t < p.n_loc; t += blockDim.x)
    rw_s[t] = (uint32_t)(blockIdx.x * p.m + p.conn[cell * p.n_loc + t]) | ((uint32_t)p.flags[cell * p.n_loc + t] << 30);
  if (warp == FE_WORK_WARPS && lane == 0) {
    tma_prefetch_desc(&tmA);
    for (int s = 0; s < FE_STAGES; ++s) {
      mbar_init(full_bar + s, FE_WORK_WARPS * 32 + 1);   // every gather thread (async, on landing) + the TMA expect_tx arrive
      mbar_init(empty_bar + s, 1);
    }
    mbar_init(accum_bar, 1);
    fence_barrier_init();
  }
  if (warp == FE_WORK_WARPS + 1) tmem_alloc(tmem_slot, tmem_cols);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = *tmem_slot;
  const bool has_g = p.G != nullptr;

  if (warp == FE_WORK_WARPS) {
    // ===== TMA producer: cell-matrix panels =====
    for (int pn = 0; pn < npanels; ++pn) {
      const int s = pn % FE_STAGES;
      mbar_wait(empty_bar + s, ((pn / FE_STAGES) & 1) ^ 1);
      if (elect_one()) {
        uint8_t *as = smem + s * stage_bytes + FE_W_BYTES;
        mbar_expect_tx(full_bar + s, p.np * 128);
        for (int hh = 0; hh < p.nh; ++hh)
          tma_load_2d(as + hh * p.nhalf * 128, &tmA, full_bar + s, 0, (int32_t)((cell * npanels + pn) * p.np + hh * p.nhalf));
      }
      __syncwarp();
    }
  } else if (warp == FE_WORK_WARPS + 1) {
    // ===== MMA issuer =====
    const uint32_t idesc = make_idesc(KIND == 0 ? 2 : 1, /*A MN-major*/ 1, /*B K-major*/ 0, 128, p.nhalf);
    const uint64_t da0 = (KIND == 0) ? make_smem_desc(smem_u32(smem), 4096, 512, 1) : make_smem_desc(smem_u32(smem), 8192, 1024, 2);
    const uint64_t db0 = make_smem_desc(smem_u32(smem) + FE_W_BYTES, 16, 1024, 2);
    for (int pn = 0; pn < npanels; ++pn) {
      const int s = pn % FE_STAGES;
      mbar_wait(full_bar + s, (pn / FE_STAGES) & 1);
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
    __syncwarp();
  } else {
    // ===== main loop: gather the operand rows into the swizzled MN-major layout =====
    {
      const int tid = threadIdx.x;                      // 0 .. 511
      const uint8_t *Wb = reinterpret_cast<const uint8_t *>(p.W);
      constexpr int EB = KIND == 0 ? 4 : 2;             // operand element bytes
      for (int pn = 0; pn < npanels; ++pn) {
        const int s = pn % FE_STAGES;
        mbar_wait(empty_bar + s, ((pn / FE_STAGES) & 1) ^ 1);
        uint8_t *ws = smem + s * stage_bytes;
#pragma unroll
        for (int i = 0; i < 2; ++i) {
          const int piece = tid + i * 512;              // 1024 16-byte pieces per panel
          int k, a, c16;
          uint32_t dst_off;
          if constexpr (KIND == 0) {                    // 32 rows x 512 B; SWIZZLE_128B_ATOM_32B
            k = piece >> 5;
            const int cc = piece & 31;
            a = cc >> 3;
            c16 = cc & 7;
            dst_off = a * 4096 + k * 128 + ((((c16 >> 1) ^ (k & 3)) << 5) | ((c16 & 1) << 4));
          } else {                                      // 64 rows x 256 B; SWIZZLE_128B
            k = piece >> 4;
            const int cc = piece & 15;
            a = cc >> 3;
            c16 = cc & 7;
            dst_off = a * 8192 + k * 128 + ((c16 ^ (k & 7)) << 4);
          }
          const int kk = pn * KR + k;
          const int cl = (a * 128 + c16 * 16) / EB;     // column inside the 128-column panel
          const bool ok = kk < p.n_loc && j0 + cl < p.N;
          const uint32_t rowp = ok ? (rw_s[kk] & 0x3FFFFFFFu) : 0u;
          // panel layout [column tile][m][128]: the rows of one tile are 128 * EB bytes apart
          cp_async16(ws + dst_off, Wb + ((uint64_t)rowp * 128 + (ok ? cl : 0)) * EB, ok ? 16u : 0u);
        }
        // the full barrier gets this thread's arrival when its copies have landed: no thread blocks on
        // its own loads, so all FE_STAGES panels are genuinely in flight
        cp_async_arrive_noinc(full_bar + s);
      }
      cp_async_commit();      // keep the epilogue's group accounting clean
      cp_async_wait<0>();
    }

    // ===== epilogue =====
    const int q4 = warp & 3;
    const int sub = warp >> 2;
    const int jl = 32 * q4 + lane;
    const int j = j0 + jl;
    const bool jok = j < p.N;
    S *__restrict__ RX = reinterpret_cast<S *>(p.RX);
    const uint8_t *srcRX = reinterpret_cast<const uint8_t *>(p.RX);
    const uint8_t *srcRY = reinterpret_cast<const uint8_t *>(p.RY);
    const uint8_t *srcG = reinterpret_cast<const uint8_t *>(p.G);
    // the update runs in the storage precision (FP32 storage: FP32 arithmetic)
    const S ly = (S)((has_g && jok) ? p.LY[j] : 0.0);
    const S ka = (S)p.k.a, kb_ = (S)p.k.b, kc = (S)p.k.cp;
    const int nchunks = (p.n_loc + R - 1) / R;
    uint8_t *ring = smem + warp * (FE_DEPTH * FE_SLOT_BYTES);
    // one slot = [array 0..2][RW rows][SEG bytes] = 192 16-byte pieces, 6 per lane: a lane copies the same
    // 16-byte column piece of two rows (h = 0, 1) for the three arrays; everything lane-constant is hoisted
    constexpr int PPR = SEG / 16;                       // pieces per row segment: 8 (FP32) / 16 (FP64)
    constexpr int RSTEP = 32 / PPR;                     // rows covered by the 32 lanes: 4 / 2
    const int t_lane = lane / PPR;
    const int pc = lane % PPR;
    const bool colok = j0 + 32 * q4 + pc * (16 / (int)sizeof(S)) < p.N;
    const uint32_t col_bytes = (uint32_t)(32 * q4 * (int)sizeof(S) + pc * 16);
    const uint32_t dst_lane = (uint32_t)(t_lane * SEG + pc * 16);
    auto issue_chunk = [&](int c) {
      if (c < nchunks) {
        uint8_t *slot = ring + (c % FE_DEPTH) * FE_SLOT_BYTES;
#pragma unroll
        for (int hsel = 0; hsel < 2; ++hsel) {
          const int a = c * R + sub * RW + t_lane + RSTEP * hsel;
          const uint32_t w = (a < p.n_loc && colok) ? rw_s[a] : 0u;
          const bool valid = (a < p.n_loc) && colok && !(p.debug_mode & 2048);     // bit 11: no epilogue loads (timing probe)
          const bool first = ((w >> 30) & 1u) && !(p.debug_mode & 4096);           // bit 12: no R_Y / G loads (timing probe)
          const uint64_t off = (uint64_t)(w & 0x3FFFFFFFu) * (128 * sizeof(S)) + col_bytes;
          uint8_t *d = slot + dst_lane + hsel * (RSTEP * SEG);
          cp_async16(d, srcRX + off, valid ? 16u : 0u);
          cp_async16(d + 1024, srcRY + off, (valid && first) ? 16u : 0u);
          // G: panel layout like R_X / R_Y, or the caller's own row-major block (g_rowmajor)
          const uint64_t offg = p.g_rowmajor ? ((uint64_t)((w & 0x3FFFFFFFu) - (uint32_t)(blockIdx.x * p.m)) * (uint64_t)p.N + j0) * sizeof(S) + col_bytes
                                             : off;
          cp_async16(d + 2048, (has_g ? srcG + offg : srcRX + off), (valid && first && has_g) ? 16u : 0u);
        }
      }
      cp_async_commit();
    };
    mbar_wait(accum_bar, 0);     // every MMA done: TMEM complete, operand stages free for the rings
    tc_fence_after();
    if (!(p.debug_mode & 4)) {
#pragma unroll
      for (int c = 0; c < FE_DEPTH - 1; ++c) issue_chunk(c);
#pragma unroll 1
      for (int c = 0; c < nchunks; ++c) {
        issue_chunk(c + FE_DEPTH - 1);
        uint32_t r[RW];
        if constexpr (RW == 8)
          tmem_ld_32x8(tmem_base + ((uint32_t)(32 * q4) << 16) + (uint32_t)(c * R + sub * RW), r);
        else
          tmem_ld_32x4(tmem_base + ((uint32_t)(32 * q4) << 16) + (uint32_t)(c * R + sub * RW), r);
        tmem_ld_wait();
        cp_async_wait<FE_DEPTH - 1>();
        __syncwarp();
        const uint8_t *slot = ring + (c % FE_DEPTH) * FE_SLOT_BYTES;
        const S *rxs = reinterpret_cast<const S *>(slot);
        const S *rys = reinterpret_cast<const S *>(slot + 1024);
        const S *gs = reinterpret_cast<const S *>(slot + 2048);
#pragma unroll
        for (int t = 0; t < RW; ++t) {
          const int a = c * R + sub * RW + t;
          if (a < p.n_loc && jok) {
            const uint32_t w = rw_s[a];
            const uint32_t flt = w >> 30;
            const int64_t idx = (int64_t)(w & 0x3FFFFFFFu) * 128 + jl;
            S T = (S)__uint_as_float(r[t]);
            if (p.dinv_out) T *= (S)p.dinv_out[(w & 0x3FFFFFFFu) - (uint32_t)(blockIdx.x * p.m)];
            S out;
            if (flt & 1u)
              out = ka * T + kb_ * rys[t * 32 + lane] + kc * rxs[t * 32 + lane] + ka * (gs[t * 32 + lane] * ly);
            else
              out = rxs[t * 32 + lane] + ka * T;
            if (!(p.debug_mode & 1024)) RX[idx] = out;                             // bit 10: no stores (timing probe)
            if (p.Wnext && (flt & 2u) && !(p.debug_mode & 1024)) {
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
        __syncwarp();     // all lanes done with this slot before it is refilled
      }
      cp_async_wait<0>();
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == FE_WORK_WARPS + 1) {
    tc_fence_after();
    tmem_dealloc(tmem_base, tmem_cols);
  }
}

}  // namespace
}  // namespace rchfsi

#include "fe_tc_host.inc"
