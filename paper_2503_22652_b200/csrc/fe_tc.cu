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
#include <type_traits>
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
  // 1 KB alignment as an OFFSET from the shared array: a pointer rebuilt from an integer loses its address
  // space and every later access compiles to a generic LD/ST with 64-bit address math instead of LDS/STS
  uint8_t *smem = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);
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
  const int npanels = PROBE(p.debug_mode, 512) ? 0 : (p.ksteps * KSTEP + KR - 1) / KR;   // bit 9: fixed-cost probe
  const uint32_t tmem_cols = (p.np <= 32) ? 32u : (p.np <= 64 ? 64u : (p.np <= 128 ? 128u : (p.np <= 256 ? 256u : 512u)));

  if (warp == FE_WORK_WARPS && lane == 0) {
    tma_prefetch_desc(&tmA);
    for (int s = 0; s < FE_STAGES; ++s) {
      mbar_init(full_bar + s, FE_WORK_WARPS * 32 + 1);   // every gather thread (async, on landing) + the TMA expect_tx arrive
      mbar_init(empty_bar + s, 1);
    }
    mbar_init(accum_bar, 1);
    fence_barrier_init();
    // the first FE_STAGES cell-matrix panels need nothing from the other warps: their TMA loads go out before the
    // node words are set up and TMEM is allocated, so ~1 us of the per-CTA fixed cost runs under their latency
    for (int pn = 0; pn < min(FE_STAGES, npanels); ++pn) {
      uint8_t *as = smem + pn * stage_bytes + FE_W_BYTES;
      if (PROBE(p.debug_mode, 8192)) { mbar_arrive(full_bar + pn); continue; }    // bit 13: MMA-only probe (no TMA, no gather reads)
      mbar_expect_tx(full_bar + pn, p.np * 128);
      for (int hh = 0; hh < p.nh; ++hh)
        tma_load_2d(as + hh * p.nhalf * 128, &tmA, full_bar + pn, 0, (int32_t)((cell * npanels + pn) * p.np + hh * p.nhalf));
    }
  }
  for (int t = threadIdx.x; t < ((p.n_loc + 31) & ~31); t += blockDim.x)      // zero padded to whole chunks
    rw_s[t] = t < p.n_loc ? ((uint32_t)(blockIdx.x * p.m + p.conn[cell * p.n_loc + t]) | ((uint32_t)p.flags[cell * p.n_loc + t] << 30)) : 0u;
  if (warp == FE_WORK_WARPS + 1) tmem_alloc(tmem_slot, tmem_cols);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = *tmem_slot;
  const bool has_g = p.G != nullptr;

  if (warp == FE_WORK_WARPS) {
    // ===== TMA producer: cell-matrix panels (the first FE_STAGES were issued during the set-up) =====
    for (int pn = FE_STAGES; pn < npanels; ++pn) {
      const int s = pn % FE_STAGES;
      mbar_wait(empty_bar + s, ((pn / FE_STAGES) & 1) ^ 1);
      if (elect_one()) {
        uint8_t *as = smem + s * stage_bytes + FE_W_BYTES;
        if (PROBE(p.debug_mode, 8192)) {
          mbar_arrive(full_bar + s);
        } else {
          mbar_expect_tx(full_bar + s, p.np * 128);
          for (int hh = 0; hh < p.nh; ++hh)
            tma_load_2d(as + hh * p.nhalf * 128, &tmA, full_bar + s, 0, (int32_t)((cell * npanels + pn) * p.np + hh * p.nhalf));
        }
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
          const bool ok = kk < p.n_loc && j0 + cl < p.N && !PROBE(p.debug_mode, 8192);
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
    // The epilogue is instruction-issue bound (16 warps, one element per lane and row: with every global
    // access disabled it still takes ~14 us of the 26 us tile), so everything lane- or tile-constant is
    // hoisted: per-lane base pointers (one IMAD.WIDE per address), the node words of a chunk as 128-bit
    // shared loads, chunks that lie fully inside n_loc without per-row range checks, uniform branches
    // around the rarely used pieces (dinv on the output rows, shadow store, row-major G).
    const int q4 = warp & 3;
    const int sub = warp >> 2;
    const int jl = 32 * q4 + lane;
    const int j = j0 + jl;
    const bool jok = j < p.N;
    const bool do_store = jok && !PROBE(p.debug_mode, 1024);           // bit 10: no stores (timing probe)
    const bool has_shadow = p.Wnext != nullptr;
    const uint32_t tile_m = (uint32_t)(blockIdx.x * p.m);
    constexpr uint32_t ROWB = 128 * sizeof(S);          // bytes of one row of a panel
    constexpr uint32_t WB = KIND == 0 ? 4 : 2;          // shadow element bytes
    const uint64_t rx_lane = (uint64_t)__cvta_generic_to_global(p.RX) + (uint64_t)jl * sizeof(S);
    const uint64_t wn_lane = has_shadow ? (uint64_t)__cvta_generic_to_global(p.Wnext) + (uint64_t)jl * WB : 0;
    // the update runs in the storage precision (FP32 storage: FP32 arithmetic)
    const S ly = (S)((has_g && jok) ? p.LY[j] : 0.0);
    const S ka = (S)p.k.a, kb_ = (S)p.k.b, kc = (S)p.k.cp;
    const int nchunks = (p.n_loc + R - 1) / R;
    uint8_t *ring = smem + warp * (FE_DEPTH * FE_SLOT_BYTES);
    // one slot = [array 0..2][RW rows][SEG bytes] = 192 16-byte pieces, 6 per lane: a lane copies the same
    // 16-byte column piece of two rows (h = 0, 1) for the three arrays
    constexpr int PPR = SEG / 16;                       // pieces per row segment: 8 (FP32) / 16 (FP64)
    constexpr int RSTEP = 32 / PPR;                     // rows covered by the 32 lanes: 4 / 2
    const int t_lane = lane / PPR;
    const int pc = lane % PPR;
    const bool colok = j0 + 32 * q4 + pc * (16 / (int)sizeof(S)) < p.N && !PROBE(p.debug_mode, 2048);   // bit 11: no epilogue loads (probe)
    const uint32_t col_bytes = (uint32_t)(32 * q4 * (int)sizeof(S) + pc * 16);
    const uint64_t srcRX = (uint64_t)__cvta_generic_to_global(p.RX) + col_bytes;
    const uint64_t srcRY = (uint64_t)__cvta_generic_to_global(p.RY) + col_bytes;
    // G: panel layout like R_X / R_Y, or the caller's own row-major block [m][N] (g_rowmajor)
    const bool g_rm = p.g_rowmajor != 0;
    const uint32_t g_rowb = g_rm ? (uint32_t)p.N * (uint32_t)sizeof(S) : ROWB;
    const uint32_t g_sub = g_rm ? tile_m : 0u;
    const uint64_t srcG = (uint64_t)__cvta_generic_to_global(has_g ? p.G : p.RX) + col_bytes + (g_rm ? (uint64_t)j0 * sizeof(S) : (uint64_t)0);
    const bool g_ok = has_g && !PROBE(p.debug_mode, 4096);              // bit 12: no R_Y / G loads (timing probe)
    const bool ry_ok = !PROBE(p.debug_mode, 4096);
    const uint32_t ring_lane = smem_u32(ring) + (uint32_t)(t_lane * SEG + pc * 16);
    const uint32_t *rw_lane = rw_s + sub * RW + t_lane;
    const int a_lane = sub * RW + t_lane;
    auto issue_chunk = [&](int c) {
      if (c < nchunks) {
        const uint32_t d0 = ring_lane + (uint32_t)((c % FE_DEPTH) * FE_SLOT_BYTES);
#pragma unroll
        for (int hsel = 0; hsel < 2; ++hsel) {
          const uint32_t w = rw_lane[c * R + RSTEP * hsel];        // padded with zeros past n_loc
          const bool valid = (c * R + RSTEP * hsel + a_lane < p.n_loc) && colok;
          const bool first = (w & 0x40000000u) != 0;
          const uint32_t rowp = w & 0x3FFFFFFFu;
          const uint32_t d = d0 + hsel * (RSTEP * SEG);
          cp_async16_sa(d, mad_wide_u32(rowp, ROWB, srcRX), valid ? 16u : 0u);
          cp_async16_sa(d + 1024, mad_wide_u32(rowp, ROWB, srcRY), (valid && first && ry_ok) ? 16u : 0u);
          cp_async16_sa(d + 2048, mad_wide_u32(rowp - g_sub, g_rowb, srcG), (valid && first && g_ok) ? 16u : 0u);
        }
      }
      cp_async_commit();
    };
    // rows of one chunk
    auto do_rows = [&](int c, const uint32_t (&r)[RW]) {
      const int a0 = c * R + sub * RW;
      const int nv = do_store ? p.n_loc - a0 : 0;                   // rows t < nv are stored by this lane
      const uint8_t *slot = ring + (c % FE_DEPTH) * FE_SLOT_BYTES;
      const S *rxs = reinterpret_cast<const S *>(slot) + lane;
      const S *rys = reinterpret_cast<const S *>(slot + 1024) + lane;
      const S *gs = reinterpret_cast<const S *>(slot + 2048) + lane;
      uint32_t wv[RW];
      S rxv[RW], ryv[RW], gv[RW], Tv[RW];
#pragma unroll
      for (int q = 0; q < RW / 4; ++q) {
        const uint4 v = *reinterpret_cast<const uint4 *>(rw_s + a0 + 4 * q);
        wv[4 * q] = v.x; wv[4 * q + 1] = v.y; wv[4 * q + 2] = v.z; wv[4 * q + 3] = v.w;
      }
#pragma unroll
      for (int t = 0; t < RW; ++t) {
        rxv[t] = rxs[t * 32];
        ryv[t] = rys[t * 32];
        gv[t] = gs[t * 32];
        Tv[t] = (S)__uint_as_float(r[t]);
      }
      if (p.dinv_out) {                                             // ChFSI: D^-1 on the output rows
#pragma unroll
        for (int t = 0; t < RW; ++t)
          if (a0 + t < p.n_loc) Tv[t] *= (S)p.dinv_out[(wv[t] & 0x3FFFFFFFu) - tile_m];
      }
      S outv[RW];
#pragma unroll
      for (int t = 0; t < RW; ++t) {
        const uint32_t w = wv[t];
        const S out_first = ka * Tv[t] + kb_ * ryv[t] + kc * rxv[t] + ka * (gv[t] * ly);
        const S out_later = rxv[t] + ka * Tv[t];
        outv[t] = (w & 0x40000000u) ? out_first : out_later;
        if (t < nv) st_global(mad_wide_u32(w & 0x3FFFFFFFu, ROWB, rx_lane), outv[t]);
      }
      if (has_shadow) {                                             // last toucher: operand-precision shadow row
#pragma unroll
        for (int t = 0; t < RW; ++t) {
          const uint32_t w = wv[t];
          if (t < nv && (w & 0x80000000u)) {
            if constexpr (KIND == 0) {
              uint32_t u;
              asm("cvt.rna.tf32.f32 %0, %1;" : "=r"(u) : "f"((float)outv[t]));
              st_global_u32(mad_wide_u32(w & 0x3FFFFFFFu, 128 * WB, wn_lane), u);
            } else {
              st_global_u16(mad_wide_u32(w & 0x3FFFFFFFu, 128 * WB, wn_lane), __bfloat16_as_ushort(__float2bfloat16_rn((float)outv[t])));
            }
          }
        }
      }
    };
    mbar_wait(accum_bar, 0);     // every MMA done: TMEM complete, operand stages free for the rings
    tc_fence_after();
    if (!PROBE(p.debug_mode, 4)) {
#pragma unroll
      for (int c = 0; c < FE_DEPTH - 1; ++c) issue_chunk(c);
      // accumulator columns of chunk c + 1 are requested while chunk c is processed
      const uint32_t tm0 = tmem_base + ((uint32_t)(32 * q4) << 16) + (uint32_t)(sub * RW);
      uint32_t rn[RW];
      if constexpr (RW == 8) tmem_ld_32x8(tm0, rn); else tmem_ld_32x4(tm0, rn);
#pragma unroll 1
      for (int c = 0; c < nchunks; ++c) {
        issue_chunk(c + FE_DEPTH - 1);
        tmem_ld_wait();
        uint32_t r[RW];
#pragma unroll
        for (int t = 0; t < RW; ++t) r[t] = rn[t];
        if (c + 1 < nchunks) {
          if constexpr (RW == 8) tmem_ld_32x8(tm0 + (uint32_t)((c + 1) * R), rn); else tmem_ld_32x4(tm0 + (uint32_t)((c + 1) * R), rn);
        }
        cp_async_wait<FE_DEPTH - 1>();
        __syncwarp();
        do_rows(c, r);
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

#include "fe_pipe.inc"
#include "fe_tc_host.inc"
