// Rayleigh-Ritz rotation X = Y E on the INT8 tensor pipe ("X = Y E", FP64 by
// PAPER.md:25 footnote 1).  cuBLAS dgemm runs this product at the FP64 rate (34 TFLOP/s measured, 40 nominal); the INT8
// tcgen05 path has >100x that rate, so an error-free split of the FP64 operands pays even at 28 integer products per
// FP64 product (Ozaki-type scheme, restated here from the arithmetic, not from any code):
//
//   * every ROW i of Y and every COLUMN j of E gets a power-of-two scale 2^ea_i / 2^eb_j with |y| 2^-ea < 1, and its
//     entries become 54-bit fixed-point integers q = rint(y 2^(54 - ea));  the largest entry of the row keeps all 53
//     mantissa bits, smaller entries are rounded at 2^-54 of the row maximum (absolute, like a fixed-point dot product);
//   * q is written in S = 7 balanced base-256 digits d_0 (most significant) .. d_6, each an int8 in [-128, 127]:
//     q = sum_s d_s 256^(6-s), exactly;
//   * digit planes multiply exactly on the tensor pipe (tcgen05.mma kind::i8, INT32 accumulators): all pairs (s, t) of
//     one anti-diagonal d = s + t share the weight 2^(-12-8d) and ONE accumulator; the pairs with d <= 6 are kept
//     (28 products), the dropped ones weigh <= 2^-54 each relative to (row max)(column max);
//     INT32 is exact while (d+1) K 2^14 < 2^31, i.e. K = N <= 18000;
//   * epilogue: X_ij = 2^(ea_i + eb_j - 12) sum_d acc_d 2^(-8d) in FP64 (Horner from d = 6).
//
// Kernels: i8_slice_kernel (digit planes of a row chunk of Y, or of the columns of E), i8_rotate_kernel (TMA ->
// shared-memory rings -> tcgen05.mma kind::i8 -> 7 TMEM accumulators -> FP64 recombination).  The rotation runs in
// place, one row chunk at a time: once the digit planes of a chunk exist its rows of Y are dead.
#include <algorithm>
#include <vector>
#include "common.cuh"
#include "tc_common.cuh"

namespace rchfsi {
namespace {

using namespace tc;

constexpr int I8_S = 7;                 // digit planes per operand
constexpr int I8_BN = 64;               // output columns per CTA (7 accumulators x 64 = 448 of 512 TMEM columns)
constexpr int I8_A_TILE = 128 * 128;    // 128 rows x 128 B of K
constexpr int I8_B_TILE = I8_BN * 128;
constexpr int I8_NA = 6;                // A ring slots (tiles are consumed and released in order)
constexpr int I8_SMEM = I8_NA * I8_A_TILE + 2 * I8_S * I8_B_TILE + 1024 /*align*/ + 256 /*barriers*/;
constexpr int32_t I8_NAN_ROW = 0x7fffffff;

__device__ __forceinline__ void umma_i8(uint32_t tmem_d, uint64_t desc_a, uint64_t desc_b, uint32_t idesc, uint32_t accumulate) {
  asm volatile(
      "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::1.kind::i8 [%0], %1, %2, %3, p;\n\t}" ::"r"(tmem_d),
      "l"(desc_a), "l"(desc_b), "r"(idesc), "r"(accumulate)
      : "memory");
}
// instruction descriptor: S32 accumulate (2 at bit 4), signed 8-bit A and B (1 at bits 7 and 10), both K-major
__host__ __device__ constexpr uint32_t make_idesc_i8(int M, int N) {
  return (2u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)(N >> 3) << 17) | ((uint32_t)(M >> 4) << 24);
}

// Balanced base-256 digits without a loop: q = sum_k d_k 256^k with d_k in [-128, 127] is the same as
// q + sum_k 128 256^k = sum_k (d_k + 128) 256^k with plain unsigned digits, so byte k of b = q + 0x0080808080808080 is
// d_k + 128 and d_k is that byte with its top bit flipped.  Digit k (0 = least significant) of four values at once:
constexpr unsigned long long I8_BIAS = 0x0080808080808080ull;
__device__ __forceinline__ uint32_t i8_digits(const uint32_t (&lo)[4], const uint32_t (&hi)[4], int k) {
  const uint32_t *w = k < 4 ? lo : hi;
  const uint32_t sel = 0x0040u + (uint32_t)(k & 3) * 0x0011u;          // bytes k of the first and of the second operand
  const uint32_t p01 = __byte_perm(w[0], w[1], sel);
  const uint32_t p23 = __byte_perm(w[2], w[3], sel);
  return __byte_perm(p01, p23, 0x5410u) ^ 0x80808080u;
}

// One warp per row of V ([rows][K], row pitch ld): row exponent, then the 7 digit planes planes[s][row][Kp].
// Columns K..Kp-1 of the planes are zero (Kp = K rounded up to 16: TMA row pitch).
__global__ void __launch_bounds__(256) i8_slice_kernel(const double *__restrict__ V, int64_t ld, int64_t rows, int32_t K,
                                                       int32_t Kp, int8_t *__restrict__ planes, int64_t plane_rows,
                                                       int32_t *__restrict__ expo) {
  const int lane = threadIdx.x & 31;
  const int64_t row = (int64_t)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
  if (row >= rows) return;
  const double *v = V + row * ld;
  double mx = 0.0;
  bool bad = false;
  for (int k = lane; k < K; k += 32) {
    const double a = fabs(v[k]);
    bad |= !(a <= 1.7976931348623157e308);      // inf or NaN
    mx = fmax(mx, a);
  }
  for (int o = 16; o > 0; o >>= 1) {
    mx = fmax(mx, __shfl_xor_sync(0xffffffffu, mx, o));
    bad |= __shfl_xor_sync(0xffffffffu, (int)bad, o) != 0;
  }
  const int e = mx > 0.0 ? ilogb(mx) + 1 : 0;   // |v| 2^-e < 1
  if (lane == 0) expo[row] = bad ? I8_NAN_ROW : e;
  const size_t plane = (size_t)plane_rows * Kp;
  int8_t *out = planes + (size_t)row * Kp;
  for (int k4 = lane * 4; k4 < Kp; k4 += 128) {
    uint32_t lo[4], hi[4];
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      const int k = k4 + u;
      const long long q = (k < K && !bad) ? __double2ll_rn(scalbn(v[k], 54 - e)) : 0ll;
      const unsigned long long b = (unsigned long long)q + I8_BIAS;      // bytes of b = digits + 128 (see i8_digits)
      lo[u] = (uint32_t)b;
      hi[u] = (uint32_t)(b >> 32);
    }
#pragma unroll
    for (int s = 0; s < I8_S; ++s)
      *reinterpret_cast<uint32_t *>(out + s * plane + k4) = i8_digits(lo, hi, I8_S - 1 - s);
  }
}

struct I8Params {
  double *Out;            // [rows][ldo] FP64, first row = first row of the chunk
  int64_t ldo;
  const int32_t *ea;      // [rows] row exponents of the chunk
  const int32_t *eb;      // [N] column exponents of E
  int32_t rows;           // rows in this chunk (= plane rows of the A planes)
  int32_t N;              // columns of E / of the output
  int32_t num_k_blocks;   // ceil(K / 128)
};

// grid (column tiles, row blocks); 192 threads: warp 0 TMA, warp 1 MMA, warps 2-5 epilogue (TMEM lane quarter warp % 4)
__global__ void __launch_bounds__(192, 1) i8_rotate_kernel(const __grid_constant__ CUtensorMap tmA,
                                                           const __grid_constant__ CUtensorMap tmB, I8Params p) {
  extern __shared__ uint8_t smem_raw[];
  uint8_t *smem = reinterpret_cast<uint8_t *>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  uint8_t *As = smem;
  uint8_t *Bs = smem + I8_NA * I8_A_TILE;
  uint64_t *a_full = reinterpret_cast<uint64_t *>(Bs + 2 * I8_S * I8_B_TILE);
  uint64_t *a_empty = a_full + I8_NA;
  uint64_t *b_full = a_empty + I8_NA;
  uint64_t *b_empty = b_full + 2;
  uint64_t *accum_bar = b_empty + 2;
  uint32_t *tmem_slot = reinterpret_cast<uint32_t *>(accum_bar + 1);

  const int warp = threadIdx.x >> 5;
  const int lane = threadIdx.x & 31;
  const int j0 = blockIdx.x * I8_BN;
  const int i0 = blockIdx.y * 128;
  const int nkb = p.num_k_blocks;

  if (warp == 0 && lane == 0) {
    tma_prefetch_desc(&tmA);
    tma_prefetch_desc(&tmB);
    for (int s = 0; s < I8_NA; ++s) {
      mbar_init(a_full + s, 1);
      mbar_init(a_empty + s, 1);
    }
    for (int g = 0; g < 2; ++g) {
      mbar_init(b_full + g, 1);
      mbar_init(b_empty + g, 1);
    }
    mbar_init(accum_bar, 1);
    fence_barrier_init();
  }
  if (warp == 2) tmem_alloc(tmem_slot, 512);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = *tmem_slot;

  if (warp == 0) {
    // ===== TMA producer: per K block the 7 digit planes of the E tile (one group barrier), then the 7 of the Y tile
    for (int kb = 0; kb < nkb; ++kb) {
      const int g = kb & 1;
      const int k0 = kb * 128;
      mbar_wait(b_empty + g, ((kb >> 1) & 1) ^ 1);
      if (elect_one()) {
        mbar_expect_tx(b_full + g, I8_S * I8_B_TILE);
#pragma unroll
        for (int t = 0; t < I8_S; ++t) tma_load_2d(Bs + (g * I8_S + t) * I8_B_TILE, &tmB, b_full + g, k0, t * p.N + j0);
      }
      __syncwarp();
      for (int s = 0; s < I8_S; ++s) {
        const int ia = kb * I8_S + s;
        const int slot = ia % I8_NA;
        mbar_wait(a_empty + slot, ((ia / I8_NA) & 1) ^ 1);
        if (elect_one()) {
          mbar_expect_tx(a_full + slot, I8_A_TILE);
          tma_load_2d(As + slot * I8_A_TILE, &tmA, a_full + slot, k0, s * p.rows + i0);
        }
        __syncwarp();
      }
    }
  } else if (warp == 1) {
    // ===== MMA issuer: for s, for t <= 6 - s: acc[s + t] += A_s B_t^T (4 K steps of 32 inside the 128-byte rows)
    constexpr uint32_t idesc = make_idesc_i8(128, I8_BN);
    const uint64_t da0 = make_smem_desc(smem_u32(As), 16, 1024, 2);
    const uint64_t db0 = make_smem_desc(smem_u32(Bs), 16, 1024, 2);
    for (int kb = 0; kb < nkb; ++kb) {
      const int g = kb & 1;
      mbar_wait(b_full + g, (kb >> 1) & 1);
      for (int s = 0; s < I8_S; ++s) {
        const int ia = kb * I8_S + s;
        const int slot = ia % I8_NA;
        mbar_wait(a_full + slot, (ia / I8_NA) & 1);
        tc_fence_after();
        if (elect_one()) {
          const uint64_t da = da0 + (uint32_t)((slot * I8_A_TILE) >> 4);
          for (int t = 0; t < I8_S - s; ++t) {
            const uint64_t db = db0 + (uint32_t)(((g * I8_S + t) * I8_B_TILE) >> 4);
#pragma unroll
            for (int q = 0; q < 4; ++q)
              umma_i8(tmem_base + (uint32_t)((s + t) * I8_BN), da + 2 * q, db + 2 * q, idesc,
                      (kb > 0 || s > 0 || q > 0) ? 1u : 0u);
          }
          umma_commit(a_empty + slot);
          if (s == I8_S - 1) umma_commit(b_empty + g);
        }
        __syncwarp();
      }
    }
    if (elect_one()) umma_commit(accum_bar);
    __syncwarp();
  } else {
    // ===== epilogue: thread = output row (TMEM lane), 8 columns at a time
    const int qd = warp & 3;
    const int r = 32 * qd + lane;
    const int64_t row = (int64_t)i0 + r;
    const bool rok = row < p.rows;
    const int ea = rok ? p.ea[row] : 0;
    double *orow = p.Out + row * p.ldo;
    mbar_wait(accum_bar, 0);
    tc_fence_after();
#pragma unroll 1
    for (int c0 = 0; c0 < I8_BN; c0 += 8) {
      uint32_t a[I8_S][8];
#pragma unroll
      for (int d = 0; d < I8_S; ++d) tmem_ld_32x8(tmem_base + ((uint32_t)(32 * qd) << 16) + (uint32_t)(d * I8_BN + c0), a[d]);
      tmem_ld_wait();
#pragma unroll
      for (int u = 0; u < 8; ++u) {
        const int j = j0 + c0 + u;
        if (rok && j < p.N) {
          double v = (double)(int32_t)a[I8_S - 1][u];
#pragma unroll
          for (int d = I8_S - 2; d >= 0; --d) v = fma(v, 0.00390625, (double)(int32_t)a[d][u]);
          const int eb = p.eb[j];
          const bool nan = ea == I8_NAN_ROW || eb == I8_NAN_ROW;
          orow[j] = nan ? __longlong_as_double(0x7ff8000000000000ll) : scalbn(v, ea + eb - 12);
        }
      }
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 2) tmem_dealloc(tmem_base, 512);
}

// ------------------------------------------------------------------------------------------------ Gram products
// H = Y^T Z (contraction over the m rows) with the same digit split, per-COLUMN scales (a column of Y / Z is a row of
// the K-major operand Y^T / Z^T), transposed digit planes planes[s][column][row], and INT32 accumulators flushed into
// FP64 registers every I8_FLUSH K blocks (7 * 16384 * 2^14 < 2^31).
constexpr int I8_FLUSH = 128;           // K blocks of 128 rows between two flushes

struct I8Maps { CUtensorMap m[I8_S]; };
struct I8Planes { int8_t *p[I8_S]; };

// mx[j] = max_i |V[i][j]| as a bit pattern (non-negative doubles order like integers; NaN / inf give >= 0x7ff0...)
__global__ void __launch_bounds__(256) i8_colmax_kernel(const double *__restrict__ V, int64_t ld, int64_t rows, int32_t cols,
                                                        int64_t rows_per_cta, unsigned long long *mx) {
  const int64_t r0 = blockIdx.x * rows_per_cta;
  const int64_t r1 = min(rows, r0 + rows_per_cta);
  for (int j = threadIdx.x; j < cols; j += blockDim.x) {
    unsigned long long best = 0ull;
    for (int64_t i = r0; i < r1; ++i) best = max(best, (unsigned long long)__double_as_longlong(fabs(V[i * ld + j])));
    atomicMax(mx + j, best);
  }
}

// Transposed digit planes of the rows [r0, r0 + rows) of V ([.][cols], pitch ld): planes.p[s][col * Rp + (row - r0)].
// Block = 128 rows x 32 columns through a padded shared tile; rows beyond the chunk are written as zeros up to Rp.
__global__ void __launch_bounds__(256) i8_slice_t_kernel(const double *__restrict__ V, int64_t ld, int64_t r0, int64_t rows,
                                                         int32_t cols, int64_t Rp, const unsigned long long *__restrict__ mx,
                                                         I8Planes planes, int32_t *__restrict__ expo) {
  __shared__ uint32_t tile[I8_S][32][33];
  const int lane = threadIdx.x & 31;
  const int w = threadIdx.x >> 5;
  const int col = blockIdx.x * 32 + lane;
  const bool cok = col < cols;
  const unsigned long long bits = cok ? mx[col] : 0ull;
  const bool bad = bits >= 0x7ff0000000000000ull;
  const double cm = __longlong_as_double((long long)bits);
  const int e = (cm > 0.0 && !bad) ? ilogb(cm) + 1 : 0;
  if (blockIdx.y == 0 && w == 0 && cok && expo) expo[col] = bad ? I8_NAN_ROW : e;
#pragma unroll 2
  for (int i = 0; i < 4; ++i) {
    const int rl = 4 * (w + 8 * i);                        // this thread: rows rl .. rl+3 of its column
    uint32_t lo[4], hi[4];
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      const int64_t r = (int64_t)blockIdx.y * 128 + rl + u;
      const long long q = (cok && !bad && r < rows) ? __double2ll_rn(scalbn(V[(r0 + r) * ld + col], 54 - e)) : 0ll;
      const unsigned long long b = (unsigned long long)q + I8_BIAS;
      lo[u] = (uint32_t)b;
      hi[u] = (uint32_t)(b >> 32);
    }
#pragma unroll
    for (int s = 0; s < I8_S; ++s) tile[s][lane][rl >> 2] = i8_digits(lo, hi, I8_S - 1 - s);
  }
  __syncthreads();
  const int64_t roff = (int64_t)blockIdx.y * 128 + lane * 4;
  for (int idx = w; idx < I8_S * 32; idx += 8) {
    const int s = idx >> 5, c = idx & 31;
    const int cg = blockIdx.x * 32 + c;
    if (cg < cols && roff < Rp) *reinterpret_cast<uint32_t *>(planes.p[s] + (size_t)cg * Rp + roff) = tile[s][c][lane];
  }
}

struct I8GramParams {
  double *Hpart;          // [KS][Nz][N] FP64 partial sums (unscaled), element (ks, b, a)
  int32_t N;              // columns of Y (M side, a)
  int32_t Nz;             // columns of Z in this slab (N side, b)
  int32_t zc0;            // global column of Z's first column: only tiles with rows a >= zc0 + b are formed
  int32_t num_k_blocks;   // ceil(rows / 128) of this row chunk
  int32_t accumulate;     // add to Hpart (row chunks after the first)
};

// grid (b tiles of 64, a tiles of 128, K splits); same warp roles as i8_rotate_kernel
__global__ void __launch_bounds__(192, 1) i8_gram_kernel(const __grid_constant__ I8Maps mapsA, const __grid_constant__ I8Maps mapsB,
                                                         I8GramParams p) {
  const int b0 = blockIdx.x * I8_BN;
  const int a0 = blockIdx.y * 128;
  if (a0 + 127 < p.zc0 + b0) return;          // tile entirely above the diagonal: never read
  extern __shared__ uint8_t smem_raw[];
  uint8_t *smem = reinterpret_cast<uint8_t *>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  uint8_t *As = smem;
  uint8_t *Bs = smem + I8_NA * I8_A_TILE;
  uint64_t *a_full = reinterpret_cast<uint64_t *>(Bs + 2 * I8_S * I8_B_TILE);
  uint64_t *a_empty = a_full + I8_NA;
  uint64_t *b_full = a_empty + I8_NA;
  uint64_t *b_empty = b_full + 2;
  uint64_t *accum_bar = b_empty + 2;
  uint64_t *drained_bar = accum_bar + 1;
  uint32_t *tmem_slot = reinterpret_cast<uint32_t *>(drained_bar + 1);

  const int warp = threadIdx.x >> 5;
  const int lane = threadIdx.x & 31;
  const int ks = gridDim.z;
  const int kb0 = (int)((int64_t)p.num_k_blocks * blockIdx.z / ks);
  const int nk = (int)((int64_t)p.num_k_blocks * (blockIdx.z + 1) / ks) - kb0;

  if (warp == 0 && lane == 0) {
    for (int s = 0; s < I8_S; ++s) {
      tma_prefetch_desc(&mapsA.m[s]);
      tma_prefetch_desc(&mapsB.m[s]);
    }
    for (int s = 0; s < I8_NA; ++s) {
      mbar_init(a_full + s, 1);
      mbar_init(a_empty + s, 1);
    }
    for (int g = 0; g < 2; ++g) {
      mbar_init(b_full + g, 1);
      mbar_init(b_empty + g, 1);
    }
    mbar_init(accum_bar, 1);
    mbar_init(drained_bar, 4);
    fence_barrier_init();
  }
  if (warp == 2) tmem_alloc(tmem_slot, 512);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = *tmem_slot;

  if (warp == 0) {
    for (int c = 0; c < nk; ++c) {
      const int g = c & 1;
      const int k0 = (kb0 + c) * 128;
      mbar_wait(b_empty + g, ((c >> 1) & 1) ^ 1);
      if (elect_one()) {
        mbar_expect_tx(b_full + g, I8_S * I8_B_TILE);
#pragma unroll
        for (int t = 0; t < I8_S; ++t) tma_load_2d(Bs + (g * I8_S + t) * I8_B_TILE, &mapsB.m[t], b_full + g, k0, b0);
      }
      __syncwarp();
      for (int s = 0; s < I8_S; ++s) {
        const int ia = c * I8_S + s;
        const int slot = ia % I8_NA;
        mbar_wait(a_empty + slot, ((ia / I8_NA) & 1) ^ 1);
        if (elect_one()) {
          mbar_expect_tx(a_full + slot, I8_A_TILE);
          tma_load_2d(As + slot * I8_A_TILE, &mapsA.m[s], a_full + slot, k0, a0);
        }
        __syncwarp();
      }
    }
  } else if (warp == 1) {
    constexpr uint32_t idesc = make_idesc_i8(128, I8_BN);
    const uint64_t da0 = make_smem_desc(smem_u32(As), 16, 1024, 2);
    const uint64_t db0 = make_smem_desc(smem_u32(Bs), 16, 1024, 2);
    for (int c = 0; c < nk; ++c) {
      const int g = c & 1;
      const int cr = c % I8_FLUSH;             // position inside the flush round
      if (c > 0 && cr == 0) {                  // the epilogue has read the accumulators of the previous round
        mbar_wait(drained_bar, ((c / I8_FLUSH) - 1) & 1);
        tc_fence_after();
      }
      mbar_wait(b_full + g, (c >> 1) & 1);
      for (int s = 0; s < I8_S; ++s) {
        const int ia = c * I8_S + s;
        const int slot = ia % I8_NA;
        mbar_wait(a_full + slot, (ia / I8_NA) & 1);
        tc_fence_after();
        if (elect_one()) {
          const uint64_t da = da0 + (uint32_t)((slot * I8_A_TILE) >> 4);
          for (int t = 0; t < I8_S - s; ++t) {
            const uint64_t db = db0 + (uint32_t)(((g * I8_S + t) * I8_B_TILE) >> 4);
#pragma unroll
            for (int q = 0; q < 4; ++q)
              umma_i8(tmem_base + (uint32_t)((s + t) * I8_BN), da + 2 * q, db + 2 * q, idesc,
                      (cr > 0 || s > 0 || q > 0) ? 1u : 0u);
          }
          umma_commit(a_empty + slot);
          if (s == I8_S - 1) {
            umma_commit(b_empty + g);
            if (cr == I8_FLUSH - 1 || c == nk - 1) umma_commit(accum_bar);
          }
        }
        __syncwarp();
      }
    }
  } else {
    const int qd = warp & 3;
    const int r = 32 * qd + lane;
    double acc[I8_BN];
#pragma unroll
    for (int u = 0; u < I8_BN; ++u) acc[u] = 0.0;
    const int rounds = (nk + I8_FLUSH - 1) / I8_FLUSH;
    for (int rd = 0; rd < rounds; ++rd) {
      mbar_wait(accum_bar, rd & 1);
      tc_fence_after();
#pragma unroll
      for (int c0 = 0; c0 < I8_BN; c0 += 8) {
        uint32_t a[I8_S][8];
#pragma unroll
        for (int d = 0; d < I8_S; ++d) tmem_ld_32x8(tmem_base + ((uint32_t)(32 * qd) << 16) + (uint32_t)(d * I8_BN + c0), a[d]);
        tmem_ld_wait();
#pragma unroll
        for (int u = 0; u < 8; ++u) {
          double v = (double)(int32_t)a[I8_S - 1][u];
#pragma unroll
          for (int d = I8_S - 2; d >= 0; --d) v = fma(v, 0.00390625, (double)(int32_t)a[d][u]);
          acc[c0 + u] += v;
        }
      }
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(drained_bar);
    }
    const int a = a0 + r;
    if (a < p.N) {
#pragma unroll
      for (int u = 0; u < I8_BN; ++u) {
        const int b = b0 + u;
        if (b < p.Nz) {
          double *dst = p.Hpart + ((size_t)blockIdx.z * p.Nz + b) * p.N + a;
          *dst = p.accumulate ? *dst + acc[u] : acc[u];
        }
      }
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 2) tmem_dealloc(tmem_base, 512);
}

// H(a, zc0 + b) = 2^(ea_a + eb_b - 12) sum_ks Hpart[ks][b][a] for the lower triangle a >= zc0 + b (column-major H).
// w2 > 0: the Nz columns are two slabs of w2 columns side by side, the second one going to H2.
__global__ void __launch_bounds__(256) i8_gram_finish_kernel(const double *__restrict__ Hpart, int32_t KS, int32_t N, int32_t Nz,
                                                             int32_t zc0, int32_t w2, const int32_t *__restrict__ ea,
                                                             const int32_t *__restrict__ eb, double *__restrict__ H,
                                                             double *__restrict__ H2) {
  const int b = blockIdx.y;
  const int eb_ = eb[b];
  const int bb = (w2 > 0 && b >= w2) ? b - w2 : b;
  double *Hd = (w2 > 0 && b >= w2) ? H2 : H;
  for (int a = blockIdx.x * blockDim.x + threadIdx.x; a < N; a += gridDim.x * blockDim.x) {
    if (a < zc0 + bb) continue;
    double v = 0.0;
    for (int k = 0; k < KS; ++k) v += Hpart[((size_t)k * Nz + b) * N + a];
    const int ea_ = ea[a];
    const bool nan = ea_ == I8_NAN_ROW || eb_ == I8_NAN_ROW;
    Hd[(size_t)(zc0 + bb) * N + a] = nan ? __longlong_as_double(0x7ff8000000000000ll) : scalbn(v, ea_ + eb_ - 12);
  }
}

// ------------------------------------------------------------------------------------------------ N_mma = 128, two passes
// The 128 x 64 x 32 MMA of the kernels above is operand-fetch bound (~80 cycles for 32 cycles of math).  With 128
// output columns an MMA costs ~96 cycles for twice the work, but only 4 accumulators fit the 512 TMEM columns, so the
// anti-diagonals are formed in two passes over K: pass 0 = d 0..3 (10 digit pairs), pass 1 = d 4..6 (18 pairs).  After
// each pass the 8 epilogue warps drain the accumulators into FP64 registers (64 columns per thread; the passes and, for
// the Gram products, the flush rounds add up there; one store at the end), and the MMA warp waits for the drain.  Inside a K block the planes are consumed as a sliding window:
// for s = 0..dhi: acc[s+t-dlo] += A_s B_t^T for t = dhi-s .. max(dlo-s, 0); A_s and B_(dhi-s) are dead after step s, so
// both operands stream through in-order rings (A ascending s, B descending t) of 6 x 16 KB each.
constexpr int I8W_BN = 128;
constexpr int I8W_TILE = 128 * 128;
constexpr int I8W_SLOTS = 6;
constexpr int I8W_SMEM = 2 * I8W_SLOTS * I8W_TILE + 1024 /*align*/ + 512 /*barriers*/;

struct I8WParams {
  int32_t MA, NB;          // valid extents of the M side (rows of the chunk / columns of Y) and of the N side
  int32_t num_k_blocks;
  // rotation (MODE 0)
  double *Out;
  int64_t ldo;
  const int32_t *ea, *eb;
  // Gram (MODE 1)
  double *Hpart;           // [KS][NB][MA]
  int32_t zc0;             // tiles with a0 + 127 < zc0 + (packed ? 0 : b0) are skipped
  int32_t packed;          // N side = several column slabs side by side (all at global column zc0)
  int32_t accumulate;      // the first drain adds to Hpart as well (row chunks after the first)
  int32_t debug_mode;      // -DRCHFSI_PROBES builds: 1 = no TMA loads (MMA rate), 2 = no MMAs (operand-stream rate)
};

// one drain of the accumulators of a pass into the thread's FP64 registers: NACC = 4 (anti-diagonals 0..3) or 3 (4..6,
// weight 2^-32); the thread owns TMEM lane 32 qd + lane and the 64 columns of its half
template <int NACC>
__device__ __forceinline__ void i8w_drain(double (&acc)[64], uint32_t tmem_base, int qd, int half) {
#pragma unroll
  for (int c0 = 0; c0 < 64; c0 += 8) {
    uint32_t v[NACC][8];
#pragma unroll
    for (int i = 0; i < NACC; ++i)
      tmem_ld_32x8(tmem_base + ((uint32_t)(32 * qd) << 16) + (uint32_t)(i * I8W_BN + half * 64 + c0), v[i]);
    tmem_ld_wait();
#pragma unroll
    for (int u = 0; u < 8; ++u) {
      double x = (double)(int32_t)v[NACC - 1][u];
#pragma unroll
      for (int i = NACC - 2; i >= 0; --i) x = fma(x, 0.00390625, (double)(int32_t)v[i][u]);
      acc[c0 + u] = (NACC == 3) ? fma(x, 2.3283064365386963e-10, acc[c0 + u]) : acc[c0 + u] + x;   // 2^-32
    }
  }
}

template <int MODE>
__global__ void __launch_bounds__(320, 1) i8w_kernel(const __grid_constant__ I8Maps mapsA, const __grid_constant__ I8Maps mapsB,
                                                     I8WParams p) {
  const int b0 = blockIdx.x * I8W_BN;
  const int a0 = blockIdx.y * 128;
  if (MODE == 1 && a0 + 127 < p.zc0 + (p.packed ? 0 : b0)) return;
  extern __shared__ uint8_t smem_raw[];
  uint8_t *smem = reinterpret_cast<uint8_t *>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  uint8_t *As = smem;
  uint8_t *Bs = smem + I8W_SLOTS * I8W_TILE;
  uint64_t *a_full = reinterpret_cast<uint64_t *>(Bs + I8W_SLOTS * I8W_TILE);
  uint64_t *a_empty = a_full + I8W_SLOTS;
  uint64_t *b_full = a_empty + I8W_SLOTS;
  uint64_t *b_empty = b_full + I8W_SLOTS;
  uint64_t *accum_bar = b_empty + I8W_SLOTS;
  uint64_t *drained_bar = accum_bar + 1;
  uint32_t *tmem_slot = reinterpret_cast<uint32_t *>(drained_bar + 1);

  const int warp = threadIdx.x >> 5;
  const int lane = threadIdx.x & 31;
  const int ks = gridDim.z;
  const int kb0 = (int)((int64_t)p.num_k_blocks * blockIdx.z / ks);
  const int nk = (int)((int64_t)p.num_k_blocks * (blockIdx.z + 1) / ks) - kb0;
  const int round_len = MODE == 1 ? I8_FLUSH : nk;                   // K blocks between two drains of one pass
  const int rounds = nk > 0 ? (nk + round_len - 1) / round_len : 0;

  if (warp == 0 && lane == 0) {
    for (int s = 0; s < I8_S; ++s) {
      tma_prefetch_desc(&mapsA.m[s]);
      tma_prefetch_desc(&mapsB.m[s]);
    }
    for (int s = 0; s < I8W_SLOTS; ++s) {
      mbar_init(a_full + s, 1);
      mbar_init(a_empty + s, 1);
      mbar_init(b_full + s, 1);
      mbar_init(b_empty + s, 1);
    }
    mbar_init(accum_bar, 1);
    mbar_init(drained_bar, 8);
    fence_barrier_init();
  }
  if (warp == 2) tmem_alloc(tmem_slot, 512);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = *tmem_slot;

  if (warp == 0) {
    // ===== TMA producer: tiles in the order the MMA loop first needs them
    int it = 0;                                  // tiles issued so far on each ring (both rings advance together)
    for (int rd = 0; rd < rounds; ++rd) {
      const int c_lo = rd * round_len, c_hi = min(nk, c_lo + round_len);
      for (int pass = 0; pass < 2; ++pass) {
        const int dlo = pass ? 4 : 0, dhi = pass ? 6 : 3;
        for (int c = c_lo; c < c_hi; ++c) {
          const int k0 = (kb0 + c) * 128;
          for (int s = 0; s <= dhi; ++s) {
            // B planes first needed at step s: t = dhi .. dlo at s = 0, t = dlo - s afterwards; ring position dhi - t
            const int t_first = s == 0 ? dhi : dlo - s, t_last = s == 0 ? dlo : dlo - s;
            for (int t = t_first; t >= t_last && t >= 0; --t) {
              const int ib = it + (dhi - t);
              const int slot = ib % I8W_SLOTS;
              mbar_wait(b_empty + slot, ((ib / I8W_SLOTS) & 1) ^ 1);
              if (elect_one()) {
                if (PROBE(p.debug_mode, 1)) {
                  mbar_arrive(b_full + slot);
                } else {
                  mbar_expect_tx(b_full + slot, I8W_TILE);
                  tma_load_2d(Bs + slot * I8W_TILE, &mapsB.m[t], b_full + slot, k0, b0);
                }
              }
              __syncwarp();
            }
            const int ia = it + s;
            const int slot = ia % I8W_SLOTS;
            mbar_wait(a_empty + slot, ((ia / I8W_SLOTS) & 1) ^ 1);
            if (elect_one()) {
              if (PROBE(p.debug_mode, 1)) {
                mbar_arrive(a_full + slot);
              } else {
                mbar_expect_tx(a_full + slot, I8W_TILE);
                tma_load_2d(As + slot * I8W_TILE, &mapsA.m[s], a_full + slot, k0, a0);
              }
            }
            __syncwarp();
          }
          it += dhi + 1;
        }
      }
    }
  } else if (warp == 1) {
    // ===== MMA issuer
    constexpr uint32_t idesc = make_idesc_i8(128, I8W_BN);
    const uint64_t da0 = make_smem_desc(smem_u32(As), 16, 1024, 2);
    const uint64_t db0 = make_smem_desc(smem_u32(Bs), 16, 1024, 2);
    int it = 0, drains = 0;
    for (int rd = 0; rd < rounds; ++rd) {
      const int c_lo = rd * round_len, c_hi = min(nk, c_lo + round_len);
      for (int pass = 0; pass < 2; ++pass) {
        const int dlo = pass ? 4 : 0, dhi = pass ? 6 : 3;
        if (drains > 0) {                        // the epilogue has read the accumulators of the previous pass
          mbar_wait(drained_bar, (drains - 1) & 1);
          tc_fence_after();
        }
        for (int c = c_lo; c < c_hi; ++c) {
          for (int s = 0; s <= dhi; ++s) {
            const int t_first = s == 0 ? dhi : dlo - s, t_last = s == 0 ? dlo : dlo - s;
            for (int t = t_first; t >= t_last && t >= 0; --t) {
              const int ib = it + (dhi - t);
              mbar_wait(b_full + ib % I8W_SLOTS, (ib / I8W_SLOTS) & 1);
            }
            const int ia = it + s;
            mbar_wait(a_full + ia % I8W_SLOTS, (ia / I8W_SLOTS) & 1);
            tc_fence_after();
            if (elect_one()) {
              const uint64_t da = da0 + (uint32_t)(((ia % I8W_SLOTS) * I8W_TILE) >> 4);
              const int t_hi = dhi - s, t_lo = dlo - s > 0 ? dlo - s : 0;
              for (int t = t_hi; t >= t_lo; --t) {
                if (PROBE(p.debug_mode, 2)) break;
                const int ib = it + (dhi - t);
                const uint64_t db = db0 + (uint32_t)(((ib % I8W_SLOTS) * I8W_TILE) >> 4);
#pragma unroll
                for (int q = 0; q < 4; ++q)
                  umma_i8(tmem_base + (uint32_t)((s + t - dlo) * I8W_BN), da + 2 * q, db + 2 * q, idesc,
                          (c > c_lo || s > 0 || q > 0) ? 1u : 0u);
              }
              umma_commit(a_empty + ia % I8W_SLOTS);
              umma_commit(b_empty + (it + s) % I8W_SLOTS);          // plane dhi - s: its last use
              if (s == dhi && c == c_hi - 1) umma_commit(accum_bar);
            }
            __syncwarp();
          }
          it += dhi + 1;
        }
        ++drains;
      }
    }
  } else {
    // ===== epilogue (8 warps): thread = accumulator row (TMEM lane 32 (warp % 4) + lane) x one 64-column half; the
    // passes (and, for the Gram products, the flush rounds) add up in FP64 registers, one store at the end
    const int qd = warp & 3;
    const int half = (warp - 2) >> 2;
    const int a = a0 + 32 * qd + lane;
    const bool aok = a < p.MA;
    double acc[64];
#pragma unroll
    for (int u = 0; u < 64; ++u) acc[u] = 0.0;
    int drains = 0;
    for (int rd = 0; rd < rounds; ++rd) {
      for (int pass = 0; pass < 2; ++pass) {
        mbar_wait(accum_bar, drains & 1);
        tc_fence_after();
        if (pass == 0) i8w_drain<4>(acc, tmem_base, qd, half);
        else i8w_drain<3>(acc, tmem_base, qd, half);
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(drained_bar);
        ++drains;
      }
    }
    const int bh = b0 + half * 64;
    if (aok) {
      if (MODE == 0) {
        const int ea = p.ea[a];
        double *__restrict__ orow = p.Out + (int64_t)a * p.ldo;
#pragma unroll
        for (int c0 = 0; c0 < 64; c0 += 8) {
          int eb[8];
#pragma unroll
          for (int u = 0; u < 8; ++u) eb[u] = (bh + c0 + u < p.NB) ? __ldg(p.eb + bh + c0 + u) : 0;
#pragma unroll
          for (int u = 0; u < 8; ++u) {
            const int b = bh + c0 + u;
            if (b < p.NB)
              orow[b] = (ea == I8_NAN_ROW || eb[u] == I8_NAN_ROW) ? __longlong_as_double(0x7ff8000000000000ll)
                                                                  : scalbn(acc[c0 + u], ea + eb[u] - 12);
          }
        }
      } else {
        double *__restrict__ hp = p.Hpart + ((size_t)blockIdx.z * p.NB) * p.MA + a;
#pragma unroll
        for (int c0 = 0; c0 < 64; c0 += 8) {
          double old[8];
#pragma unroll
          for (int u = 0; u < 8; ++u) old[u] = (p.accumulate && bh + c0 + u < p.NB) ? hp[(size_t)(bh + c0 + u) * p.MA] : 0.0;
#pragma unroll
          for (int u = 0; u < 8; ++u)
            if (bh + c0 + u < p.NB) hp[(size_t)(bh + c0 + u) * p.MA] = old[u] + acc[c0 + u];
        }
      }
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 2) tmem_dealloc(tmem_base, 512);
}

}  // namespace

// scratch the two products need at least (one 128-row chunk of digit planes): tiny problems fall back to dgemm
bool rr_i8_scratch_ok(const rchfsi_ctx *h, size_t bytes) {
  const size_t Kp = ((size_t)h->N + 15) / 16 * 16;
  return bytes >= (size_t)2 * I8_S * h->N * 128 + 8192 && bytes >= ((size_t)I8_S * Kp + 4) * 128 + 4096;
}

bool rotate_i8_supported(const rchfsi_ctx *h) {
  if (h->knobs.rr_split == 0) return false;
  if (h->N > 16384) return false;                         // INT32 exactness: 7 N 2^14 < 2^31
  return true;   // every size: cuBLAS dgemm stays behind RCHFSI_RR_SPLIT=0 as the reference the tests compare with
}

size_t rotate_i8_fixed_bytes(int32_t N) {
  const size_t Kp = ((size_t)N + 15) / 16 * 16;
  return (size_t)I8_S * N * Kp + 4 * (size_t)N + 1024;
}

namespace {

bool wide(const rchfsi_ctx *h) { return h->knobs.rr_i8_bn != 64; }   // N_mma = 128 two-pass kernel (default) or 64

bool plane_maps(rchfsi_ctx *h, I8Maps *maps, const I8Planes &pl, int64_t rows, int64_t K, uint32_t box_rows) {
  for (int s = 0; s < I8_S; ++s)
    if (!get_tmap_2d(h, &maps->m[s], pl.p[s], 1, false, (uint64_t)rows, (uint64_t)K, (uint64_t)K, 128, box_rows)) return false;
  return true;
}

}  // namespace

// Out[r][:] = In[r][:] E for r < rows (E column-major N x N); Out may be In.  `scratch` holds the digit planes and
// exponents of one row chunk: the more rows fit, the fewer chunk launches.
rchfsi_status rotate_i8(rchfsi_ctx *h, const double *In, int64_t rows, const double *E, double *Out, void *scratch,
                        size_t scratch_bytes) {
  const int32_t N = h->N;
  const int32_t Kp = (N + 15) / 16 * 16;
  if (!h->i8_E) RCHFSI_TRY(dev_alloc(h, &h->i8_E, rotate_i8_fixed_bytes(h->N_cap)));
  int8_t *Eplanes = reinterpret_cast<int8_t *>(h->i8_E);
  int32_t *eb = reinterpret_cast<int32_t *>(Eplanes + ((size_t)I8_S * N * Kp + 255) / 256 * 256);
  const size_t per_row = (size_t)I8_S * Kp + 4;
  int64_t R = (int64_t)((scratch_bytes > 4096 ? scratch_bytes - 4096 : 0) / per_row);
  R = std::min<int64_t>(R, rows);
  if (h->knobs.rr_i8_rows > 0) R = std::min<int64_t>(R, h->knobs.rr_i8_rows);
  if (R >= 128) R = R / 128 * 128;
  R = std::min<int64_t>({R, (int64_t)0x7fffff00 / I8_S, (int64_t)65535 * 128});   // TMA row coordinates, grid.y
  if (R < 1) { h->err = "rotate_i8: scratch too small"; return RCHFSI_EINVAL; }
  int8_t *Aplanes = reinterpret_cast<int8_t *>(scratch);
  int32_t *ea = reinterpret_cast<int32_t *>(Aplanes + ((size_t)I8_S * R * Kp + 255) / 256 * 256);
  cudaStream_t st = h->stream;
  // digit planes of the columns of E (column-major: column j is contiguous, i.e. a "row" of the slicing kernel)
  i8_slice_kernel<<<(unsigned)cdiv(N, 8), 256, 0, st>>>(E, N, N, N, Kp, Eplanes, N, eb);
  LAUNCH_CHECK(h);
  if (wide(h)) {
    RCHFSI_TRY(ensure_func_smem(h, (const void *)i8w_kernel<0>, I8W_SMEM));
    I8Planes pe;
    for (int s = 0; s < I8_S; ++s) pe.p[s] = Eplanes + (size_t)s * N * Kp;
    I8Maps mb;
    if (!plane_maps(h, &mb, pe, N, Kp, 128)) { h->err = "rotate_i8: cuTensorMapEncodeTiled failed (E planes)"; return RCHFSI_ECUDA; }
    for (int64_t r0 = 0; r0 < rows; r0 += R) {
      const int64_t rc = std::min<int64_t>(R, rows - r0);
      i8_slice_kernel<<<(unsigned)cdiv(rc, 8), 256, 0, st>>>(In + (size_t)r0 * N, N, rc, N, Kp, Aplanes, rc, ea);
      LAUNCH_CHECK(h);
      I8Planes pa;
      for (int s = 0; s < I8_S; ++s) pa.p[s] = Aplanes + (size_t)s * rc * Kp;
      I8Maps ma;
      if (!plane_maps(h, &ma, pa, rc, Kp, 128)) { h->err = "rotate_i8: cuTensorMapEncodeTiled failed (Y planes)"; return RCHFSI_ECUDA; }
      I8WParams p{};
      p.MA = (int32_t)rc; p.NB = N; p.num_k_blocks = (int32_t)cdiv(N, 128);
      p.Out = Out + (size_t)r0 * N; p.ldo = N; p.ea = ea; p.eb = eb;
      p.debug_mode = h->knobs.tc_debug;
      dim3 grid((unsigned)cdiv(N, I8W_BN), (unsigned)cdiv(rc, 128), 1);
      i8w_kernel<0><<<grid, 320, I8W_SMEM, st>>>(ma, mb, p);
      LAUNCH_CHECK(h);
    }
    return RCHFSI_OK;
  }
  RCHFSI_TRY(ensure_func_smem(h, (const void *)i8_rotate_kernel, I8_SMEM));
  CUtensorMap tmB;
  if (!get_tmap_2d(h, &tmB, Eplanes, 1, false, (uint64_t)I8_S * N, (uint64_t)Kp, (uint64_t)Kp, 128, I8_BN)) {
    h->err = "rotate_i8: cuTensorMapEncodeTiled failed (E planes)";
    return RCHFSI_ECUDA;
  }
  for (int64_t r0 = 0; r0 < rows; r0 += R) {
    const int64_t rc = std::min<int64_t>(R, rows - r0);
    i8_slice_kernel<<<(unsigned)cdiv(rc, 8), 256, 0, st>>>(In + (size_t)r0 * N, N, rc, N, Kp, Aplanes, rc, ea);
    LAUNCH_CHECK(h);
    CUtensorMap tmA;
    if (!get_tmap_2d(h, &tmA, Aplanes, 1, false, (uint64_t)I8_S * rc, (uint64_t)Kp, (uint64_t)Kp, 128, 128)) {
      h->err = "rotate_i8: cuTensorMapEncodeTiled failed (Y planes)";
      return RCHFSI_ECUDA;
    }
    I8Params p{Out + (size_t)r0 * N, N, ea, eb, (int32_t)rc, N, (int32_t)cdiv(N, 128)};
    dim3 grid((unsigned)cdiv(N, I8_BN), (unsigned)cdiv(rc, 128));
    i8_rotate_kernel<<<grid, 192, I8_SMEM, st>>>(tmA, tmB, p);
    LAUNCH_CHECK(h);
  }
  return RCHFSI_OK;
}

// ---------------------------------------------------------------------------------------- Gram products (host side)
bool gram_i8_supported(const rchfsi_ctx *h) {
  if (h->knobs.rr_gram_i8 == 0) return false;
  return h->N <= 16384;                                   // every size (RCHFSI_RR_GRAM_I8=0: cuBLAS dgemm, the tests' reference)
}

bool carve_buf(std::vector<I8Buf> &bufs, size_t bytes, void **out) {
  for (I8Buf &b : bufs) {
    const size_t off = (256 - (reinterpret_cast<uintptr_t>(b.ptr) & 255)) & 255;
    if (b.bytes >= bytes + off) {
      *out = reinterpret_cast<uint8_t *>(b.ptr) + off;
      b.ptr = reinterpret_cast<uint8_t *>(*out) + bytes;
      b.bytes -= bytes + off;
      return true;
    }
  }
  return false;
}

namespace {

// column maxima (bit patterns) and exponents: Y [N], Z [2 N] (two slabs side by side)
rchfsi_status i8_fixed(rchfsi_ctx *h) {
  if (!h->i8_cols) RCHFSI_TRY(dev_alloc(h, &h->i8_cols, (size_t)h->N_cap * 36 + 1024));
  return RCHFSI_OK;
}
unsigned long long *mx_of(rchfsi_ctx *h, int which) { return reinterpret_cast<unsigned long long *>(h->i8_cols) + (size_t)which * h->N_cap; }
int32_t *exp_of(rchfsi_ctx *h, int which) { return reinterpret_cast<int32_t *>(mx_of(h, 3)) + (size_t)which * h->N_cap; }

rchfsi_status colmax(rchfsi_ctx *h, const double *V, int64_t ld, int32_t cols, unsigned long long *mx) {
  RCHFSI_CUDA_CHECK(h, cudaMemsetAsync(mx, 0, sizeof(unsigned long long) * cols, h->stream));
  int64_t ctas = std::min<int64_t>(h->m, 148 * 8);
  const int64_t rows = cdiv(h->m, ctas);
  ctas = cdiv(h->m, rows);
  i8_colmax_kernel<<<(unsigned)ctas, 256, 0, h->stream>>>(V, ld, h->m, cols, rows, mx);
  LAUNCH_CHECK(h);
  return RCHFSI_OK;
}

I8Planes shifted(const I8Planes &pl, size_t bytes) {
  I8Planes o;
  for (int s = 0; s < I8_S; ++s) o.p[s] = pl.p[s] + bytes;
  return o;
}

rchfsi_status slice_t(rchfsi_ctx *h, const double *V, int64_t ld, int64_t r0, int64_t rows, int32_t cols, int64_t Rp,
                      const unsigned long long *mx, const I8Planes &pl, int32_t *expo) {
  const int64_t span = (int64_t)65535 * 128;             // rows one launch covers (grid.y limit)
  for (int64_t off = 0; off < rows; off += span) {
    const int64_t rc = std::min<int64_t>(span, rows - off);
    dim3 grid((unsigned)cdiv(cols, 32), (unsigned)cdiv(rc, 128));
    i8_slice_t_kernel<<<grid, 256, 0, h->stream>>>(V, ld, r0 + off, rc, cols, Rp, mx, shifted(pl, (size_t)off), off == 0 ? expo : nullptr);
    LAUNCH_CHECK(h);
  }
  return RCHFSI_OK;
}


int32_t choose_ks(const rchfsi_ctx *h, int32_t N, int32_t Nz, int32_t zc0, bool packed, int64_t rows) {
  const int bn = wide(h) ? I8W_BN : I8_BN;
  int64_t tiles = 0;
  for (int a0 = 0; a0 < N; a0 += 128)
    for (int b0 = 0; b0 < Nz; b0 += bn) tiles += (a0 + 127 >= zc0 + (packed ? 0 : b0));
  const int64_t nkb = cdiv(rows, 128);
  const int64_t ks = ((int64_t)4 * 148) / std::max<int64_t>(tiles, 1);      // at most 4 full waves of CTAs (one per SM)
  return (int32_t)std::max<int64_t>(1, std::min<int64_t>({ks, (int64_t)32, nkb}));
}

// Hpart (+)= Y^T Z over the K blocks of this row chunk
rchfsi_status gram_launch(rchfsi_ctx *h, const I8Planes &yp, const I8Planes &zp, int64_t Rp, int64_t rows, int32_t Nz, int32_t zc0,
                          bool packed, bool accumulate, int32_t KS) {
  I8Maps ma, mb;
  const bool w = wide(h);
  if (!plane_maps(h, &ma, yp, h->N, Rp, 128) || !plane_maps(h, &mb, zp, Nz, Rp, w ? 128 : I8_BN)) {
    h->err = "gram_i8: cuTensorMapEncodeTiled failed";
    return RCHFSI_ECUDA;
  }
  if (w) {
    RCHFSI_TRY(ensure_func_smem(h, (const void *)i8w_kernel<1>, I8W_SMEM));
    I8WParams p{};
    p.MA = h->N; p.NB = Nz; p.num_k_blocks = (int32_t)cdiv(rows, 128);
    p.Hpart = reinterpret_cast<double *>(h->i8_hpart); p.zc0 = zc0; p.packed = packed ? 1 : 0; p.accumulate = accumulate ? 1 : 0;
    p.debug_mode = h->knobs.tc_debug;
    dim3 grid((unsigned)cdiv(Nz, I8W_BN), (unsigned)cdiv(h->N, 128), (unsigned)KS);
    i8w_kernel<1><<<grid, 320, I8W_SMEM, h->stream>>>(ma, mb, p);
    LAUNCH_CHECK(h);
    return RCHFSI_OK;
  }
  if (packed) { h->err = "gram_i8: the 64-column kernel takes one slab at a time"; return RCHFSI_EINVAL; }
  RCHFSI_TRY(ensure_func_smem(h, (const void *)i8_gram_kernel, I8_SMEM));
  I8GramParams p{reinterpret_cast<double *>(h->i8_hpart), h->N, Nz, zc0, (int32_t)cdiv(rows, 128), accumulate ? 1 : 0};
  dim3 grid((unsigned)cdiv(Nz, I8_BN), (unsigned)cdiv(h->N, 128), (unsigned)KS);
  i8_gram_kernel<<<grid, 192, I8_SMEM, h->stream>>>(ma, mb, p);
  LAUNCH_CHECK(h);
  return RCHFSI_OK;
}

rchfsi_status ensure_hpart(rchfsi_ctx *h, size_t bytes) {
  if (h->i8_hpart_bytes < bytes) {
    RCHFSI_TRY(dev_alloc(h, &h->i8_hpart, bytes));
    h->i8_hpart_bytes = bytes;
  }
  return RCHFSI_OK;
}

rchfsi_status gram_finish(rchfsi_ctx *h, int32_t KS, int32_t Nz, int32_t zc0, int32_t w2, const int32_t *ea, const int32_t *eb,
                          double *H, double *H2) {
  dim3 grid((unsigned)cdiv(h->N, 256), (unsigned)Nz);
  i8_gram_finish_kernel<<<grid, 256, 0, h->stream>>>(reinterpret_cast<const double *>(h->i8_hpart), KS, h->N, Nz, zc0, w2, ea, eb, H, H2);
  LAUNCH_CHECK(h);
  return RCHFSI_OK;
}

}  // namespace

// workspace the INT8 Rayleigh-Ritz products hold beyond the blocks they borrow (planner: automatic choice only)
size_t rr_i8_plan_bytes(int64_t m, int32_t N) {
  if (N > 16384) return 0;
  auto al = [](size_t b) { return (b + 255) / 256 * 256; };
  int64_t tiles = 0;
  for (int a0 = 0; a0 < N; a0 += 128)
    for (int b0 = 0; b0 < N; b0 += I8W_BN) tiles += (a0 + 127 >= b0);
  const int64_t ks = std::max<int64_t>(1, std::min<int64_t>({((int64_t)4 * 148) / std::max<int64_t>(tiles, 1), (int64_t)32, cdiv(m, 128)}));
  return al(rotate_i8_fixed_bytes(N)) + al((size_t)N * 36 + 1024) + al(sizeof(double) * (size_t)ks * N * N);
}

// every buffer the INT8 products of one Rayleigh-Ritz hold themselves (the digit planes live in borrowed blocks)
rchfsi_status rr_i8_preallocate(rchfsi_ctx *h, bool chunked, int32_t cw) {
  if (rotate_i8_supported(h) && !h->i8_E) RCHFSI_TRY(dev_alloc(h, &h->i8_E, rotate_i8_fixed_bytes(h->N_cap)));
  if (gram_i8_supported(h)) {
    RCHFSI_TRY(i8_fixed(h));
    const size_t hp = chunked ? sizeof(double) * (size_t)32 * h->N * 2 * cw
                              : sizeof(double) * (size_t)choose_ks(h, h->N, h->N, 0, false, h->m) * h->N * h->N;
    RCHFSI_TRY(ensure_hpart(h, hp));
  }
  return RCHFSI_OK;
}

// Full-block variant: H_a = Y^T (AY), H_b = Y^T (BY) (BY == NULL: Y^T Y), lower triangles, column-major.  `scratch`
// holds the transposed digit planes of one row chunk of Y and of Z.
rchfsi_status gram_i8_full(rchfsi_ctx *h, const double *Y, const double *AY, const double *BY, double *Ha, double *Hb,
                           void *scratch, size_t scratch_bytes) {
  const int32_t N = h->N;
  const int64_t m = h->m;
  RCHFSI_TRY(i8_fixed(h));
  // rows per chunk: 2 x 7 planes of N x Rp bytes
  int64_t R = (int64_t)((scratch_bytes > 8192 ? scratch_bytes - 8192 : 0) / ((size_t)2 * I8_S * N));
  R = std::min<int64_t>(R / 128 * 128, (m + 127) / 128 * 128);
  if (h->knobs.rr_i8_rows > 0) R = std::min<int64_t>(R, (h->knobs.rr_i8_rows + 127) / 128 * 128);
  if (R < 128) { h->err = "gram_i8: scratch too small"; return RCHFSI_EINVAL; }
  const int64_t Rp = R;
  I8Planes yp, zp;
  uint8_t *base = reinterpret_cast<uint8_t *>(scratch);
  base += (256 - (reinterpret_cast<uintptr_t>(base) & 255)) & 255;
  for (int s = 0; s < I8_S; ++s) {
    yp.p[s] = reinterpret_cast<int8_t *>(base + (size_t)s * N * Rp);
    zp.p[s] = reinterpret_cast<int8_t *>(base + (size_t)(I8_S + s) * N * Rp);
  }
  const int32_t KS = choose_ks(h, N, N, 0, false, R);
  RCHFSI_TRY(ensure_hpart(h, sizeof(double) * (size_t)KS * N * N));
  RCHFSI_TRY(colmax(h, Y, N, N, mx_of(h, 0)));
  for (int prod = 0; prod < 2; ++prod) {
    const double *Z = prod == 0 ? AY : BY;
    const bool same = Z == nullptr;                       // Y^T Y
    if (!same) RCHFSI_TRY(colmax(h, Z, N, N, mx_of(h, 1)));
    for (int64_t r0 = 0; r0 < m; r0 += R) {
      const int64_t rc = std::min<int64_t>(R, m - r0);
      RCHFSI_TRY(slice_t(h, Y, N, r0, rc, N, Rp, mx_of(h, 0), yp, exp_of(h, 0)));
      if (!same) RCHFSI_TRY(slice_t(h, Z, N, r0, rc, N, Rp, mx_of(h, 1), zp, exp_of(h, 1)));
      RCHFSI_TRY(gram_launch(h, yp, same ? yp : zp, Rp, rc, N, 0, false, r0 > 0, KS));
    }
    RCHFSI_TRY(gram_finish(h, KS, N, 0, 0, exp_of(h, 0), same ? exp_of(h, 0) : exp_of(h, 1), prod == 0 ? Ha : Hb, nullptr));
  }
  return RCHFSI_OK;
}

// Column-slab variant (memory-light Rayleigh-Ritz): the transposed planes of ALL rows of Y are built once into the
// caller's buffers (the filter's dead blocks), then every column slab contributes H_a[:, c0:c0+w] = Y^T (A Y_c) and
// H_b[:, c0:c0+w] = Y^T (B Y_c) in ONE launch (the two slabs side by side on the N side: Y's planes are read once).
// Returns false (nothing launched) when the buffers cannot hold the planes.
bool gram_i8_begin(rchfsi_ctx *h, const double *Y, std::vector<I8Buf> &bufs, int32_t max_w, rchfsi_status *st) {
  *st = RCHFSI_OK;
  const int32_t N = h->N;
  const int64_t m = h->m;
  const int64_t Rp = (m + 127) / 128 * 128;
  I8GramState &g = h->i8g;
  g.active = false;
  std::vector<I8Buf> trial = bufs;
  for (int s = 0; s < I8_S; ++s)
    if (!carve_buf(trial, (size_t)N * Rp, reinterpret_cast<void **>(&g.yp[s]))) return false;
  for (int s = 0; s < I8_S; ++s)
    if (!carve_buf(trial, (size_t)2 * max_w * Rp, reinterpret_cast<void **>(&g.zp[s]))) return false;
  bufs = trial;                                           // only a successful placement consumes the caller's buffers
  g.Rp = Rp;
  g.max_w = max_w;
  if ((*st = i8_fixed(h)) != RCHFSI_OK) return false;
  if ((*st = ensure_hpart(h, sizeof(double) * (size_t)32 * N * 2 * max_w)) != RCHFSI_OK) return false;
  if ((*st = colmax(h, Y, N, N, mx_of(h, 0))) != RCHFSI_OK) return false;
  I8Planes yp;
  for (int s = 0; s < I8_S; ++s) yp.p[s] = g.yp[s];
  if ((*st = slice_t(h, Y, N, 0, m, N, Rp, mx_of(h, 0), yp, exp_of(h, 0))) != RCHFSI_OK) return false;
  g.active = true;
  return true;
}

// Z1 = A Y_c, Z2 = B Y_c ([m][w], pitch ldz) or NULL for B = I (the slab of Y itself)
rchfsi_status gram_i8_slab(rchfsi_ctx *h, const double *Y, const double *Z1, const double *Z2, int64_t ldz, int32_t w, int32_t zc0,
                           double *Ha, double *Hb) {
  I8GramState &g = h->i8g;
  if (!g.active || w > g.max_w) { h->err = "gram_i8_slab: no planes"; return RCHFSI_EINVAL; }
  const int64_t m = h->m;
  I8Planes yp, zp;
  for (int s = 0; s < I8_S; ++s) { yp.p[s] = g.yp[s]; zp.p[s] = g.zp[s]; }
  RCHFSI_TRY(colmax(h, Z1, ldz, w, mx_of(h, 1)));
  RCHFSI_TRY(slice_t(h, Z1, ldz, 0, m, w, g.Rp, mx_of(h, 1), zp, exp_of(h, 1)));
  const double *Zb = Z2 ? Z2 : Y + zc0;
  const int64_t ldb = Z2 ? ldz : h->N;
  RCHFSI_TRY(colmax(h, Zb, ldb, w, mx_of(h, 1) + w));
  RCHFSI_TRY(slice_t(h, Zb, ldb, 0, m, w, g.Rp, mx_of(h, 1) + w, shifted(zp, (size_t)w * g.Rp), exp_of(h, 1) + w));
  if (wide(h)) {
    const int32_t KS = choose_ks(h, h->N, 2 * w, zc0, true, m);
    RCHFSI_TRY(gram_launch(h, yp, zp, g.Rp, m, 2 * w, zc0, true, false, KS));
    return gram_finish(h, KS, 2 * w, zc0, w, exp_of(h, 0), exp_of(h, 1), Ha, Hb);
  }
  for (int prod = 0; prod < 2; ++prod) {                  // 64-column kernel: one slab per launch
    const int32_t KS = choose_ks(h, h->N, w, zc0, false, m);
    RCHFSI_TRY(gram_launch(h, yp, prod ? shifted(zp, (size_t)w * g.Rp) : zp, g.Rp, m, w, zc0, false, false, KS));
    RCHFSI_TRY(gram_finish(h, KS, w, zc0, 0, exp_of(h, 0), exp_of(h, 1) + prod * w, prod ? Hb : Ha, nullptr));
  }
  return RCHFSI_OK;
}

}  // namespace rchfsi
