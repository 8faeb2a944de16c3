// rchfsi_residual_static: the residual block and residual norms of Algorithm 1 / 3 without a handle and without any
// allocation, for callers that cannot call cudaMalloc (CUDA graph capture, tight serving loops, harnesses that forbid
// it).  G = A X - B X diag(eps) and r_j = ||A x_j - eps_j B x_j||_2, FP64.
//
// A variant of residual_kernel (elementwise.cu): there every CTA adds its slab's column sums of squares into the
// output with atomicAdd; here every CTA writes its partial sums to a slot of a FILE-SCOPE device array and the last CTA
// to finish (a ticket counter in the same array's header) adds the slots in slot order, so r_j is also bitwise
// reproducible from call to call.  The array is RCHFSI_STATIC_SCRATCH_BYTES per GPU that loads the library, held
// until the process exits.  Every call shares it: calls that overlap on the GPU (two streams, two threads) race.
#include <cuda_runtime.h>
#include <cstdint>
#include <cstdio>
#include <mutex>
#include "rchfsi.h"

namespace {

constexpr int RS_MAX_N = RCHFSI_STATIC_MAX_N;          // widest block
constexpr int RS_SLOTS = 148;                          // CTAs per call = partial-sum slots (one per SM of a B200)
constexpr int RS_HEADER = 32;                          // doubles in front of the slots (256 bytes): [0] = ticket counter
constexpr size_t RS_DOUBLES = RS_HEADER + (size_t)RS_SLOTS * RS_MAX_N;
static_assert(RS_DOUBLES * sizeof(double) == RCHFSI_STATIC_SCRATCH_BYTES, "header and kernel disagree on the scratch size");

// In HOST code this name is a host-side stand-in, not a device address: only cudaGetSymbolAddress gives the pointer a
// kernel can be handed.  Device code below never names it either; it gets the pointer as an argument.
static __device__ __align__(256) double g_residual_scratch[RS_DOUBLES];

constexpr int RS_MAX_DEVICES = 64;
double *g_scratch_ptr[RS_MAX_DEVICES] = {};            // device address of g_residual_scratch, per device
std::mutex g_setup_mutex;
thread_local char g_static_err[320] = "";          // fixed buffer: the error path allocates nothing either

rchfsi_status fail(rchfsi_status st, const char *what, const char *detail = "") {
  snprintf(g_static_err, sizeof(g_static_err), "%s%s", what, detail);
  return st;
}

// Once per device, with that device current: the array's device address, and the ticket counter cleared.
rchfsi_status setup_current_device(double **out) {
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return fail(RCHFSI_ECUDA, "rchfsi_static_setup: cudaGetDevice: ", cudaGetErrorString(e));
  if (dev < 0 || dev >= RS_MAX_DEVICES) return fail(RCHFSI_EINVAL, "rchfsi_static_setup: device ordinal beyond 63");
  std::lock_guard<std::mutex> lock(g_setup_mutex);
  if (!g_scratch_ptr[dev]) {
    double *p = nullptr;
    e = cudaGetSymbolAddress((void **)&p, g_residual_scratch);
    if (e != cudaSuccess || !p)
      return fail(RCHFSI_ECUDA, "rchfsi_static_setup: cudaGetSymbolAddress: ", cudaGetErrorString(e));
    e = cudaMemset(p, 0, RS_HEADER * sizeof(double));       // the ticket counter must start at zero
    if (e != cudaSuccess) return fail(RCHFSI_ECUDA, "rchfsi_static_setup: cudaMemset: ", cudaGetErrorString(e));
    g_scratch_ptr[dev] = p;
  }
  if (out) *out = g_scratch_ptr[dev];
  return RCHFSI_OK;
}

// CTA b owns rows [b*rows_per_cta, ...); thread t owns columns t, t+256, ...  partial[b][j] = sum over the slab of
// G_ij^2.  The last CTA to arrive adds the slots 0..gridDim-1 in that order, writes r_j and re-arms the counter.
__global__ void __launch_bounds__(256) residual_static_kernel(const double *__restrict__ AX, const double *__restrict__ BX,
                                                              const double *__restrict__ ritz, double *__restrict__ G,
                                                              double *__restrict__ resnorm, int64_t m, int32_t N,
                                                              int64_t rows_per_cta, double *scratch) {
  double *partial = scratch + RS_HEADER;
  unsigned int *ticket = reinterpret_cast<unsigned int *>(scratch);
  const int64_t r0 = blockIdx.x * rows_per_cta;
  const int64_t r1 = min(m, r0 + rows_per_cta);
  for (int j = threadIdx.x; j < N; j += blockDim.x) {
    const double lam = ritz[j];
    double s = 0.0;
#pragma unroll 4
    for (int64_t i = r0; i < r1; ++i) {
      const double g = AX[i * N + j] - BX[i * N + j] * lam;
      if (G) G[i * N + j] = g;
      s += g * g;
    }
    partial[(size_t)blockIdx.x * RS_MAX_N + j] = s;
  }
  if (!resnorm) return;
  __shared__ bool last;
  __threadfence();                                   // this CTA's partial sums are visible before its ticket
  __syncthreads();
  if (threadIdx.x == 0) last = atomicAdd(ticket, 1u) == gridDim.x - 1;
  __syncthreads();
  if (!last) return;
  __threadfence();
  for (int j = threadIdx.x; j < N; j += blockDim.x) {
    double s = 0.0;
    for (unsigned b = 0; b < gridDim.x; ++b) s += __ldcg(partial + (size_t)b * RS_MAX_N + j);
    resnorm[j] = sqrt(s);
  }
  if (threadIdx.x == 0) *ticket = 0u;                // the next call on this device starts from zero again
}

}  // namespace

extern "C" {

const char *rchfsi_static_last_error(void) { return g_static_err; }

rchfsi_status rchfsi_static_setup(void) { return setup_current_device(nullptr); }

rchfsi_status rchfsi_residual_static(const double *AX, const double *BX, const double *ritz, int64_t m, int32_t N,
                                     double *G_out, double *resnorm_out, void *stream) {
  if (!AX || !BX || !ritz) return fail(RCHFSI_EINVAL, "rchfsi_residual_static: null input");
  if (!G_out && !resnorm_out) return fail(RCHFSI_EINVAL, "rchfsi_residual_static: no output requested");
  if (m < 1 || N < 1) return fail(RCHFSI_EINVAL, "rchfsi_residual_static: m and N must be positive");
  if (N > RS_MAX_N) {
    char what[64];
    snprintf(what, sizeof(what), "rchfsi_residual_static: N = %d", (int)N);
    return fail(RCHFSI_EINVAL, what, " exceeds RCHFSI_STATIC_MAX_N = 4096 (the static scratch holds 148 x 4096 partial "
                                     "sums); use rchfsi_rayleigh_ritz with a workspace for wider blocks");
  }
  double *scratch = nullptr;
  rchfsi_status st = setup_current_device(&scratch);
  if (st != RCHFSI_OK) return st;
  int64_t ctas = m < RS_SLOTS ? m : RS_SLOTS;
  const int64_t rows = (m + ctas - 1) / ctas;
  ctas = (m + rows - 1) / rows;
  residual_static_kernel<<<(unsigned)ctas, 256, 0, (cudaStream_t)stream>>>(AX, BX, ritz, G_out, resnorm_out, m, N, rows, scratch);
  const cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return fail(RCHFSI_ECUDA, "rchfsi_residual_static: launch: ", cudaGetErrorString(e));
  return RCHFSI_OK;
}

}  // extern "C"
