// Dense tensor-core step (tcgen05 / TMEM / TMA).  Placeholder until the kernel lands: reports
// "not supported" so rchfsi_filter uses the FP32 ALU path.
#include "common.cuh"
namespace rchfsi {
bool dense_tc_supported(const rchfsi_ctx *) { return false; }
rchfsi_status dense_tc_step(rchfsi_ctx *h, const FusedStep &) {
  h->err = "dense tensor-core step not built";
  return RCHFSI_EINVAL;
}
}  // namespace rchfsi
