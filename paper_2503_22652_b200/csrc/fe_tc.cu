// FE cell-batched tensor-core step.  Placeholder until the kernel lands.
#include "common.cuh"
namespace rchfsi {
bool fe_tc_supported(const rchfsi_ctx *) { return false; }
rchfsi_status fe_tc_step(rchfsi_ctx *h, const FusedStep &) {
  h->err = "FE tensor-core step not built";
  return RCHFSI_EINVAL;
}
}  // namespace rchfsi
