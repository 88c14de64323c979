// BF16 tcgen05 tensor-core variant of the fused step (placeholder until the UMMA path lands).
#include "dsmc_internal.h"

namespace dsmc {
int build_tc_blob(const dsmc_mlp_desc *, void **, MlpTcDev *out, cudaStream_t) {
  out->H = 0;
  return DSMC_ERR_UNSUPPORTED_SHAPE;
}
int launch_collide_tc(dsmc_ctx *, const StepParams &, const MlpTcDev *) { return DSMC_ERR_UNSUPPORTED_SHAPE; }
int launch_chi_batch_tc(dsmc_ctx *, int64_t, const float *, const float *, float *, float, float, float,
                        const MlpTcDev *) {
  return DSMC_ERR_UNSUPPORTED_SHAPE;
}
}  // namespace dsmc
