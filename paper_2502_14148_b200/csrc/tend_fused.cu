// tend_fused.cu — OCN_KERNEL_FUSED: shared-memory x-y tiles + register-sliding z (2.5-D blocking).
// (placeholder translation unit until the fused kernels land: reports "not applicable")
#include "ocn_internal.h"

bool fused_applicable(const ocn_grid *, const ModelDev &, std::string *why) {
  if (why) *why = "fused kernels not built yet";
  return false;
}
int launch_tendencies_fused(const ocn_grid *, const ModelDev &, const FieldsDev &, const void *, const FieldsDev &, cudaStream_t) {
  return ocn_fail(OCN_ERR_UNSUPPORTED, "fused kernels not built yet");
}
