// fx_fused.cu -- fused stage kernel (placeholder until the column kernel lands).
#include "fx_internal.h"

bool fx_fused_supported(const FxParams &) { return false; }

int fx_launch_fused_stage(const FxParams &, const double *, const double *, double *, const double *, double,
                          const double *, double, int, cudaStream_t) {
  return fx_fail(FX_ERR_UNSUPPORTED, "fused stage kernel not built");
}
