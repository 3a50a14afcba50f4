// mg_fused.cu -- tuned uniform-grid fp32 kernels (placeholder: not yet enabled).
#include "fused.h"
#include "solver.h"

namespace mgb {
bool fused_supported(const mg_solver*) { return false; }
int fused_apply(mg_solver*, const float*, float*) { set_error("fused path not built"); return MG_EINVAL; }
int fused_smooth(mg_solver*, float*, const float*, int) { set_error("fused path not built"); return MG_EINVAL; }
int fused_vcycle(mg_solver*, float*, const float*) { set_error("fused path not built"); return MG_EINVAL; }
void fused_release(mg_solver*) {}
}  // namespace mgb
