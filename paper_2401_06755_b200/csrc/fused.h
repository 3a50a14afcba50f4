// fused.h -- interface of the tuned uniform-grid fp32 path (mg_fused.cu) used by mg_api.cu.
#pragma once
struct mg_solver;

namespace mgb {
// true when the solver's grid / dtype / parameters are covered by the tuned kernels
bool fused_supported(const mg_solver* s);
int fused_apply(mg_solver* s, const float* x, float* y);
int fused_smooth(mg_solver* s, float* x, const float* b, int sweeps);
int fused_vcycle(mg_solver* s, float* x, const float* b);
void fused_release(mg_solver* s);
}  // namespace mgb
