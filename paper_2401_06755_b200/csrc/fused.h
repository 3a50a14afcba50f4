// fused.h -- interface of the tuned uniform-grid fp32 path (mg_fused.cu) used by mg_api.cu.
#pragma once
struct mg_solver;

namespace mgb {
// true when the solver's grid / dtype are covered by the tuned kernels
bool fused_supported(const mg_solver* s);
// (re)build the per-level data the tuned path derives from the coefficient (1/D of the coarse levels)
int fused_prepare(mg_solver* s);
int fused_smooth(mg_solver* s, float* x, const float* b, int sweeps);
int fused_vcycle(mg_solver* s, float* x, const float* b, int zero_guess = 0);   // 1: x = 0 implied; 2: x holds b / D (mg_fused.cu)
int fused_vcycle_prepare(mg_solver* s);        // state + tabulated coarsest solve: before recording fused_vcycle_enqueue in a graph
int fused_vcycle_enqueue(mg_solver* s, float* x, const float* b, int zero_guess);   // the cycle's launches on s->st, no graph of its own
bool fused_seed_supported(mg_solver* s);
bool fused_residual_supported(mg_solver* s);   // the fine level is a streaming-kernel level
int fused_residual(mg_solver* s, const float* x, const float* b, float* r, double* acc);   // r = b - A x, or A x if b == NULL; ||.||^2 added to *acc
void fused_release(mg_solver* s);
// TMA descriptor of a 3-D fp32 field, box = px x py cells of one z plane, out-of-bounds cells read as 0 (tm: CUtensorMap*)
int make_tmap_f32(void* tm, const float* ptr, int nx, int ny, int nz, int px, int py);
}  // namespace mgb
