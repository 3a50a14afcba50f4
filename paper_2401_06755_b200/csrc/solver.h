// solver.h -- the mg_solver object behind the C ABI of include/mg.h (product code).
#pragma once
#include <vector>

#include "../../include/mg.h"
#include "common.cuh"

namespace mgb {

struct LevelData {
    int nx = 0, ny = 0, nz = 0;
    double hx = 0, hy = 0, hz = 0;
    size_t n = 0;
    bool uniform = false;
    // device buffers of the solver's dtype.  Level 0: x and b are the caller's (set per call);
    // k (NULL while the coefficient is constant) and tmp are the solver's.  Levels >= 1: all owned.
    void *x = nullptr, *b = nullptr, *k = nullptr, *tmp = nullptr;
    Level<float> Lf;
    Level<double> Ld;
};

}  // namespace mgb

struct mg_solver {
    mg_grid grid{};
    int levels = 0;
    int bc[6] = {0, 0, 0, 0, 0, 0};
    int dtype = MG_F32;
    int device = 0;
    cudaStream_t st = nullptr;
    mg_params p{2, 2, 50, 1, 2.0 / 3.0, 1, 1};
    bool var_k = false;
    int fused = 1;
    std::vector<mgb::LevelData> lv;
    // mixed-precision outer loop (MG_F32 only): fp64 iterate and fine coefficient, fp32 residual / correction
    double* x64 = nullptr;
    double* k64 = nullptr;
    float* r32 = nullptr;
    float* e32 = nullptr;
    // mg_pcg_solve (mg_pcg.cu): fp64 CG vectors b, r, p, q (and z for MG_F64), device scalars
    double* pcg_v[5] = {nullptr, nullptr, nullptr, nullptr, nullptr};
    double* pcg_s = nullptr;
    // host-buffer entry points
    void* hx_dev = nullptr;
    void* hb_dev = nullptr;
    // norms
    double* d_acc = nullptr;
    int* d_ctr = nullptr;     // device-side index of the next residual-history slot (solve-cycle graph)
    double* h_acc = nullptr;  // pinned
    std::vector<double> history;
    std::vector<int> history_cycles;   // V-cycles (iterations) completed when history[i] was taken
    long long launches = 0;
    // per-level instrumentation of mg_vcycle_timed
    bool timing = false;
    std::vector<cudaEvent_t> ev;
    // CUDA-graph replay of recorded launch sequences (a V-cycle, a zero-guess cycle, a whole solve cycle), keyed by the (x, b)
    // pointers and the flavour they were captured with; a small cache, least recently used slot replaced
    struct GraphSlot {
        cudaGraphExec_t exec = nullptr;
        const void* x = nullptr;
        const void* b = nullptr;
        int flavour = 0;
        long long launches = 0;    // kernels inside one replay
        long long used = 0;        // stamp of the last replay
    };
    static constexpr int GRAPH_SLOTS = 6;
    GraphSlot graphs[GRAPH_SLOTS];
    long long graph_clock = 0;
    long long epoch = 0;              // bumped whenever the recorded graphs are dropped (parameters, coefficient kind, fused switch)
    cudaStream_t cap_st = nullptr;    // private stream used only to record graphs
    void* fused_state = nullptr;   // owned by mg_fused.cu
};

namespace mgb {

// Replay `enqueue` (which launches one V-cycle on s->st for the pointer pair (x, b)) from a CUDA graph: recorded once per
// pointer pair on a private stream (the caller's may be the legacy default stream, which cannot be captured), then launched
// on the caller's stream.  mg_set_params / mg_set_coefficient / mg_set_fused drop the recorded graph.
template <class F>
int replay_graph(mg_solver* s, const void* x, const void* b, F&& enqueue, int flavour = 0) {
    mg_solver::GraphSlot* slot = nullptr;
    for (auto& g : s->graphs)
        if (g.exec && g.x == x && g.b == b && g.flavour == flavour) { slot = &g; break; }
    if (!slot) {
        slot = &s->graphs[0];
        for (auto& g : s->graphs) {
            if (!g.exec) { slot = &g; break; }
            if (g.used < slot->used) slot = &g;
        }
        if (slot->exec) { cudaGraphExecDestroy(slot->exec); slot->exec = nullptr; }
        const long long before = s->launches;
        cudaGraph_t graph = nullptr;
        if (!s->cap_st) MGB_CUDA(cudaStreamCreateWithFlags(&s->cap_st, cudaStreamNonBlocking));
        cudaStream_t user_st = s->st;
        MGB_CUDA(cudaStreamBeginCapture(s->cap_st, cudaStreamCaptureModeThreadLocal));
        s->st = s->cap_st;
        const int rc = enqueue();
        s->st = user_st;
        const cudaError_t e = cudaStreamEndCapture(s->cap_st, &graph);
        slot->launches = s->launches - before;
        s->launches = before;
        if (rc) { if (graph) cudaGraphDestroy(graph); return rc; }
        if (e != cudaSuccess) { set_error("graph capture failed: %s", cudaGetErrorString(e)); return MG_ECUDA; }
        const cudaError_t e2 = cudaGraphInstantiate(&slot->exec, graph, 0);
        cudaGraphDestroy(graph);
        if (e2 != cudaSuccess) { slot->exec = nullptr; set_error("graph instantiate failed: %s", cudaGetErrorString(e2)); return MG_ECUDA; }
        slot->x = x; slot->b = b; slot->flavour = flavour;
    }
    slot->used = ++s->graph_clock;
    MGB_CUDA(cudaGraphLaunch(slot->exec, s->st));
    s->launches += slot->launches;
    return 0;
}

}  // namespace mgb
