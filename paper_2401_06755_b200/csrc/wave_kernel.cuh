// wave_kernel.cuh -- temporal blocking of the fp32 smoother / transfer passes: several dependent stencil stages of one
// level in ONE launch (north_star "fuses several sweeps temporally per pass"; BASELINE config 4 "temporal blocking of 4
// sweeps per pass").
//
// The grid holds one group of lean_kernel blocks per stage: stage s + 1 follows stage s a few planes behind, tile by tile,
// and reads the iterate stage s has just written while it is still in L2 (126 MB; the band between the two fronts is a few
// planes of three fields).  The coefficient and right-hand-side planes that stage s fetched from HBM are re-read by stage
// s + 1 from L2 as well, so a pass of T stages moves about 12 + 4 T bytes per point through HBM instead of 16 T.
// Scheduling, dependencies and the in-place ping-pong of the iterate are described at WaveCtx in lean_kernel.cuh; the stage
// bodies are the lean_kernel code itself (SWEEP / PRO / RR / SEED), one mode per stage.
#pragma once
#include "lean_kernel.cuh"

namespace mgb {
namespace wk {

constexpr int MAXS = 4;        // stages per launch

struct WStage {
    CUtensorMap tmx, tmk, tmb, tmc;
    lk::LParams P;
    int mode;
};

struct WParams {
    int nstages, nch, gx, gy;
    int* prog;                 // progress flags [nstages][nch][gy][gx], all zero between launches
    int* done;                 // blocks that have finished (the last one clears the flags and this counter)
    int* err;
    WStage st[MAXS];
};

template <int LX, int LY, bool VAR, int MINB>
__global__ void __launch_bounds__(LX * LY, MINB) wave_kernel(const __grid_constant__ WParams W) {
    using C = lk::LCfg<LX, LY, VAR, lk::MODE_PRO, MINB>;      // ring slots sized for the largest mode
    const int stage = blockIdx.z / W.nch, chunk = blockIdx.z - stage * W.nch;
    const WStage& S = W.st[stage];
    const size_t per = (size_t)W.nch * W.gy * W.gx;
    lk::WaveCtx wc;
    wc.dir = (chunk & 1) ? -1 : 1;
    wc.tx = blockIdx.x; wc.ty = blockIdx.y; wc.chunk = chunk;
    wc.gx = W.gx; wc.gy = W.gy; wc.nch = W.nch; wc.zchunk = S.P.zchunk;
    wc.my_prog = stage + 1 < W.nstages ? W.prog + stage * per + ((size_t)chunk * W.gy + blockIdx.y) * W.gx + blockIdx.x : nullptr;
    wc.dep_prog = stage > 0 ? W.prog + (stage - 1) * per : nullptr;
    wc.err = W.err;
    switch (S.mode) {
        case lk::MODE_SWEEP: lk::lean_body<C, lk::MODE_SWEEP, true>(S.tmx, S.tmk, S.tmb, S.tmc, S.P, blockIdx.x, blockIdx.y, chunk, wc); break;
        case lk::MODE_PRO: lk::lean_body<C, lk::MODE_PRO, true>(S.tmx, S.tmk, S.tmb, S.tmc, S.P, blockIdx.x, blockIdx.y, chunk, wc); break;
        case lk::MODE_RR: lk::lean_body<C, lk::MODE_RR, true>(S.tmx, S.tmk, S.tmb, S.tmc, S.P, blockIdx.x, blockIdx.y, chunk, wc); break;
        default: lk::lean_body<C, lk::MODE_SEED, true>(S.tmx, S.tmk, S.tmb, S.tmc, S.P, blockIdx.x, blockIdx.y, chunk, wc); break;
    }
    // the last block to finish leaves the flags cleared for the next launch (launches are ordered by the stream)
    __shared__ int last;
    __syncthreads();
    if (threadIdx.x == 0) {
        __threadfence();
        const int total = gridDim.x * gridDim.y * gridDim.z;
        last = atomicAdd(W.done, 1) == total - 1;
    }
    __syncthreads();
    if (last) {
        const int nflags = (int)(per * (W.nstages - 1));
        for (int e = threadIdx.x; e < nflags; e += LX * LY) W.prog[e] = 0;
        if (threadIdx.x == 0) *W.done = 0;
    }
}

}  // namespace wk
}  // namespace mgb
