// mg_fused.cu -- host side of the tuned fp32 path: pass planning for the streaming smoother / transfer kernel
// (lean_kernel.cuh: one stage per launch; wave_kernel.cuh: up to `sweeps_per_pass` dependent stages per launch), TMA
// descriptors, the cluster / single-block coarse tail (ctail_kernel.cuh, tail_kernel.cuh), and CUDA-graph replay of the
// whole V-cycle (north_star "fused" kernels).
#include <algorithm>
#include <cstdlib>
#include <cstring>

#include "fused.h"
#include "solver.h"
#include "lean_kernel.cuh"
#include "wave_kernel.cuh"
#include "ctail_kernel.cuh"
#include "tail_kernel.cuh"

namespace mgb {
namespace {

// ---- TMA descriptor encoding through the driver entry point (no link-time libcuda dependency) ----
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                  const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn encode_fn() {
    static EncodeTiledFn fn = nullptr;
    if (!fn) {
        void* p = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess &&
            q == cudaDriverEntryPointSuccess)
            fn = (EncodeTiledFn)p;
    }
    return fn;
}

// 3-D fp32 field (nx, ny, nz), box = one z plane of px x py cells, out-of-bounds cells read as 0.
int make_tmap(CUtensorMap* tm, const float* ptr, int nx, int ny, int nz, int px, int py) {
    EncodeTiledFn fn = encode_fn();
    if (!fn) { set_error("cuTensorMapEncodeTiled is not available from the driver"); return MG_ECUDA; }
    const cuuint64_t dims[3] = {(cuuint64_t)nx, (cuuint64_t)ny, (cuuint64_t)nz};
    const cuuint64_t strides[2] = {(cuuint64_t)nx * 4, (cuuint64_t)nx * ny * 4};
    const cuuint32_t box[3] = {(cuuint32_t)px, (cuuint32_t)py, 1};
    const cuuint32_t estr[3] = {1, 1, 1};
    const CUresult r = fn(tm, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, const_cast<float*>(ptr), dims, strides, box, estr,
                          CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                          CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) { set_error("cuTensorMapEncodeTiled failed (%d) for %dx%dx%d box %dx%d", (int)r, nx, ny, nz, px, py); return MG_ECUDA; }
    return 0;
}

// Launch with programmatic stream serialisation: the kernel may start while its predecessor in the stream is still running
// and synchronises with it by griddepcontrol.wait before it first touches dependent data.
template <typename... KArgs, typename... Args>
cudaError_t launch_pdl(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st, Args... args) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr; cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kernel, KArgs(args)...);
}

}  // namespace
// the same encoder for the explicit kernels (flow.cu, flow_tma.cuh); tm points to a CUtensorMap
int make_tmap_f32(void* tm, const float* ptr, int nx, int ny, int nz, int px, int py) { return make_tmap((CUtensorMap*)tm, ptr, nx, ny, nz, px, py); }
namespace {

// ---- small helper kernels for levels below the tile size ------------------------------------
__global__ void first_sweep_kernel(size_t n, const float* __restrict__ bc, const float* __restrict__ dinv, float g,
                                   float* __restrict__ xc) {
    const size_t n4 = n >> 2, stride = (size_t)gridDim.x * blockDim.x, t = blockIdx.x * (size_t)blockDim.x + threadIdx.x;
    for (size_t c = t; c < n4; c += stride) {                 // cudaMalloc'ed level arrays: 16-byte aligned
        float4 v = reinterpret_cast<const float4*>(bc)[c];
        if (dinv) {
            const float4 d = reinterpret_cast<const float4*>(dinv)[c];
            v.x *= d.x; v.y *= d.y; v.z *= d.z; v.w *= d.w;
        }
        reinterpret_cast<float4*>(xc)[c] = make_float4(g * v.x, g * v.y, g * v.z, g * v.w);
    }
    for (size_t c = 4 * n4 + t; c < n; c += stride) xc[c] = dinv ? g * (dinv[c] * bc[c]) : g * bc[c];
}

// 1 / D_i of a level (variable k): D_i = sum_{j != i} (-w_ij) (k_i + k_j)/2, halo of k by copy
__global__ void dinv_kernel(int nx, int ny, int nz, float ce, float cc, float cdiag, const float* __restrict__ k,
                            float* __restrict__ dinv) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y * blockDim.y + threadIdx.y, kz = blockIdx.z;
    if (i >= nx || j >= ny) return;
    float e = 0.f, cn = 0.f;
    for (int c = -1; c <= 1; ++c)
        for (int b = -1; b <= 1; ++b)
            for (int a = -1; a <= 1; ++a) {
                const int m = (a != 0) + (b != 0) + (c != 0);
                if (m < 2) continue;
                const int ii = min(max(i + a, 0), nx - 1), jj = min(max(j + b, 0), ny - 1), kk = min(max(kz + c, 0), nz - 1);
                const float v = k[(size_t)ii + (size_t)nx * (jj + (size_t)ny * kk)];
                if (m == 2) e += v; else cn += v;
            }
    const size_t c0 = (size_t)i + (size_t)nx * (j + (size_t)ny * kz);
    dinv[c0] = 1.f / (cdiag * k[c0] + ce * e + cc * cn);
}

struct LevelPlan {
    bool stream = false;      // handled by lean_kernel / wave_kernel
    float* dinv = nullptr;    // 1/D (variable k), levels >= 1
    float* tmp2 = nullptr;    // residual scratch of levels the streaming kernels do not cover
    float ce = 0, cc = 0, cdiag = 0, w0 = 0;
};

struct FusedState {
    std::vector<LevelPlan> lp;
    int sm_count = 148;       // multiprocessors of the solver's device
    float* cmat = nullptr;    // the coarsest solve tabulated as a matrix (ctail_kernel.cuh), n_c <= 64
    bool cmat_valid = false;
    long long cmat_epoch = -1;  // mg_solver::epoch the table was built in (a parameter change bumps it)
    int* wave_sync = nullptr; // wave_kernel: progress flags [WAVE_FLAGS], then the finished-block counter and the error word
};
constexpr int WAVE_FLAGS = 8192;

// One stage of a pass on level l: what it reads and writes besides the iterate.
struct StageSpec {
    int mode = lk::MODE_SWEEP;
    const float* xc = nullptr;      // PRO: coarse correction
    float* bc_out = nullptr;        // RR: restricted residual
    float* xc_out = nullptr;        // RR: the coarse level's first sweep (or zeros)
    int first_sweep = 0;            // RR
    int zero_x = 0;                 // SWEEP: the incoming iterate is zero whatever the buffer holds
    float rsign = 1.f;              // RES: out = rsign (b - A x)
    double* acc = nullptr;          // RES: sum of out^2 (fp64, added to *acc)
};

// tensor maps and parameters of one stage (shared by the one-stage and the wave launches)
template <class C>
int fill_stage(mg_solver* s, int l, const StageSpec& sp, const float* src, const float* b, float* dst, int zchunk,
               CUtensorMap* tmx, CUtensorMap* tmk, CUtensorMap* tmb, CUtensorMap* tmc, lk::LParams* Pout) {
    FusedState* fs = (FusedState*)s->fused_state;
    LevelData& L = s->lv[l];
    const LevelPlan& lp = fs->lp[l];
    int rc;
    if ((rc = make_tmap(tmx, src, L.nx, L.ny, L.nz, C::PX, C::PY))) return rc;
    if ((rc = make_tmap(tmb, b ? b : src, L.nx, L.ny, L.nz, C::TX, C::TY))) return rc;     // b == NULL (RES: y = A x): never fetched
    if (C::VAR) { if ((rc = make_tmap(tmk, (const float*)L.k, L.nx, L.ny, L.nz, C::PX, C::PY))) return rc; }
    else *tmk = *tmx;
    if (sp.mode == lk::MODE_PRO) { if ((rc = make_tmap(tmc, sp.xc, L.nx / 2, L.ny / 2, L.nz / 2, C::CPX, C::CPY))) return rc; }
    else *tmc = *tmx;
    lk::LParams P;
    std::memset(&P, 0, sizeof(P));
    P.nx = L.nx; P.ny = L.ny; P.nz = L.nz;
    P.zchunk = zchunk;
    P.sx0 = L.Lf.s[0]; P.sx1 = L.Lf.s[1]; P.sy0 = L.Lf.s[2]; P.sy1 = L.Lf.s[3]; P.sz0 = L.Lf.s[4]; P.sz1 = L.Lf.s[5];
    P.cc = lp.cc; P.icc = (float)(24.0 * L.hx * L.hx);
    P.omega = (float)s->p.omega;
    P.out = dst; P.xc = sp.xc; P.bc_out = sp.bc_out; P.xc_out = sp.xc_out; P.first_sweep = sp.first_sweep;
    P.zero_x = (sp.mode == lk::MODE_SWEEP && sp.zero_x) ? 1 : 0;
    if (sp.mode == lk::MODE_RES) { P.rsign = sp.rsign; P.zero_b = b ? 0 : 1; P.acc = sp.acc; }
    if (sp.mode == lk::MODE_SEED) { P.om_g = P.omega * P.omega; P.om_x = P.omega * (2.f - P.omega); P.icc = 0.f; }
    if (sp.mode == lk::MODE_RR) {
        const LevelPlan& cp = fs->lp[l + 1];
        P.dinv_c = cp.dinv;
        P.gc_const = sp.first_sweep ? (float)(s->p.omega / cp.w0) : 0.f;
    }
    *Pout = P;
    return 0;
}

// ---- one stage per launch (lean_kernel.cuh) ---------------------------------------------------------
template <int LX, int LY, int MINB, bool VAR, int MODE>
int launch_stream_cfg(mg_solver* s, int l, const StageSpec& sp, const float* src, const float* b, float* dst) {
    using C = lk::LCfg<LX, LY, VAR, MODE, MINB>;
    FusedState* fs = (FusedState*)s->fused_state;
    LevelData& L = s->lv[l];
    int ctas_per_sm = 1, rc;
    if ((rc = kernel_setup((const void*)lk::lean_kernel<C>, C::NT, C::SMEM, &ctas_per_sm, true))) return rc;
    const int tiles = ((L.nx + C::TX - 1) / C::TX) * ((L.ny + C::TY - 1) / C::TY);
    // z chunking: minimise (waves over the resident CTA slots) x (planes per block incl. the two halo planes)
    double best_cost = 1e30;
    int zchunk = L.nz;
    const int slots = fs->sm_count * ctas_per_sm;
    for (int nch = 1; nch <= std::max(1, L.nz / 2); ++nch) {
        int zc = (L.nz + nch - 1) / nch; zc += zc & 1;
        const int real = (L.nz + zc - 1) / zc;
        const double waves = std::ceil((double)tiles * real / (double)slots);
        const double cost = waves * (zc + 2 + 2);
        if (cost < best_cost - 1e-9) { best_cost = cost; zchunk = zc; }
    }
    const int nchunks = (L.nz + zchunk - 1) / zchunk;
    CUtensorMap tmx, tmk, tmb, tmc;
    lk::LParams P;
    if ((rc = fill_stage<C>(s, l, sp, src, b, dst, zchunk, &tmx, &tmk, &tmb, &tmc, &P))) return rc;
    dim3 grid((L.nx + C::TX - 1) / C::TX, (L.ny + C::TY - 1) / C::TY, nchunks);
    MGB_CUDA(launch_pdl(lk::lean_kernel<C>, grid, dim3(C::NT), C::SMEM, s->st, tmx, tmk, tmb, tmc, P));
    ++s->launches;
    return 0;
}

template <bool VAR, int MODE>
int launch_stream_lx(mg_solver* s, int l, const StageSpec& sp, const float* src, const float* b, float* dst) {
    const int nx = s->lv[l].nx;
    // 128-thread blocks, 3 per SM: 168 registers per thread keep the per-point state and the staged rows out of local memory
    if (nx >= 96) return launch_stream_cfg<32, 4, 3, VAR, MODE>(s, l, sp, src, b, dst);
    if (nx >= 48) return launch_stream_cfg<16, 8, 3, VAR, MODE>(s, l, sp, src, b, dst);
    return launch_stream_cfg<8, 16, 3, VAR, MODE>(s, l, sp, src, b, dst);
}

// one streaming pass on level l
int launch_stream(mg_solver* s, int l, const StageSpec& sp, const float* src, const float* b, float* dst) {
#define MGB_SCASE(m)                                                                       \
    if (sp.mode == m)                                                                      \
        return s->var_k ? launch_stream_lx<true, m>(s, l, sp, src, b, dst)                 \
                        : launch_stream_lx<false, m>(s, l, sp, src, b, dst);
    MGB_SCASE(lk::MODE_SWEEP)
    MGB_SCASE(lk::MODE_PRO)
    MGB_SCASE(lk::MODE_RR)
    MGB_SCASE(lk::MODE_SEED)
    MGB_SCASE(lk::MODE_RES)
#undef MGB_SCASE
    set_error("stream pass mode %d is not instantiated", sp.mode);
    return MG_EINVAL;
}

// ---- several dependent stages per launch (wave_kernel.cuh) ------------------------------------------
// Stages st[0 .. n) of level l in one launch; the iterate starts in `cur` and ping-pongs with `oth` (RR stages do not
// write it).  Returns MG_ESHAPE-like "does not fit" as +1 so that the caller can fall back to fewer stages per launch.
template <int LX, int LY, int MINB, bool VAR>
int launch_wave_cfg(mg_solver* s, int l, const StageSpec* st, int n, float* cur, float* oth, const float* b) {
    using C = lk::LCfg<LX, LY, VAR, lk::MODE_PRO, MINB>;
    FusedState* fs = (FusedState*)s->fused_state;
    LevelData& L = s->lv[l];
    auto kern = wk::wave_kernel<LX, LY, VAR, MINB>;
    int ctas_per_sm = 1, rc;
    if ((rc = kernel_setup((const void*)kern, C::NT, C::SMEM, &ctas_per_sm, true))) return rc;
    const int gx = (L.nx + C::TX - 1) / C::TX, gy = (L.ny + C::TY - 1) / C::TY, tiles = gx * gy;
    const int slots = fs->sm_count * ctas_per_sm;
    // every block of every stage has to be resident at once for the stages to overlap: as many z chunks as fit
    int nch = slots / (tiles * n);
    if (nch < 1) return 1;
    nch = std::min(nch, std::max(1, L.nz / 8));
    int zchunk = (L.nz + nch - 1) / nch; zchunk += zchunk & 1;
    nch = (L.nz + zchunk - 1) / zchunk;
    if ((size_t)(n - 1) * nch * tiles > (size_t)WAVE_FLAGS) return 1;
    wk::WParams W;
    std::memset(&W, 0, sizeof(W));
    W.nstages = n; W.nch = nch; W.gx = gx; W.gy = gy;
    W.prog = fs->wave_sync; W.done = fs->wave_sync + WAVE_FLAGS; W.err = fs->wave_sync + WAVE_FLAGS + 1;
    for (int i = 0; i < n; ++i) {
        wk::WStage& S = W.st[i];
        S.mode = st[i].mode;
        const bool writes = st[i].mode != lk::MODE_RR;
        if ((rc = fill_stage<C>(s, l, st[i], cur, b, writes ? oth : nullptr, zchunk, &S.tmx, &S.tmk, &S.tmb, &S.tmc, &S.P))) return rc;
        if (writes) std::swap(cur, oth);
    }
    dim3 grid(gx, gy, nch * n);
    MGB_CUDA(launch_pdl(kern, grid, dim3(C::NT), C::SMEM, s->st, W));
    ++s->launches;
    return 0;
}

int launch_wave(mg_solver* s, int l, const StageSpec* st, int n, float* cur, float* oth, const float* b) {
    const int nx = s->lv[l].nx;
#define MGB_WCASE(lx, ly)                                                                   \
    return s->var_k ? launch_wave_cfg<lx, ly, 3, true>(s, l, st, n, cur, oth, b)            \
                    : launch_wave_cfg<lx, ly, 3, false>(s, l, st, n, cur, oth, b);
    if (nx >= 96) { MGB_WCASE(32, 4) }
    if (nx >= 48) { MGB_WCASE(16, 8) }
    MGB_WCASE(8, 16)
#undef MGB_WCASE
}

// A chain of stages on a streaming level: groups of up to `sweeps_per_pass` stages per launch.  *res = the buffer that
// holds the iterate afterwards.
int run_chain(mg_solver* s, int l, float* cur, float* oth, const float* b, const StageSpec* st, int n, float** res) {
    int i = 0;
    while (i < n) {
        int g = std::min(std::min(s->p.sweeps_per_pass, wk::MAXS), n - i);
        int rc = 1;
        while (g >= 2 && (rc = launch_wave(s, l, st + i, g, cur, oth, b)) == 1) --g;     // 1: does not fit the machine
        if (g >= 2 && rc) return rc;
        if (g < 2) {
            g = 1;
            const bool writes = st[i].mode != lk::MODE_RR;
            if ((rc = launch_stream(s, l, st[i], cur, b, writes ? oth : nullptr))) return rc;
        }
        for (int q = i; q < i + g; ++q)
            if (st[q].mode != lk::MODE_RR) std::swap(cur, oth);
        i += g;
    }
    *res = cur;
    return 0;
}

int ensure_state(mg_solver* s) {
    if (s->fused_state) return 0;
    FusedState* fs = new FusedState();
    fs->lp.resize(s->levels);
    s->fused_state = fs;                  // owned by the solver from here on (fused_release frees partial state)
    fs->sm_count = sm_count();
    for (int l = 0; l < s->levels; ++l) {
        LevelData& L = s->lv[l];
        LevelPlan& lp = fs->lp[l];
        const double h2 = L.hx * L.hx;
        lp.ce = (float)(1.0 / (12.0 * h2)); lp.cc = (float)(1.0 / (24.0 * h2));
        lp.cdiag = (float)(4.0 / (3.0 * h2)); lp.w0 = (float)(8.0 / (3.0 * h2));
        lp.stream = (L.nx % 4 == 0) && (L.ny % 2 == 0) && (L.nz % 2 == 0) && L.nx >= 8 && L.ny >= 4 && L.nz >= 2;
        if (!lp.stream && cudaMalloc(&lp.tmp2, L.n * sizeof(float)) != cudaSuccess) { set_error("fused: out of memory"); return MG_EALLOC; }
    }
    if (cudaMalloc(&fs->wave_sync, (WAVE_FLAGS + 2) * sizeof(int)) != cudaSuccess) { set_error("fused: out of memory"); return MG_EALLOC; }
    MGB_CUDA(cudaMemsetAsync(fs->wave_sync, 0, (WAVE_FLAGS + 2) * sizeof(int), s->st));
    return 0;
}

// refresh 1/D of the levels >= 1 after a coefficient change (cheap: all coarse levels together are n/7 points)
int refresh_dinv(mg_solver* s) {
    FusedState* fs = (FusedState*)s->fused_state;
    for (int l = 1; l < s->levels; ++l) {
        LevelData& L = s->lv[l];
        LevelPlan& lp = fs->lp[l];
        if (!s->var_k) { cudaFree(lp.dinv); lp.dinv = nullptr; continue; }
        if (!lp.dinv && cudaMalloc(&lp.dinv, L.n * sizeof(float)) != cudaSuccess) { set_error("fused: out of memory"); return MG_EALLOC; }
        dim3 blk(32, 4), grd((L.nx + 31) / 32, (L.ny + 3) / 4, L.nz);
        dinv_kernel<<<grd, blk, 0, s->st>>>(L.nx, L.ny, L.nz, lp.ce, lp.cc, lp.cdiag, (const float*)L.k, lp.dinv);
        MGB_LAUNCH_CHECK();
        ++s->launches;
    }
    return 0;
}

inline void mark(mg_solver* s, int idx) {
    if (s->timing) cudaEventRecord(s->ev[idx], s->st);
}

// `sweeps` Jacobi sweeps on level l starting from `cur` (other buffer `oth`), optionally preceded by
// x += P xc.  Returns the buffer holding the result through *res.  `zero_x`: the incoming iterate is zero whatever
// `cur` holds (streaming levels with sweeps >= 1 only; the caller checks).
int sweeps_level(mg_solver* s, int l, float* cur, float* oth, const float* b, int sweeps, const float* xc, float** res,
                 int zero_x = 0) {
    FusedState* fs = (FusedState*)s->fused_state;
    LevelData& L = s->lv[l];
    int rc;
    if (fs->lp[l].stream) {
        bool pro = xc != nullptr;
        // the PRO pass stages x_c by TMA: its row pitch (nx / 2 floats) must be a multiple of 16 bytes
        if (pro && (sweeps == 0 || (L.nx / 2) % 4 != 0)) {
            if ((rc = launch_prolong_add<float>(L.nx, L.ny, L.nz, xc, cur, s->st))) return rc;
            ++s->launches;
            pro = false;
        }
        std::vector<StageSpec> st((size_t)sweeps);
        if (sweeps > 0) {
            if (pro) { st[0].mode = lk::MODE_PRO; st[0].xc = xc; }
            st[0].zero_x = zero_x;
        }
        return run_chain(s, l, cur, oth, b, st.data(), sweeps, res);
    }
    if (xc) {
        if ((rc = launch_prolong_add<float>(L.nx, L.ny, L.nz, xc, cur, s->st))) return rc;
        ++s->launches;
    }
    for (int it = 0; it < sweeps; ++it) {
        if ((rc = launch_jacobi<float>(L.Lf, (const float*)L.k, cur, b, oth, s->st))) return rc;
        ++s->launches;
        std::swap(cur, oth);
    }
    *res = cur;
    return 0;
}

// All levels from l down to the coarsest in one thread block (tail_kernel.cuh), if they fit on chip.
bool tail_fits(const mg_solver* s, int l, size_t* smem_out) {
    if (l < 1 || s->levels - l > tk::MAXL) return false;
    const LevelData& L = s->lv[l];
    if (L.nx > 16 || L.ny > 16 || L.nz > 16) return false;
    size_t fl = 0;
    for (int t = l; t < s->levels; ++t) fl += 5 * s->lv[t].n;
    *smem_out = fl * sizeof(float);
    return *smem_out <= 200 * 1024;
}

int launch_tail(mg_solver* s, int l, float* x, const float* b, int done, size_t smem) {
    FusedState* fs = (FusedState*)s->fused_state;
    tk::TailParams P;
    std::memset(&P, 0, sizeof(P));
    P.nlev = s->levels - l;
    for (int t = 0; t < P.nlev; ++t) {
        const LevelData& L = s->lv[l + t];
        const LevelPlan& lp = fs->lp[l + t];
        P.nx[t] = L.nx; P.ny[t] = L.ny; P.nz[t] = L.nz;
        P.k[t] = s->var_k ? (const float*)L.k : nullptr;
        P.dinv[t] = s->var_k ? lp.dinv : nullptr;
        P.ce[t] = lp.ce; P.cc[t] = lp.cc; P.dinv_const[t] = 1.f / lp.w0;
    }
    for (int f = 0; f < 6; ++f) P.s[f] = s->lv[l].Lf.s[f];
    P.omega = (float)s->p.omega;
    P.nu_pre = s->p.nu_pre; P.nu_post = s->p.nu_post; P.coarse_sweeps = s->p.coarse_sweeps;
    P.first_done = done; P.x = x; P.b = b;
    { int rc = kernel_setup((const void*)tk::tail_kernel, tk::NT, 200 * 1024, nullptr); if (rc) return rc; }
    MGB_CUDA(launch_pdl(tk::tail_kernel, dim3(1), dim3(tk::NT), smem, s->st, P));
    ++s->launches;
    return 0;
}

// All levels from l down on one 8-block cluster (ctail_kernel.cuh): a prefix of "distributed" levels whose nz is a
// multiple of 8 (the last of them with nz = 8), then 1-2 "solo" levels in block 0.
bool ctail_fits(const mg_solver* s, int l, size_t* smem_out, int* nd_out, int* ns_out) {
    static const bool disabled = getenv("MG_NO_CLUSTER_TAIL") != nullptr;
    // measured on B200: a 32^3 level is faster as five lean_kernel launches (13 us in the graph) than inside the cluster
    // (31 us); from 16^3 down the cluster beats the single-block tail (29 us vs 41 us)
    if (disabled || l < 1 || s->lv[l].n > 8192) return false;
    int nd = 0;
    while (l + nd < s->levels && s->lv[l + nd].nz >= ck::NC) ++nd;
    const int ns = s->levels - l - nd;
    if (nd < 1 || nd > ck::MAXD || ns < 1 || ns > ck::MAXS) return false;
    size_t fl = 0;
    for (int t = 0; t < nd; ++t) {
        const LevelData& L = s->lv[l + t];
        if (L.nz % ck::NC || L.nx % 4 || L.ny % 2) return false;
        const size_t ps = (size_t)L.nx * L.ny, nzl = L.nz / ck::NC;
        fl += 3 * (nzl + 2) * ps + 2 * nzl * ps;
    }
    if (s->lv[l + nd - 1].nz != ck::NC) return false;
    for (int u = 0; u < ns; ++u) {
        if (s->lv[l + nd + u].n > 4096) return false;
        fl += 5 * s->lv[l + nd + u].n;
    }
    const LevelData& Ld = s->lv[l + nd - 1];
    fl += (size_t)ck::NC * (Ld.nx / 2) * (Ld.ny / 2) + s->lv[l + nd].n;
    *smem_out = fl * sizeof(float);
    *nd_out = nd; *ns_out = ns;
    return *smem_out <= 200 * 1024;
}

struct Fac6 { float v[6]; };
// column `blockIdx.x` of the coarsest-solve matrix: `sweeps` Jacobi sweeps from a zero guess on the unit vector
__global__ void __launch_bounds__(tk::NT, 1) coarse_matrix_kernel(int nx, int ny, int nz, const float* __restrict__ k, const float* __restrict__ dinv,
                                                                 float dinv_const, float ce, float cc, Fac6 fac, float omega, int sweeps,
                                                                 float* __restrict__ cmat) {
    extern __shared__ __align__(16) float sm[];
    __shared__ float sf[6];
    tk::Lv L;
    L.nx = nx; L.ny = ny; L.nz = nz; L.n = nx * ny * nz; L.ce = ce; L.cc = cc;
    L.X = sm; L.Y = sm + L.n; L.B = sm + 2 * L.n; L.K = sm + 3 * L.n; L.DI = sm + 4 * L.n;
    if (threadIdx.x < 6) sf[threadIdx.x] = fac.v[threadIdx.x];
    const int col = blockIdx.x;
    for (int idx = threadIdx.x; idx < L.n; idx += tk::NT) {
        L.K[idx] = k ? k[idx] : 1.f;
        L.DI[idx] = dinv ? dinv[idx] : dinv_const;
        const float bi = idx == col ? 1.f : 0.f;
        L.B[idx] = bi;
        L.X[idx] = sweeps >= 1 ? omega * L.DI[idx] * bi : 0.f;
        L.Y[idx] = 0.f;
    }
    __syncthreads();
    tk::sweeps(L, sf, omega, max(0, sweeps - 1));
    for (int idx = threadIdx.x; idx < L.n; idx += tk::NT) cmat[(size_t)col * L.n + idx] = L.X[idx];
}

// (re)tabulate the coarsest solve; stream-ordered after the coefficient set-up, before the cycle that uses it
int refresh_cmat(mg_solver* s) {
    FusedState* fs = (FusedState*)s->fused_state;
    const int lc = s->levels - 1;
    const LevelData& L = s->lv[lc];
    static const bool disabled = getenv("MG_NO_COARSE_MATRIX") != nullptr;
    if (disabled || s->levels < 2 || L.n > 64 || L.n % 4 || s->p.coarse_sweeps < 1) { fs->cmat_valid = false; return 0; }
    if (!fs->cmat && cudaMalloc(&fs->cmat, 64 * 64 * sizeof(float)) != cudaSuccess) { set_error("fused: out of memory"); return MG_EALLOC; }
    const LevelPlan& lp = fs->lp[lc];
    Fac6 fac;
    for (int f = 0; f < 6; ++f) fac.v[f] = L.Lf.s[f];
    coarse_matrix_kernel<<<(int)L.n, tk::NT, 5 * L.n * sizeof(float), s->st>>>(L.nx, L.ny, L.nz, s->var_k ? (const float*)L.k : nullptr,
                                                                             s->var_k ? lp.dinv : nullptr, 1.f / lp.w0, lp.ce, lp.cc, fac,
                                                                             (float)s->p.omega, s->p.coarse_sweeps, fs->cmat);
    MGB_LAUNCH_CHECK();
    ++s->launches;
    fs->cmat_valid = true;
    return 0;
}

// the tabulated coarsest solve follows the coefficient (fused_prepare clears the flag) and the parameters (the solver's epoch)
int ensure_cmat(mg_solver* s) {
    FusedState* fs = (FusedState*)s->fused_state;
    if (fs->cmat_valid && fs->cmat_epoch == s->epoch) return 0;
    fs->cmat_epoch = s->epoch;
    return refresh_cmat(s);
}

int launch_ctail(mg_solver* s, int l, float* x, const float* b, int done, size_t smem, int nd, int ns) {
    FusedState* fs = (FusedState*)s->fused_state;
    ck::CParams P;
    std::memset(&P, 0, sizeof(P));
    P.nd = nd; P.ns = ns;
    for (int t = 0; t < nd + ns; ++t) {
        const LevelData& L = s->lv[l + t];
        const LevelPlan& lp = fs->lp[l + t];
        P.nx[t] = L.nx; P.ny[t] = L.ny; P.nz[t] = L.nz;
        P.k[t] = s->var_k ? (const float*)L.k : nullptr;
        P.dinv[t] = s->var_k ? lp.dinv : nullptr;
        P.ce[t] = lp.ce; P.cc[t] = lp.cc; P.dinv_const[t] = 1.f / lp.w0;
    }
    for (int f = 0; f < 6; ++f) P.s[f] = s->lv[l].Lf.s[f];
    P.omega = (float)s->p.omega;
    P.nu_pre = s->p.nu_pre; P.nu_post = s->p.nu_post; P.coarse_sweeps = s->p.coarse_sweeps;
    P.first_done = done; P.x = x; P.b = b;
    P.cmat = fs->cmat_valid ? fs->cmat : nullptr;
    { int rc = kernel_setup((const void*)ck::ctail_kernel, ck::NT, 200 * 1024, nullptr); if (rc) return rc; }
    MGB_CUDA(launch_pdl(ck::ctail_kernel, dim3(ck::NC), dim3(ck::NT), smem, s->st, P));
    ++s->launches;
    return 0;
}

// Level l of the V-cycle.  `A` holds the incoming iterate (for l > 0 the parent's fused first sweep
// has already been applied when `done` = 1); the final iterate of the level is returned in *res.
// Level 0 only: `zero_x` = the incoming iterate is zero whatever A holds; `seed` = A holds the Jacobi seed y = b / D and the
// first stage turns it into the iterate after two sweeps (then `done` = 2).
int cycle_level(mg_solver* s, int l, float* A, float* B, const float* b, int done, float** res, int zero_x = 0, int seed = 0) {
    FusedState* fs = (FusedState*)s->fused_state;
    LevelData& L = s->lv[l];
    int rc;
    mark(s, l);
    size_t tail_smem = 0;
    int cnd = 0, cns = 0;
    const bool ctail = ctail_fits(s, l, &tail_smem, &cnd, &cns);
    if (ctail || tail_fits(s, l, &tail_smem)) {
        rc = ctail ? launch_ctail(s, l, A, b, done, tail_smem, cnd, cns) : launch_tail(s, l, A, b, done, tail_smem);
        for (int t = l + 1; t <= s->levels; ++t) mark(s, t);                                   // sub-levels are not timed apart
        for (int t = s->levels - 2; t >= l; --t) mark(s, s->levels + 1 + (s->levels - 2 - t));
        *res = A;
        return rc;
    }
    if (l == s->levels - 1) {
        rc = sweeps_level(s, l, A, B, b, std::max(0, s->p.coarse_sweeps - done), nullptr, res);
        mark(s, s->levels);
        return rc;
    }
    LevelData& C = s->lv[l + 1];
    const bool child_coarsest = (l + 1 == s->levels - 1);
    const int first = child_coarsest ? (s->p.coarse_sweeps >= 1) : (s->p.nu_pre >= 1);
    float *cur = A, *oth = B;
    const int rem = std::max(0, s->p.nu_pre - done);
    if (fs->lp[l].stream) {
        // down leg: [SEED] + pre-smoothing sweeps + residual / restriction / coarse first sweep, as one chain of stages
        std::vector<StageSpec> st;
        if (seed) { StageSpec sp; sp.mode = lk::MODE_SEED; st.push_back(sp); }
        for (int q = 0; q < rem; ++q) { StageSpec sp; sp.zero_x = (q == 0 && zero_x); st.push_back(sp); }
        StageSpec rr; rr.mode = lk::MODE_RR; rr.bc_out = (float*)C.b; rr.xc_out = (float*)C.x; rr.first_sweep = first;
        st.push_back(rr);
        if ((rc = run_chain(s, l, cur, oth, b, st.data(), (int)st.size(), &cur))) return rc;
        oth = (cur == A) ? B : A;
    } else {
        if ((rc = sweeps_level(s, l, cur, oth, b, rem, nullptr, &cur))) return rc;
        oth = (cur == A) ? B : A;
        float* r = fs->lp[l].tmp2;
        if ((rc = launch_residual<float>(L.Lf, (const float*)L.k, cur, b, r, s->st))) return rc;
        if ((rc = launch_restrict<float>(C.nx, C.ny, C.nz, r, (float*)C.b, s->st))) return rc;
        s->launches += 2;
        if (first) {
            const LevelPlan& cp = fs->lp[l + 1];
            const float g = s->var_k ? (float)s->p.omega : (float)(s->p.omega / cp.w0);
            first_sweep_kernel<<<(int)std::min<size_t>((C.n + 255) / 256, 1184), 256, 0, s->st>>>(C.n, (const float*)C.b, s->var_k ? cp.dinv : nullptr, g, (float*)C.x);
            MGB_LAUNCH_CHECK();
            ++s->launches;
        } else {
            MGB_CUDA(cudaMemsetAsync(C.x, 0, C.n * sizeof(float), s->st));
        }
    }
    float* child = nullptr;
    if ((rc = cycle_level(s, l + 1, (float*)C.x, (float*)C.tmp, (const float*)C.b, first, &child))) return rc;
    if ((rc = sweeps_level(s, l, cur, oth, b, s->p.nu_post, child, &cur))) return rc;
    mark(s, s->levels + 1 + (s->levels - 2 - l));
    *res = cur;
    return 0;
}

// zero_guess 1: x is taken as 0 whatever it holds: the first pre-smoothing pass does not read it (12 bytes per point instead
// of 16, and the caller need not clear x).  zero_guess 2: x holds the Jacobi seed y = b / D of a cycle from a zero guess
// (written by the defect kernel); the first pass turns it into the iterate after TWO sweeps,
// x_2 = omega (2 - omega) y - omega^2 D^-1 (A - D) y, without reading b: one 12-byte pass instead of two sweeps.
int enqueue_vcycle(mg_solver* s, float* x, const float* b, int zero_guess) {
    float* res = nullptr;
    float *A = x, *B = (float*)s->lv[0].tmp;
    int rc;
    if ((rc = cycle_level(s, 0, A, B, b, zero_guess == 2 ? 2 : 0, &res, zero_guess == 1, zero_guess == 2))) return rc;
    if (res != x) MGB_CUDA(cudaMemcpyAsync(x, res, s->lv[0].n * sizeof(float), cudaMemcpyDeviceToDevice, s->st));
    return 0;
}

}  // namespace

bool fused_supported(const mg_solver* s) {
    if (s->dtype != MG_F32 || s->levels < 1) return false;
    const LevelData& L = s->lv[0];
    return L.uniform;
}

int fused_prepare(mg_solver* s) {
    int rc = ensure_state(s);
    if (rc) return rc;
    ((FusedState*)s->fused_state)->cmat_valid = false;       // rebuilt before the next cycle (fused_vcycle)
    return refresh_dinv(s);
}

int fused_smooth(mg_solver* s, float* x, const float* b, int sweeps) {
    int rc = ensure_state(s);
    if (rc) return rc;
    float* res = nullptr;
    if ((rc = sweeps_level(s, 0, x, (float*)s->lv[0].tmp, b, sweeps, nullptr, &res))) return rc;
    if (res != x) MGB_CUDA(cudaMemcpyAsync(x, res, s->lv[0].n * sizeof(float), cudaMemcpyDeviceToDevice, s->st));
    return 0;
}

// r = b - A x (b != NULL) or y = A x (b == NULL) on the fine level with the streaming kernel (MODE_RES); r may be NULL;
// acc (may be NULL): ||out||^2 is ADDED to *acc in fp64
bool fused_residual_supported(mg_solver* s) {
    if (!fused_supported(s) || ensure_state(s)) return false;
    return ((FusedState*)s->fused_state)->lp[0].stream;
}
int fused_residual(mg_solver* s, const float* x, const float* b, float* r, double* acc) {
    int rc = ensure_state(s);
    if (rc) return rc;
    StageSpec sp;
    sp.mode = lk::MODE_RES; sp.rsign = b ? 1.f : -1.f; sp.acc = acc;
    return launch_stream(s, 0, sp, x, b, r);
}

// Everything a cycle needs that must NOT be recorded with it (state, the tabulated coarsest solve): call before
// fused_vcycle_enqueue when the enqueue happens inside a graph capture.
int fused_vcycle_prepare(mg_solver* s) {
    int rc = ensure_state(s);
    if (rc) return rc;
    // the tabulated coarsest solve follows the coefficient (fused_prepare clears the flag) and the parameters (the epoch)
    return ensure_cmat(s);
}

// Launch the kernels of one cycle on s->st (no graph of its own: the caller may be recording one).
int fused_vcycle_enqueue(mg_solver* s, float* x, const float* b, int zero_guess) {
    if (zero_guess) {
        // the first launch of the cycle has to be a lean_kernel sweep of level 0; otherwise clear x and run the general cycle
        FusedState* fs = (FusedState*)s->fused_state;
        size_t sm = 0; int a = 0, c = 0;
        const bool lean0 = fs->lp[0].stream && s->p.nu_pre >= 1 && s->levels > 1 &&
                           !ctail_fits(s, 0, &sm, &a, &c) && !tail_fits(s, 0, &sm);
        if (zero_guess == 2 && !(lean0 && s->p.nu_pre >= 2)) { set_error("fused_vcycle: the seeded cycle is not available"); return MG_EINVAL; }
        if (!lean0) {
            MGB_CUDA(cudaMemsetAsync(x, 0, s->lv[0].n * sizeof(float), s->st));
            zero_guess = 0;
        }
    }
    return enqueue_vcycle(s, x, b, zero_guess);
}

int fused_vcycle(mg_solver* s, float* x, const float* b, int zero_guess) {
    int rc = fused_vcycle_prepare(s);
    if (rc) return rc;
    if (s->timing) return fused_vcycle_enqueue(s, x, b, zero_guess);
    return replay_graph(s, x, b, [&]() { return fused_vcycle_enqueue(s, x, b, zero_guess); }, zero_guess);
}

// the seeded cycle (zero_guess 2) needs a lean_kernel sweep as the first launch of level 0 and two pre-smoothing sweeps
bool fused_seed_supported(mg_solver* s) {
    if (ensure_state(s)) return false;
    FusedState* fs = (FusedState*)s->fused_state;
    size_t sm = 0; int a = 0, c = 0;
    return fs->lp[0].stream && s->p.nu_pre >= 2 && s->levels > 1 && !ctail_fits(s, 0, &sm, &a, &c) &&
           !tail_fits(s, 0, &sm);
}

void fused_release(mg_solver* s) {
    FusedState* fs = (FusedState*)s->fused_state;
    if (!fs) return;
    for (auto& lp : fs->lp) { cudaFree(lp.dinv); cudaFree(lp.tmp2); }
    cudaFree(fs->cmat);
    cudaFree(fs->wave_sync);
    delete fs;
    s->fused_state = nullptr;
}

}  // namespace mgb
