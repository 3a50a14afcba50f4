// mg_api.cu -- the C ABI of include/mg.h: solver object, level hierarchy, V-cycle and solve
// loops.  Kernels live in mg_generic.cu (any grid / dtype) and mg_fused.cu (tuned fp32 path).
#include <cmath>
#include <limits>
#include <cstdarg>
#include <cstring>
#include <mutex>
#include <new>

#include "fused.h"
#include "solver.h"

namespace mgb {

static thread_local char g_err[512] = "";

void set_error(const char* fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
}

int sm_count() {
    static std::mutex mu;
    static int cache[64];
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) return 148;
    std::lock_guard<std::mutex> lock(mu);
    if (!cache[dev] && (cudaDeviceGetAttribute(&cache[dev], cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || cache[dev] < 1))
        cache[dev] = 148;
    return cache[dev];
}

int kernel_setup(const void* fn, int threads, size_t smem, int* ctas_per_sm, bool max_carveout) {
    struct Entry { int device; const void* fn; int ctas_per_sm; };
    static std::mutex mu;
    static std::vector<Entry> done;
    int dev = 0;
    MGB_CUDA(cudaGetDevice(&dev));
    std::lock_guard<std::mutex> lock(mu);
    for (const Entry& e : done)
        if (e.device == dev && e.fn == fn) { if (ctas_per_sm) *ctas_per_sm = e.ctas_per_sm; return 0; }
    if (smem > 48 * 1024) MGB_CUDA(cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    if (max_carveout) MGB_CUDA(cudaFuncSetAttribute(fn, cudaFuncAttributePreferredSharedMemoryCarveout, 100));
    int nb = 0;
    MGB_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, fn, threads, smem));
    done.push_back({dev, fn, nb > 0 ? nb : 1});
    if (ctas_per_sm) *ctas_per_sm = done.back().ctas_per_sm;
    return 0;
}

// Nodal 27-point filter of -Laplace from the trilinear-FE integrals (reading C1):
// 1-D stiffness (1/d)[-1,2,-1], consistent mass (d/6)[1,4,1]; w = (K M M + M K M + M M K)/(dx dy dz).
static void build_weights(double hx, double hy, double hz, double w[27]) {
    const double h[3] = {hx, hy, hz};
    double K[3][3], M[3][3];
    for (int d = 0; d < 3; ++d) {
        K[d][0] = K[d][2] = -1.0 / h[d]; K[d][1] = 2.0 / h[d];
        M[d][0] = M[d][2] = h[d] / 6.0;  M[d][1] = 4.0 * h[d] / 6.0;
    }
    const double ml = hx * hy * hz;
    for (int c = 0; c < 3; ++c)
        for (int b = 0; b < 3; ++b)
            for (int a = 0; a < 3; ++a)
                w[a + 3 * b + 9 * c] =
                    (K[0][a] * M[1][b] * M[2][c] + M[0][a] * K[1][b] * M[2][c] + M[0][a] * M[1][b] * K[2][c]) / ml;
}

static double bc_factor(int code) { return code == MG_BC_NEUMANN ? 1.0 : (code == MG_BC_DIRICHLET ? -1.0 : 0.0); }

static void fill_level_structs(mg_solver* s) {
    for (auto& L : s->lv) {
        double w[27];
        build_weights(L.hx, L.hy, L.hz, w);
        L.Lf.nx = L.Ld.nx = L.nx; L.Lf.ny = L.Ld.ny = L.ny; L.Lf.nz = L.Ld.nz = L.nz;
        for (int q = 0; q < 27; ++q) { L.Ld.w[q] = w[q]; L.Lf.w[q] = (float)w[q]; }
        for (int f = 0; f < 6; ++f) { L.Ld.s[f] = bc_factor(s->bc[f]); L.Lf.s[f] = (float)L.Ld.s[f]; }
        L.Ld.omega = s->p.omega; L.Lf.omega = (float)s->p.omega;
    }
}

template <typename T> static const Level<T>& lvl(const LevelData& L);
template <> const Level<float>& lvl<float>(const LevelData& L) { return L.Lf; }
template <> const Level<double>& lvl<double>(const LevelData& L) { return L.Ld; }

static size_t esize(const mg_solver* s) { return s->dtype == MG_F64 ? 8 : 4; }

struct DeviceGuard {
    int prev = -1;
    explicit DeviceGuard(int dev) { if (cudaGetDevice(&prev) != cudaSuccess) prev = -1; cudaSetDevice(dev); }
    ~DeviceGuard() { if (prev >= 0) cudaSetDevice(prev); }
};

// ---------------------------------------------------------------------------------------------
// un-fused path: one kernel per sweep / residual / restriction / prolongation (reading C6)
// ---------------------------------------------------------------------------------------------
template <typename T>
static int smooth_level(mg_solver* s, int l, T* x, const T* b, int sweeps) {
    LevelData& L = s->lv[l];
    T* cur = x; T* nxt = (T*)L.tmp;
    for (int it = 0; it < sweeps; ++it) {
        int rc = launch_jacobi<T>(lvl<T>(L), (const T*)L.k, cur, b, nxt, s->st);
        if (rc) return rc;
        ++s->launches;
        T* t = cur; cur = nxt; nxt = t;
    }
    if (cur != x) MGB_CUDA(cudaMemcpyAsync(x, cur, L.n * sizeof(T), cudaMemcpyDeviceToDevice, s->st));
    return 0;
}

// Optional per-level instrumentation (mg_vcycle_timed): ev[l] at the start of level l's down leg,
// ev[levels] after the coarsest solve, ev[levels + 1 + (levels - 2 - l)] after level l's up leg.
static inline void mark(mg_solver* s, int idx) {
    if (s->timing) cudaEventRecord(s->ev[idx], s->st);
}

template <typename T>
static int vcycle_unfused(mg_solver* s, int l, T* x, const T* b) {
    LevelData& L = s->lv[l];
    mark(s, l);
    if (l == s->levels - 1) {
        int rc0 = smooth_level<T>(s, l, x, b, s->p.coarse_sweeps);
        mark(s, s->levels);
        return rc0;
    }
    LevelData& C = s->lv[l + 1];
    int rc;
    if ((rc = smooth_level<T>(s, l, x, b, s->p.nu_pre))) return rc;
    if ((rc = launch_residual<T>(lvl<T>(L), (const T*)L.k, x, b, (T*)L.tmp, s->st))) return rc;
    if ((rc = launch_restrict<T>(C.nx, C.ny, C.nz, (const T*)L.tmp, (T*)C.b, s->st))) return rc;
    s->launches += 2;
    MGB_CUDA(cudaMemsetAsync(C.x, 0, C.n * sizeof(T), s->st));
    if ((rc = vcycle_unfused<T>(s, l + 1, (T*)C.x, (const T*)C.b))) return rc;
    if ((rc = launch_prolong_add<T>(L.nx, L.ny, L.nz, (const T*)C.x, x, s->st))) return rc;
    ++s->launches;
    rc = smooth_level<T>(s, l, x, b, s->p.nu_post);
    mark(s, s->levels + 1 + (s->levels - 2 - l));
    return rc;
}

// The un-fused cycle replayed from a CUDA graph (one capture per (x, b) pair), like the fused one: at 32^3 the ~60 small
// launches of a cycle are launch-bound otherwise.  Timed cycles (events between the levels) are enqueued directly.
template <typename T>
static int vcycle_unfused_graph(mg_solver* s, T* x, const T* b) {
    if (s->timing) return vcycle_unfused<T>(s, 0, x, b);
    return replay_graph(s, x, b, [&]() { return vcycle_unfused<T>(s, 0, x, b); });
}

template <typename T>
static int vcycle_any(mg_solver* s, T* x, const T* b) {
    return s->fused ? vcycle_unfused_graph<T>(s, x, b) : vcycle_unfused<T>(s, 0, x, b);
}
template <>
int vcycle_any<float>(mg_solver* s, float* x, const float* b) {
    if (s->fused && fused_supported(s)) return fused_vcycle(s, x, b);
    return s->fused ? vcycle_unfused_graph<float>(s, x, b) : vcycle_unfused<float>(s, 0, x, b);
}

// V-cycle from a zero initial guess: x need not be initialised.  The fused fp32 cycle replaces the first fine sweep by
// x = omega b / D; the other paths clear x first.
int vcycle_zero_guess(mg_solver* s, void* x, const void* b) {
    if (s->dtype == MG_F32 && s->fused && fused_supported(s)) return fused_vcycle(s, (float*)x, (const float*)b, 1);
    MGB_CUDA(cudaMemsetAsync(x, 0, s->lv[0].n * esize(s), s->st));
    return s->dtype == MG_F32 ? vcycle_any<float>(s, (float*)x, (const float*)b) : vcycle_any<double>(s, (double*)x, (const double*)b);
}

// accumulators: slot 0 is read back at once; slots 1.. hold the per-cycle squared residual norms of a fixed-count solve
// (tol = 0, the paper's mode), which are read back together after the last cycle: no host round trip per cycle
constexpr int ACC_N = 1 + 4096;

static int read_acc(mg_solver* s, double* out) {
    MGB_CUDA(cudaMemcpyAsync(s->h_acc, s->d_acc, sizeof(double), cudaMemcpyDeviceToHost, s->st));
    MGB_CUDA(cudaStreamSynchronize(s->st));
    *out = *s->h_acc;
    return 0;
}

template <typename T>
static int norm2(mg_solver* s, size_t n, const T* v, double* out) {
    MGB_CUDA(cudaMemsetAsync(s->d_acc, 0, sizeof(double), s->st));
    int rc = launch_sumsq<T>(n, v, s->d_acc, s->st);
    if (rc) return rc;
    ++s->launches;
    double sq;
    if ((rc = read_acc(s, &sq))) return rc;
    *out = std::sqrt(sq);
    return 0;
}

template <typename T>
static int residual_norm(mg_solver* s, const T* x, const T* b, double* out) {
    LevelData& L = s->lv[0];
    MGB_CUDA(cudaMemsetAsync(s->d_acc, 0, sizeof(double), s->st));
    int rc;
    if (sizeof(T) == 4 && s->fused && fused_residual_supported(s))
        rc = fused_residual(s, (const float*)x, (const float*)b, nullptr, s->d_acc);
    else if (s->fused && march_supported(L.nx, L.ny, L.nz, L.hx, L.hy, L.hz))
        rc = launch_march_residual<T, T>(L.nx, L.ny, L.nz, L.hx, L.Ld.s, x, (const T*)L.k, b, (T*)nullptr, s->d_acc, s->st);
    else rc = launch_residual_norm<T>(lvl<T>(L), (const T*)L.k, x, b, (T*)nullptr, s->d_acc, s->st);
    if (rc) return rc;
    ++s->launches;
    double sq;
    if ((rc = read_acc(s, &sq))) return rc;
    *out = std::sqrt(sq);
    return 0;
}

// Stopping bookkeeping shared by the solve loops (reading C6; stagnation rule of include/mg.h).
struct Stop {
    double tol; int stag = 0; double prev;
    double rate = 0.95;      // "no progress" = the residual fell by less than this factor since the last evaluation
    // returns -1 to continue, else the status
    int update(double rel) {
        if (!std::isfinite(rel)) return MG_STAGNATED;
        if (rel < tol) return MG_OK;
        if (tol == 0.0) return -1;  // fixed cycle count (the paper's mode): no stagnation test
        stag = (rel > rate * prev) ? stag + 1 : 0;
        prev = rel;
        return stag >= 3 ? MG_STAGNATED : -1;
    }
};

// a right-hand side with NaN / Inf in it (a time step that has blown up): say so instead of reporting ||r|| / ||b|| = 0
static int nonfinite_rhs(int* cycles_out, double* rel_out) {
    set_error("mg_solve: the right-hand side is not finite");
    if (cycles_out) *cycles_out = 0;
    if (rel_out) *rel_out = std::numeric_limits<double>::quiet_NaN();
    return MG_STAGNATED;
}

template <typename T>
static int solve_plain(mg_solver* s, T* x, const T* b, double tol, int max_cycles, int* cycles_out, double* rel_out) {
    LevelData& L = s->lv[0];
    int rc; double nb, nr;
    if ((rc = norm2<T>(s, L.n, b, &nb))) return rc;
    if (!std::isfinite(nb)) return nonfinite_rhs(cycles_out, rel_out);
    if ((rc = residual_norm<T>(s, x, b, &nr))) return rc;
    double rel = nb > 0.0 ? nr / nb : 0.0;
    Stop stop{tol, 0, rel};
    int cycles = 0, status = (rel < tol) ? MG_OK : MG_NOT_CONVERGED;
    while (status == MG_NOT_CONVERGED && cycles < max_cycles) {
        if ((rc = vcycle_any<T>(s, x, b))) return rc;
        if ((rc = residual_norm<T>(s, x, b, &nr))) return rc;
        rel = nb > 0.0 ? nr / nb : 0.0;
        s->history.push_back(rel);
        ++cycles;
        s->history_cycles.push_back(cycles);
        const int u = stop.update(rel);
        if (u >= 0) status = u;
    }
    if (cycles_out) *cycles_out = cycles;
    if (rel_out) *rel_out = rel;
    return status;
}

// fp32 solver with the fp64 outer defect-correction loop (reading C6 "fp32 reading", C8):
//   x64 = x;  repeat { r32 = float(b - A64 x64); stop on ||r||/||b||;  e = m V-cycles on A e = r32 from e = 0;  x64 += e }
// m = cycles_per_defect (1 by default).  One round of the loop -- the m cycles, the update and the next defect with its norm --
// is ONE CUDA graph: a one-thread kernel files the squared norm in the residual history on the device, so the launches of a
// round have no gaps between them and a fixed-count solve (tol = 0, the paper's mode) never waits for the host.
static int solve_mixed(mg_solver* s, float* x, const float* b, double tol, int max_cycles, int* cycles_out,
                       double* rel_out) {
    LevelData& L = s->lv[0];
    int rc; double nb, sq;
    if ((rc = norm2<float>(s, L.n, b, &nb))) return rc;
    if (!std::isfinite(nb)) return nonfinite_rhs(cycles_out, rel_out);
    if ((rc = launch_cast_f2d(L.n, x, s->x64, s->st))) return rc;
    ++s->launches;
    const bool marching = s->fused && march_supported(L.nx, L.ny, L.nz, L.hx, L.hy, L.hz);
    // Seeded correction cycles: the defect kernel also writes y = r32 / D into e32, and the cycle's first pass turns y into the
    // iterate after two sweeps from a zero guess (mg_fused.cu) -- one 12-byte pass instead of a 12-byte and a 16-byte one.
    const bool seeded = s->fused && fused_supported(s) && marching && fused_seed_supported(s);
    auto defect_into = [&](double* dacc) -> int {      // r32 = float(b - A64 x64), ||r||^2 ADDED to *dacc
        int r2;
        if (marching)
            r2 = launch_march_residual<double, float>(L.nx, L.ny, L.nz, L.hx, L.Ld.s, s->x64, s->var_k ? s->k64 : nullptr, b, s->r32,
                                                      dacc, s->st, 0, seeded ? s->e32 : nullptr);
        else r2 = launch_residual_mixed(L.Ld, s->var_k ? s->k64 : nullptr, s->x64, b, s->r32, dacc, s->st);
        if (!r2) ++s->launches;
        return r2;
    };
    MGB_CUDA(cudaMemsetAsync(s->d_acc, 0, sizeof(double), s->st));
    if ((rc = defect_into(s->d_acc))) return rc;
    if ((rc = read_acc(s, &sq))) return rc;
    double rel = nb > 0.0 ? std::sqrt(sq) / nb : 0.0;
    int cycles = 0, status = (rel < tol) ? MG_OK : MG_NOT_CONVERGED;
    // cycles per round: the parameter, or (cycles_per_defect = 0) chosen round by round: as many cycles as the observed contraction
    // says are still needed, at most M_AUTO -- defects cost time, cycles beyond the tolerance cost more
    constexpr int M_AUTO = 4, M_AUTO_TOL = 8;     // fixed-count solves; tolerance-driven solves (bounded by the contraction, below)
    const bool adaptive = s->p.cycles_per_defect == 0;
    const int m_max = adaptive ? M_AUTO : std::max(1, std::min(s->p.cycles_per_defect, 8));
    int m_next = adaptive && tol > 0.0 ? 1 : m_max;
    Stop stop{tol, 0, rel};
    // one round: mm cycles on A e = r32, x64 += e, next defect, its squared norm filed at hist[ctr++]
    auto round = [&](int mm, bool in_graph) -> int {
        int r2;
        for (int i = 0; i < mm; ++i) {
            if (in_graph) r2 = fused_vcycle_enqueue(s, s->e32, s->r32, i == 0 ? (seeded ? 2 : 1) : 0);
            else if (i == 0) r2 = seeded ? fused_vcycle(s, s->e32, s->r32, 2) : vcycle_zero_guess(s, s->e32, s->r32);
            else r2 = vcycle_any<float>(s, s->e32, s->r32);
            if (r2) return r2;
        }
        if ((r2 = launch_axpy_mixed(L.n, s->x64, s->e32, s->st))) return r2;
        ++s->launches;
        if ((r2 = defect_into(s->d_acc))) return r2;
        if ((r2 = launch_record_acc(s->d_acc, s->d_acc + 1, s->d_ctr, s->st))) return r2;
        ++s->launches;
        return 0;
    };
    MGB_CUDA(cudaMemsetAsync(s->d_acc, 0, sizeof(double), s->st));
    MGB_CUDA(cudaMemsetAsync(s->d_ctr, 0, sizeof(int), s->st));
    const bool graphs = seeded && !s->timing;          // the fused cycle can be recorded together with the rest of the round
    if (graphs && (rc = fused_vcycle_prepare(s))) return rc;
    int rounds = 0, read = 0;
    std::vector<int> round_cycles;
    auto fetch = [&](int upto) -> int {                // history entries [read, upto) from the device
        if (upto <= read) return 0;
        MGB_CUDA(cudaMemcpyAsync(s->h_acc + 1 + read, s->d_acc + 1 + read, (upto - read) * sizeof(double), cudaMemcpyDeviceToHost, s->st));
        MGB_CUDA(cudaStreamSynchronize(s->st));
        for (int c = read; c < upto; ++c) {
            rel = nb > 0.0 ? std::sqrt(s->h_acc[1 + c]) / nb : 0.0;
            s->history.push_back(rel);
            s->history_cycles.push_back(round_cycles[c]);
            if (!std::isfinite(rel)) status = MG_STAGNATED;
        }
        read = upto;
        return 0;
    };
    while (status == MG_NOT_CONVERGED && cycles < max_cycles && rounds < ACC_N - 1) {
        int mm = std::min(m_next, max_cycles - cycles);
        if (adaptive) {                                // round lengths 1, 2, 4, 8 only: every length is a recorded graph of its own
            int p2 = 1;
            while (2 * p2 <= mm) p2 *= 2;
            mm = p2;
        }
        if (graphs) rc = replay_graph(s, s->x64, b, [&]() { return round(mm, true); }, 16 + mm);
        else rc = round(mm, false);
        if (rc) return rc;
        cycles += mm; ++rounds;
        round_cycles.push_back(cycles);
        if (tol > 0.0) {                               // tolerance-driven: the host decides after every round
            const double before = rel;
            if ((rc = fetch(rounds))) return rc;
            if (status == MG_NOT_CONVERGED) {
                stop.rate = std::pow(0.95, mm);
                const int u = stop.update(rel);
                if (u >= 0) status = u;
            }
            if (adaptive && status == MG_NOT_CONVERGED) {
                // per-cycle contraction of the last round -> cycles still needed.  Early cycles contract faster than late ones, so
                // this errs towards too few cycles per round (one more defect), not towards cycles past the tolerance.
                // A round must not contract the correction below what fp32 resolves of it: rho^m >= 1e-5.
                const double rho = before > 0.0 ? std::pow(rel / before, 1.0 / mm) : 1.0;
                double need = M_AUTO, cap = M_AUTO;
                if (rho > 0.0 && rho < 1.0 && rel > tol) {
                    need = std::ceil(std::log(tol / rel) / std::log(rho));
                    cap = std::min((double)M_AUTO_TOL, std::floor(std::log(1e-5) / std::log(rho)));
                }
                m_next = (int)std::max(1.0, std::min(cap, need));
            }
        }
    }
    if ((rc = fetch(rounds))) return rc;               // fixed cycle count: all norms at once
    if ((rc = launch_cast_d2f(L.n, s->x64, x, s->st))) return rc;
    ++s->launches;
    MGB_CUDA(cudaStreamSynchronize(s->st));
    if (cycles_out) *cycles_out = cycles;
    if (rel_out) *rel_out = rel;
    return status;
}

int ensure_mixed_buffers(mg_solver* s) {
    if (s->x64 && s->k64 && s->r32 && s->e32) return 0;
    const size_t n = s->lv[0].n;
    if ((!s->x64 && cudaMalloc(&s->x64, n * 8) != cudaSuccess) || (!s->k64 && cudaMalloc(&s->k64, n * 8) != cudaSuccess) ||
        (!s->r32 && cudaMalloc(&s->r32, n * 4) != cudaSuccess) || (!s->e32 && cudaMalloc(&s->e32, n * 4) != cudaSuccess)) {
        // all or nothing: a later call must not find x64 set and the others NULL
        cudaFree(s->x64); cudaFree(s->k64); cudaFree(s->r32); cudaFree(s->e32);
        s->x64 = s->k64 = nullptr; s->r32 = s->e32 = nullptr;
        cudaGetLastError();
        set_error("mixed-precision buffers: out of device memory");
        return MG_EALLOC;
    }
    return 0;
}

template <typename T>
static int coarsen_coefficient(mg_solver* s) {
    for (int l = 0; l + 1 < s->levels; ++l) {
        LevelData& C = s->lv[l + 1];
        int rc = launch_restrict<T>(C.nx, C.ny, C.nz, (const T*)s->lv[l].k, (T*)C.k, s->st);
        if (rc) return rc;
        ++s->launches;
    }
    return 0;
}

static int alloc_k(mg_solver* s) {
    for (auto& L : s->lv)
        if (!L.k && cudaMalloc(&L.k, L.n * esize(s)) != cudaSuccess) {
            set_error("coefficient hierarchy: out of device memory");
            return MG_EALLOC;
        }
    return 0;
}

static void invalidate_graph(mg_solver* s) {
    for (auto& g : s->graphs) {
        if (g.exec) cudaGraphExecDestroy(g.exec);
        g = mg_solver::GraphSlot();
    }
    ++s->epoch;
}

}  // namespace mgb

using namespace mgb;

#define CHECK_SOLVER(s)                                         \
    if (!(s)) { set_error("NULL solver"); return MG_EINVAL; }   \
    DeviceGuard guard_((s)->device)

extern "C" {

const char* mg_last_error(void) { return g_err; }
const char* mg_version(void) { return "libmg_b200 0.1 (sm_100a)"; }

int mg_create(mg_solver** out, const mg_grid* grid, int levels, const int bc[6], int dtype, void* cuda_stream) {
    if (!out || !grid || !bc) { set_error("mg_create: NULL argument"); return MG_EINVAL; }
    *out = nullptr;
    if (levels < 1 || levels > 16 || (dtype != MG_F32 && dtype != MG_F64) || !(grid->hx > 0) || !(grid->hy > 0) ||
        !(grid->hz > 0) || grid->nx < 1 || grid->ny < 1 || grid->nz < 1) {
        set_error("mg_create: invalid levels / dtype / grid");
        return MG_EINVAL;
    }
    for (int f = 0; f < 6; ++f)
        if (bc[f] < 0 || bc[f] > 2) { set_error("mg_create: bc[%d] = %d is not an mg_bc", f, bc[f]); return MG_EINVAL; }
    const int div = 1 << (levels - 1);
    if (grid->nx % div || grid->ny % div || grid->nz % div || grid->nx / div < 2 || grid->ny / div < 2 ||
        grid->nz / div < 2) {
        set_error("mg_create: %dx%dx%d is not divisible into %d levels with a coarsest dimension >= 2", grid->nx,
                  grid->ny, grid->nz, levels);
        return MG_ESHAPE;
    }
    if ((long long)grid->nx * grid->ny * grid->nz > 2147483647LL) {           // element indices of a level are 32-bit in places
        set_error("mg_create: %dx%dx%d has more than 2^31 - 1 points", grid->nx, grid->ny, grid->nz);
        return MG_ESHAPE;
    }
    int dev = 0;
    MGB_CUDA(cudaGetDevice(&dev));
    mg_solver* s = new (std::nothrow) mg_solver();
    if (!s) { set_error("mg_create: out of host memory"); return MG_EALLOC; }
    s->grid = *grid; s->levels = levels; s->dtype = dtype; s->device = dev; s->st = (cudaStream_t)cuda_stream;
    for (int f = 0; f < 6; ++f) s->bc[f] = bc[f];
    s->lv.resize(levels);
    for (int l = 0; l < levels; ++l) {
        LevelData& L = s->lv[l];
        L.nx = grid->nx >> l; L.ny = grid->ny >> l; L.nz = grid->nz >> l;
        L.hx = grid->hx * (1 << l); L.hy = grid->hy * (1 << l); L.hz = grid->hz * (1 << l);
        L.n = npts(L.nx, L.ny, L.nz);
        L.uniform = (grid->hx == grid->hy && grid->hy == grid->hz);
    }
    fill_level_structs(s);
    bool ok = true;
    const size_t es = esize(s);
    for (int l = 0; l < levels && ok; ++l) {
        LevelData& L = s->lv[l];
        ok = ok && cudaMalloc(&L.tmp, L.n * es) == cudaSuccess;
        if (l > 0) ok = ok && cudaMalloc(&L.x, L.n * es) == cudaSuccess && cudaMalloc(&L.b, L.n * es) == cudaSuccess;
    }
    ok = ok && cudaMalloc(&s->d_acc, ACC_N * sizeof(double)) == cudaSuccess;
    ok = ok && cudaMalloc(&s->d_ctr, sizeof(int)) == cudaSuccess;
    ok = ok && cudaMallocHost(&s->h_acc, ACC_N * sizeof(double)) == cudaSuccess;
    if (!ok) {
        set_error("mg_create: allocation failed: %s", cudaGetErrorString(cudaGetLastError()));
        mg_destroy(s);
        return MG_EALLOC;
    }
    *out = s;
    return MG_OK;
}

void mg_destroy(mg_solver* s) {
    if (!s) return;
    DeviceGuard guard_(s->device);
    cudaStreamSynchronize(s->st);
    invalidate_graph(s);
    fused_release(s);
    if (s->cap_st) cudaStreamDestroy(s->cap_st);
    for (auto& e : s->ev) cudaEventDestroy(e);
    for (size_t l = 0; l < s->lv.size(); ++l) {
        LevelData& L = s->lv[l];
        if (l > 0) { cudaFree(L.x); cudaFree(L.b); }
        cudaFree(L.k); cudaFree(L.tmp);
    }
    cudaFree(s->x64); cudaFree(s->k64); cudaFree(s->r32); cudaFree(s->e32);
    for (double* v : s->pcg_v) cudaFree(v);
    cudaFree(s->pcg_s);
    cudaFree(s->hx_dev); cudaFree(s->hb_dev);
    cudaFree(s->d_acc); cudaFree(s->d_ctr);
    if (s->h_acc) cudaFreeHost(s->h_acc);
    delete s;
}

int mg_set_params(mg_solver* s, const mg_params* p) {
    CHECK_SOLVER(s);
    if (!p || p->nu_pre < 0 || p->nu_post < 0 || p->coarse_sweeps < 0 || !(p->omega > 0.0) || !(p->omega < 2.0)) {
        set_error("mg_set_params: invalid parameters");
        return MG_EINVAL;
    }
    if (p->cycles_per_defect < 0 || p->cycles_per_defect > 8) {
        set_error("mg_set_params: cycles_per_defect = %d is out of range (0 = adaptive, 1 .. 8)", p->cycles_per_defect);
        return MG_EINVAL;
    }
    // stages per launch of the wave kernel (wave_kernel.cuh): 1 .. 4 are implemented; anything else is refused
    if (p->sweeps_per_pass < 1 || p->sweeps_per_pass > 4) {
        set_error("mg_set_params: sweeps_per_pass = %d is not implemented (1 .. 4)", p->sweeps_per_pass);
        return MG_EINVAL;
    }
    s->p = *p;
    fill_level_structs(s);
    invalidate_graph(s);
    return MG_OK;
}

int mg_get_params(const mg_solver* s, mg_params* p) {
    if (!s || !p) { set_error("mg_get_params: NULL argument"); return MG_EINVAL; }
    *p = s->p;
    return MG_OK;
}

int mg_set_fused(mg_solver* s, int fused) {
    CHECK_SOLVER(s);
    s->fused = fused ? 1 : 0;
    invalidate_graph(s);
    return MG_OK;
}

int mg_set_coefficient(mg_solver* s, const void* d_k) {
    CHECK_SOLVER(s);
    // the recorded cycle holds pointers and sizes, not coefficient values: it stays valid while the solver goes from one
    // variable coefficient to the next (same buffers), and is dropped when it changes between constant and variable
    if (!d_k || !s->var_k) invalidate_graph(s);
    if (!d_k) {
        for (auto& L : s->lv) { cudaFree(L.k); L.k = nullptr; }
        s->var_k = false;
        return (s->dtype == MG_F32 && fused_supported(s)) ? fused_prepare(s) : MG_OK;
    }
    int rc = alloc_k(s);
    if (rc) return rc;
    const size_t n = s->lv[0].n;
    MGB_CUDA(cudaMemcpyAsync(s->lv[0].k, d_k, n * esize(s), cudaMemcpyDeviceToDevice, s->st));
    s->var_k = true;
    if (s->dtype == MG_F32) {
        if ((rc = ensure_mixed_buffers(s))) return rc;
        if ((rc = launch_cast_f2d(n, (const float*)d_k, s->k64, s->st))) return rc;
        ++s->launches;
        if ((rc = coarsen_coefficient<float>(s))) return rc;
        return fused_supported(s) ? fused_prepare(s) : MG_OK;
    }
    return coarsen_coefficient<double>(s);
}

int mg_set_coefficient_from_vof(mg_solver* s, const void* d_alpha, double rho_l, double rho_g) {
    CHECK_SOLVER(s);
    if (!d_alpha || !(rho_l > 0.0) || !(rho_g > 0.0)) { set_error("mg_set_coefficient_from_vof: invalid argument"); return MG_EINVAL; }
    if (!s->var_k) invalidate_graph(s);
    int rc = alloc_k(s);
    if (rc) return rc;
    const size_t n = s->lv[0].n;
    s->var_k = true;
    if (s->dtype == MG_F32) {
        if ((rc = ensure_mixed_buffers(s))) return rc;
        if ((rc = launch_k_from_vof<float>(n, (const float*)d_alpha, rho_l, rho_g, (float*)s->lv[0].k, s->st))) return rc;
        if ((rc = launch_k64_from_vof(n, (const float*)d_alpha, rho_l, rho_g, s->k64, s->st))) return rc;
        s->launches += 2;
        if ((rc = coarsen_coefficient<float>(s))) return rc;
        return fused_supported(s) ? fused_prepare(s) : MG_OK;
    }
    if ((rc = launch_k_from_vof<double>(n, (const double*)d_alpha, rho_l, rho_g, (double*)s->lv[0].k, s->st))) return rc;
    ++s->launches;
    return coarsen_coefficient<double>(s);
}

int mg_apply_operator(mg_solver* s, const void* d_x, void* d_y) {
    CHECK_SOLVER(s);
    if (!d_x || !d_y || d_x == d_y) { set_error("mg_apply_operator: NULL or aliased argument"); return MG_EINVAL; }
    LevelData& L = s->lv[0];
    if (s->dtype == MG_F32 && s->fused && fused_residual_supported(s))      // fp32 uniform grid: streaming kernel, MODE_RES
        return fused_residual(s, (const float*)d_x, nullptr, (float*)d_y, nullptr);
    ++s->launches;
    if (s->fused && march_supported(L.nx, L.ny, L.nz, L.hx, L.hy, L.hz)) {   // uniform grid: z-marching kernel, b = NULL -> y = A x
        if (s->dtype == MG_F32)
            return launch_march_residual<float, float>(L.nx, L.ny, L.nz, L.hx, L.Ld.s, (const float*)d_x, (const float*)L.k,
                                                       (const float*)nullptr, (float*)d_y, nullptr, s->st);
        return launch_march_residual<double, double>(L.nx, L.ny, L.nz, L.hx, L.Ld.s, (const double*)d_x, (const double*)L.k,
                                                     (const double*)nullptr, (double*)d_y, nullptr, s->st);
    }
    if (s->dtype == MG_F32) return launch_apply<float>(L.Lf, (const float*)L.k, (const float*)d_x, (float*)d_y, s->st);
    return launch_apply<double>(L.Ld, (const double*)L.k, (const double*)d_x, (double*)d_y, s->st);
}

int mg_residual(mg_solver* s, const void* d_x, const void* d_b, void* d_r) {
    CHECK_SOLVER(s);
    if (!d_x || !d_b || !d_r || d_x == d_r) { set_error("mg_residual: NULL or aliased argument"); return MG_EINVAL; }
    LevelData& L = s->lv[0];
    if (s->dtype == MG_F32 && s->fused && fused_residual_supported(s))
        return fused_residual(s, (const float*)d_x, (const float*)d_b, (float*)d_r, nullptr);
    ++s->launches;
    if (s->fused && march_supported(L.nx, L.ny, L.nz, L.hx, L.hy, L.hz)) {
        if (s->dtype == MG_F32)
            return launch_march_residual<float, float>(L.nx, L.ny, L.nz, L.hx, L.Ld.s, (const float*)d_x, (const float*)L.k,
                                                       (const float*)d_b, (float*)d_r, nullptr, s->st);
        return launch_march_residual<double, double>(L.nx, L.ny, L.nz, L.hx, L.Ld.s, (const double*)d_x, (const double*)L.k,
                                                     (const double*)d_b, (double*)d_r, nullptr, s->st);
    }
    if (s->dtype == MG_F32)
        return launch_residual<float>(L.Lf, (const float*)L.k, (const float*)d_x, (const float*)d_b, (float*)d_r, s->st);
    return launch_residual<double>(L.Ld, (const double*)L.k, (const double*)d_x, (const double*)d_b, (double*)d_r, s->st);
}

int mg_smooth(mg_solver* s, void* d_x, const void* d_b, int sweeps) {
    CHECK_SOLVER(s);
    if (!d_x || !d_b || sweeps < 0) { set_error("mg_smooth: invalid argument"); return MG_EINVAL; }
    if (s->dtype == MG_F32) {
        if (s->fused && fused_supported(s)) return fused_smooth(s, (float*)d_x, (const float*)d_b, sweeps);
        return smooth_level<float>(s, 0, (float*)d_x, (const float*)d_b, sweeps);
    }
    return smooth_level<double>(s, 0, (double*)d_x, (const double*)d_b, sweeps);
}

int mg_vcycle(mg_solver* s, void* d_x, const void* d_b) {
    CHECK_SOLVER(s);
    if (!d_x || !d_b) { set_error("mg_vcycle: NULL argument"); return MG_EINVAL; }
    if (s->dtype == MG_F32) return vcycle_any<float>(s, (float*)d_x, (const float*)d_b);
    return vcycle_any<double>(s, (double*)d_x, (const double*)d_b);
}

int mg_solve(mg_solver* s, void* d_x, const void* d_b, double tol, int max_cycles, int* cycles_out, double* relres_out) {
    CHECK_SOLVER(s);
    if (!d_x || !d_b || max_cycles < 0 || !(tol >= 0.0)) { set_error("mg_solve: invalid argument"); return MG_EINVAL; }
    s->history.clear(); s->history_cycles.clear();
    if (s->dtype == MG_F64) return solve_plain<double>(s, (double*)d_x, (const double*)d_b, tol, max_cycles, cycles_out, relres_out);
    if (!s->p.mixed_precision) return solve_plain<float>(s, (float*)d_x, (const float*)d_b, tol, max_cycles, cycles_out, relres_out);
    int rc = ensure_mixed_buffers(s);
    if (rc) return rc;
    return solve_mixed(s, (float*)d_x, (const float*)d_b, tol, max_cycles, cycles_out, relres_out);
}

static int solve_host(mg_solver* s, void* h_x, const void* h_b, bool zero_guess, double tol, int max_cycles, int* cycles_out,
                      double* relres_out) {
    CHECK_SOLVER(s);
    if (!h_x || !h_b) { set_error("mg_solve_host: NULL argument"); return MG_EINVAL; }
    const size_t bytes = s->lv[0].n * esize(s);
    if (!s->hx_dev && (cudaMalloc(&s->hx_dev, bytes) != cudaSuccess || cudaMalloc(&s->hb_dev, bytes) != cudaSuccess)) {
        set_error("mg_solve_host: out of device memory");
        return MG_EALLOC;
    }
    if (zero_guess) MGB_CUDA(cudaMemsetAsync(s->hx_dev, 0, bytes, s->st));         // all-zero bytes = +0.0 in fp32 and fp64
    else MGB_CUDA(cudaMemcpyAsync(s->hx_dev, h_x, bytes, cudaMemcpyHostToDevice, s->st));
    MGB_CUDA(cudaMemcpyAsync(s->hb_dev, h_b, bytes, cudaMemcpyHostToDevice, s->st));
    const int status = mg_solve(s, s->hx_dev, s->hb_dev, tol, max_cycles, cycles_out, relres_out);
    if (status < 0) return status;
    MGB_CUDA(cudaMemcpyAsync(h_x, s->hx_dev, bytes, cudaMemcpyDeviceToHost, s->st));
    MGB_CUDA(cudaStreamSynchronize(s->st));
    return status;
}

int mg_solve_host(mg_solver* s, void* h_x, const void* h_b, double tol, int max_cycles, int* cycles_out, double* relres_out) {
    return solve_host(s, h_x, h_b, false, tol, max_cycles, cycles_out, relres_out);
}

int mg_solve_host_zero(mg_solver* s, void* h_x, const void* h_b, double tol, int max_cycles, int* cycles_out, double* relres_out) {
    return solve_host(s, h_x, h_b, true, tol, max_cycles, cycles_out, relres_out);
}

int mg_get_history_cycles(const mg_solver* s, int* h_cycles, int n) {
    if (!s) { set_error("NULL solver"); return MG_EINVAL; }
    const int m = (int)s->history_cycles.size();
    for (int c = 0; c < m && c < n && h_cycles; ++c) h_cycles[c] = s->history_cycles[c];
    return m;
}

int mg_get_history(const mg_solver* s, double* h_history, int n) {
    if (!s) { set_error("NULL solver"); return MG_EINVAL; }
    const int m = (int)s->history.size();
    for (int c = 0; c < m && c < n && h_history; ++c) h_history[c] = s->history[c];
    return m;
}

long long mg_level_info(const mg_solver* s, int level, int* nx, int* ny, int* nz) {
    if (!s || level < 0 || level >= s->levels) { set_error("mg_level_info: out of range"); return MG_EINVAL; }
    const LevelData& L = s->lv[level];
    if (nx) *nx = L.nx;
    if (ny) *ny = L.ny;
    if (nz) *nz = L.nz;
    return (long long)L.n;
}

long long mg_launch_count(const mg_solver* s) { return s ? s->launches : 0; }

int mg_vcycle_timed(mg_solver* s, void* d_x, const void* d_b, float* h_ms_down, float* h_ms_up) {
    CHECK_SOLVER(s);
    if (!d_x || !d_b || !h_ms_down || !h_ms_up) { set_error("mg_vcycle_timed: NULL argument"); return MG_EINVAL; }
    const int L = s->levels;
    if (s->ev.empty()) {
        s->ev.resize(2 * L);
        for (auto& e : s->ev) MGB_CUDA(cudaEventCreate(&e));
    }
    s->timing = true;
    int rc = (s->dtype == MG_F32) ? vcycle_any<float>(s, (float*)d_x, (const float*)d_b)
                                  : vcycle_any<double>(s, (double*)d_x, (const double*)d_b);
    s->timing = false;
    if (rc) return rc;
    MGB_CUDA(cudaStreamSynchronize(s->st));
    for (int l = 0; l < L; ++l) { h_ms_down[l] = 0.f; h_ms_up[l] = 0.f; }
    for (int l = 0; l < L; ++l) MGB_CUDA(cudaEventElapsedTime(&h_ms_down[l], s->ev[l], s->ev[l + 1]));
    for (int l = L - 2; l >= 0; --l) {
        const int e = L + 1 + (L - 2 - l);
        MGB_CUDA(cudaEventElapsedTime(&h_ms_up[l], s->ev[e - 1], s->ev[e]));
    }
    return MG_OK;
}

}  // extern "C"
