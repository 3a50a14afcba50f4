// mg_pcg.cu -- mg_pcg_solve: V-cycle-preconditioned conjugate gradients (SURVEY 8(f) "next 1").
// Not in the paper (which runs plain cycles): the remedy for their slow convergence under a 1000:1 coefficient
// jump.  Textbook PCG, the preconditioner being one V(nu, nu) cycle from a zero guess:
//   r = b - A x;  z = M r;  p = z;  rz = <r, z>
//   repeat:  q = A p;  alpha = rz / <p, q>;  x += alpha p;  r -= alpha q;  stop on ||r|| / ||b|| < tol;
//            z = M r;  rz' = <r, z>;  beta = rz' / rz;  p = z + beta p;  rz = rz'
// The CG vectors x, r, p, q are fp64 whatever the solver's dtype; for MG_F32 the preconditioner is the fused fp32 cycle
// (r is handed to it rounded to fp32, z comes back in fp32), for MG_F64 the fp64 cycle.  alpha and beta are formed on
// the device from accumulated dot products; the host reads one double per iteration (the residual norm).
#include <cmath>

#include "solver.h"

namespace mgb {
namespace {

// device scalars
enum { S_RZ = 0, S_RZ_NEW = 1, S_PQ = 2, S_RR = 3, S_N = 8 };

__device__ __forceinline__ double block_sum_d(double v) {
    __shared__ double red[32];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = v;
    __syncthreads();
    double t = 0.0;
    if (threadIdx.x < 32) {
        t = threadIdx.x < (blockDim.x >> 5) ? red[threadIdx.x] : 0.0;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) t += __shfl_xor_sync(0xffffffffu, t, o);
    }
    return t;
}

// sc[slot] += <r, z>; optionally r32 = float(r) was written by the caller
template <typename TZ>
__global__ void __launch_bounds__(256) dot_rz_kernel(size_t n, const double* __restrict__ r, const TZ* __restrict__ z, double* __restrict__ sc,
                                                     int slot) {
    double s = 0.0;
    for (size_t c = blockIdx.x * (size_t)blockDim.x + threadIdx.x; c < n; c += (size_t)gridDim.x * blockDim.x) s += r[c] * (double)z[c];
    s = block_sum_d(s);
    if (threadIdx.x == 0) atomicAdd(sc + slot, s);
}

// first: p = z;  later: p = z + (rz_new / rz) p
template <typename TZ>
__global__ void __launch_bounds__(256) update_p_kernel(size_t n, const TZ* __restrict__ z, double* __restrict__ p, const double* __restrict__ sc,
                                                       int first) {
    const double beta = first ? 0.0 : sc[S_RZ_NEW] / sc[S_RZ];
    for (size_t c = blockIdx.x * (size_t)blockDim.x + threadIdx.x; c < n; c += (size_t)gridDim.x * blockDim.x)
        p[c] = first ? (double)z[c] : (double)z[c] + beta * p[c];
}

// alpha = rz / pq;  x += alpha p;  r -= alpha q;  sc[S_RR] += ||r||^2;  rout = r in the preconditioner's precision
template <typename TZ>
__global__ void __launch_bounds__(256) update_xr_kernel(size_t n, const double* __restrict__ p, const double* __restrict__ q, double* __restrict__ x,
                                                        double* __restrict__ r, TZ* __restrict__ rout, double* __restrict__ sc) {
    const double alpha = sc[S_RZ] / sc[S_PQ];
    double s = 0.0;
    for (size_t c = blockIdx.x * (size_t)blockDim.x + threadIdx.x; c < n; c += (size_t)gridDim.x * blockDim.x) {
        x[c] += alpha * p[c];
        const double rv = r[c] - alpha * q[c];
        r[c] = rv;
        if (rout) rout[c] = (TZ)rv;
        s += rv * rv;
    }
    s = block_sum_d(s);
    if (threadIdx.x == 0) atomicAdd(sc + S_RR, s);
}

// between iterations: rz <- rz_new (when `shift`), clear the accumulators
__global__ void scalars_kernel(double* sc, int shift) {
    if (shift) sc[S_RZ] = sc[S_RZ_NEW];
    sc[S_RZ_NEW] = 0.0; sc[S_PQ] = 0.0; sc[S_RR] = 0.0;
}

template <typename TA, typename TB>
__global__ void __launch_bounds__(256) cast_kernel2(size_t n, const TA* __restrict__ a, TB* __restrict__ b) {
    for (size_t c = blockIdx.x * (size_t)blockDim.x + threadIdx.x; c < n; c += (size_t)gridDim.x * blockDim.x) b[c] = (TB)a[c];
}

inline int blocks_for(size_t n) { return (int)std::min<size_t>((n + 255) / 256, (size_t)sm_count() * 16); }

template <typename TZ>   // TZ = float: MG_F32 solver (mixed), double: MG_F64 solver
int pcg_t(mg_solver* s, void* d_x, const void* d_b, double tol, int max_iter, int* iters_out, double* rel_out) {
    LevelData& L = s->lv[0];
    const size_t n = L.n;
    const bool f32 = sizeof(TZ) == 4;
    cudaStream_t st = s->st;
    // buffers: [0] b64 (f32 only), [1] r, [2] p, [3] q, [4] z64 (f64 only)
    for (int v = 0; v < 5; ++v) {
        if ((v == 0 && !f32) || (v == 4 && f32) || s->pcg_v[v]) continue;
        if (cudaMalloc(&s->pcg_v[v], n * sizeof(double)) != cudaSuccess) { set_error("mg_pcg_solve: out of device memory"); return MG_EALLOC; }
    }
    if (!s->pcg_s && cudaMalloc(&s->pcg_s, S_N * sizeof(double)) != cudaSuccess) { set_error("mg_pcg_solve: out of device memory"); return MG_EALLOC; }
    int rc;
    if (f32 && (rc = ensure_mixed_buffers(s))) return rc;
    double* x = f32 ? s->x64 : (double*)d_x;
    const double* b = f32 ? s->pcg_v[0] : (const double*)d_b;
    const double* k = s->var_k ? (f32 ? s->k64 : (const double*)L.k) : nullptr;
    double *r = s->pcg_v[1], *p = s->pcg_v[2], *q = s->pcg_v[3], *sc = s->pcg_s;
    TZ* z = f32 ? (TZ*)s->e32 : (TZ*)s->pcg_v[4];          // preconditioner output
    TZ* rin = f32 ? (TZ*)s->r32 : (TZ*)r;                  // preconditioner input (fp64: r itself)
    const int nb = blocks_for(n);
    if (f32) {
        cast_kernel2<float, double><<<nb, 256, 0, st>>>(n, (const float*)d_x, x);
        cast_kernel2<float, double><<<nb, 256, 0, st>>>(n, (const float*)d_b, s->pcg_v[0]);
        s->launches += 2;
    }
    auto read = [&](int slot, double* out) -> int {
        MGB_CUDA(cudaMemcpyAsync(s->h_acc, sc + slot, sizeof(double), cudaMemcpyDeviceToHost, st));
        MGB_CUDA(cudaStreamSynchronize(st));
        *out = *s->h_acc;
        return 0;
    };
    auto precondition = [&]() -> int {            // z = M rin from a zero guess
        return vcycle_zero_guess(s, z, rin);
    };
    // ||b||, r = b - A x, ||r||
    double bb, rr;
    MGB_CUDA(cudaMemsetAsync(sc, 0, S_N * sizeof(double), st));
    if ((rc = launch_sumsq<double>(n, b, sc + S_PQ, st))) return rc;
    if ((rc = read(S_PQ, &bb))) return rc;
    if (!std::isfinite(bb)) {          // a right-hand side with NaN / Inf in it: say so instead of reporting a zero residual
        set_error("mg_pcg_solve: the right-hand side is not finite");
        if (iters_out) *iters_out = 0;
        if (rel_out) *rel_out = std::nan("");
        return MG_STAGNATED;
    }
    if ((rc = launch_march_residual<double, double>(L.nx, L.ny, L.nz, L.hx, L.Ld.s, x, k, b, r, sc + S_RR, st))) return rc;
    s->launches += 2;
    if ((rc = read(S_RR, &rr))) return rc;
    const double nbn = std::sqrt(bb);
    double rel = nbn > 0.0 ? std::sqrt(rr) / nbn : 0.0;
    int it = 0, status = (rel < tol) ? MG_OK : MG_NOT_CONVERGED;
    if (status == MG_NOT_CONVERGED && max_iter > 0) {
        if (f32) { cast_kernel2<double, TZ><<<nb, 256, 0, st>>>(n, r, rin); ++s->launches; }
        if ((rc = precondition())) return rc;
        scalars_kernel<<<1, 1, 0, st>>>(sc, 0);
        dot_rz_kernel<TZ><<<nb, 256, 0, st>>>(n, r, z, sc, S_RZ);
        update_p_kernel<TZ><<<nb, 256, 0, st>>>(n, z, p, sc, 1);
        s->launches += 3;
        while (it < max_iter) {
            // q = A p, pq = <p, q>
            if ((rc = launch_march_residual<double, double>(L.nx, L.ny, L.nz, L.hx, L.Ld.s, p, k, (const double*)nullptr, q, sc + S_PQ, st, 1)))
                return rc;
            update_xr_kernel<TZ><<<nb, 256, 0, st>>>(n, p, q, x, r, f32 ? rin : (TZ*)nullptr, sc);
            s->launches += 2;
            if ((rc = read(S_RR, &rr))) return rc;
            rel = std::sqrt(rr) / nbn;
            s->history.push_back(rel);
            s->history_cycles.push_back((int)s->history.size());
            ++it;
            if (!std::isfinite(rel)) { status = MG_STAGNATED; break; }
            if (rel < tol) { status = MG_OK; break; }
            if (it == max_iter) break;
            if ((rc = precondition())) return rc;
            dot_rz_kernel<TZ><<<nb, 256, 0, st>>>(n, r, z, sc, S_RZ_NEW);
            update_p_kernel<TZ><<<nb, 256, 0, st>>>(n, z, p, sc, 0);
            scalars_kernel<<<1, 1, 0, st>>>(sc, 1);
            s->launches += 3;
        }
    }
    MGB_LAUNCH_CHECK();
    if (f32) { cast_kernel2<double, float><<<nb, 256, 0, st>>>(n, x, (float*)d_x); ++s->launches; }
    MGB_CUDA(cudaStreamSynchronize(st));
    if (iters_out) *iters_out = it;
    if (rel_out) *rel_out = rel;
    return status;
}

}  // namespace
}  // namespace mgb

using namespace mgb;

extern "C" int mg_pcg_solve(mg_solver* s, void* d_x, const void* d_b, double tol, int max_iter, int* iters_out, double* relres_out) {
    if (!s || !d_x || !d_b || max_iter < 0 || !(tol >= 0.0)) { set_error("mg_pcg_solve: invalid argument"); return MG_EINVAL; }
    const LevelData& L = s->lv[0];
    if (s->p.nu_pre != s->p.nu_post || s->p.nu_pre < 1) {
        set_error("mg_pcg_solve: the preconditioner needs nu_pre == nu_post >= 1 (a symmetric cycle)");
        return MG_EINVAL;
    }
    if (!march_supported(L.nx, L.ny, L.nz, L.hx, L.hy, L.hz)) {
        set_error("mg_pcg_solve: needs a uniform grid with nx %% 4 == 0");
        return MG_EINVAL;
    }
    int prev = -1;
    cudaGetDevice(&prev);
    cudaSetDevice(s->device);
    s->history.clear(); s->history_cycles.clear();
    const int rc = s->dtype == MG_F32 ? pcg_t<float>(s, d_x, d_b, tol, max_iter, iters_out, relres_out)
                                      : pcg_t<double>(s, d_x, d_b, tol, max_iter, iters_out, relres_out);
    if (prev >= 0) cudaSetDevice(prev);
    return rc;
}
