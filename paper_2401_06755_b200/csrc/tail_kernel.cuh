// tail_kernel.cuh -- the coarse tail of the V-cycle in ONE thread block: every level whose grid
// fits in shared memory (<= 16^3 points at its finest) is smoothed, restricted, solved and
// prolonged on chip, so the small levels cost one launch instead of ~60 launch-bound ones
// (north_star: "small coarse levels run as single-CTA kernels"; SURVEY hard part 6).
//
// Same arithmetic as the generic kernels (difference form of Eq. 13, reading C2):
//   (A x)_i = sum_{j != i} c_j (k_i + k_j) (x_i - ghost x_j),  c_j = -w_ij / 2  (uniform grid: 12 edge
//   neighbours ce = 1/(12 h^2), 8 corner neighbours cc = 1/(24 h^2), face weights vanish),
//   sweep x' = x + omega (b - A x) / D with 1/D precomputed per level; constant k is k == 1.
#pragma once
#include <cuda_runtime.h>

namespace mgb {
namespace tk {

constexpr int MAXL = 6;
constexpr int NT = 512;

struct TailParams {
    int nlev;
    int nx[MAXL], ny[MAXL], nz[MAXL];
    const float* k[MAXL];      // NULL: constant coefficient
    const float* dinv[MAXL];   // 1/D per point (variable k)
    float ce[MAXL], cc[MAXL], dinv_const[MAXL];
    float s[6];
    float omega;
    int nu_pre, nu_post, coarse_sweeps;
    int first_done;            // the parent already applied the first sweep to x (level 0 of the tail)
    float* x;                  // level-0 iterate of the tail (in / out)
    const float* b;            // level-0 right-hand side
};

struct Lv { int nx, ny, nz, n; float ce, cc; float *X, *Y, *B, *K, *DI; };

// mode 0: Y = X + omega (B - A X) DI;  mode 1: Y = B - A X
template <int MODE>
__device__ __forceinline__ void stencil_pass(const Lv& L, const float* __restrict__ s, float omega) {
    for (int idx = threadIdx.x; idx < L.n; idx += NT) {
        const int i = idx % L.nx, t = idx / L.nx, j = t % L.ny, k = t / L.ny;
        const float xi = L.X[idx], ki = L.K[idx];
        float ax = 0.f;
#pragma unroll
        for (int c = -1; c <= 1; ++c) {
            int kk = k + c; float fz = 1.f;
            if (kk < 0) { kk = 0; fz = s[4]; } else if (kk >= L.nz) { kk = L.nz - 1; fz = s[5]; }
#pragma unroll
            for (int b = -1; b <= 1; ++b) {
                int jj = j + b; float fy = fz;
                if (jj < 0) { jj = 0; fy *= s[2]; } else if (jj >= L.ny) { jj = L.ny - 1; fy *= s[3]; }
                const int row = (kk * L.ny + jj) * L.nx;
#pragma unroll
                for (int a = -1; a <= 1; ++a) {
                    const int m = (a != 0) + (b != 0) + (c != 0);
                    if (m < 2) continue;
                    int ii = i + a; float f = fy;
                    if (ii < 0) { ii = 0; f *= s[0]; } else if (ii >= L.nx) { ii = L.nx - 1; f *= s[1]; }
                    const float w = (m == 2) ? L.ce : L.cc;
                    ax = fmaf(w * (ki + L.K[row + ii]), xi - f * L.X[row + ii], ax);
                }
            }
        }
        const float r = L.B[idx] - ax;
        L.Y[idx] = MODE == 0 ? fmaf(omega * L.DI[idx], r, xi) : r;
    }
}

__device__ __forceinline__ void sweeps(Lv& L, const float* s, float omega, int n) {
    for (int it = 0; it < n; ++it) {
        stencil_pass<0>(L, s, omega);
        __syncthreads();
        float* t = L.X; L.X = L.Y; L.Y = t;
    }
}

__global__ void __launch_bounds__(NT, 1) tail_kernel(const TailParams P) {
    extern __shared__ __align__(16) float sm[];
    __shared__ float s[6];
    Lv lv[MAXL];
    if (threadIdx.x < 6) s[threadIdx.x] = P.s[threadIdx.x];
    float* p = sm;
#pragma unroll
    for (int t = 0; t < MAXL; ++t) {
        if (t >= P.nlev) break;
        Lv& L = lv[t];
        L.nx = P.nx[t]; L.ny = P.ny[t]; L.nz = P.nz[t]; L.n = L.nx * L.ny * L.nz;
        L.ce = P.ce[t]; L.cc = P.cc[t];
        L.X = p; L.Y = p + L.n; L.B = p + 2 * L.n; L.K = p + 3 * L.n; L.DI = p + 4 * L.n;
        p += 5 * L.n;
        for (int idx = threadIdx.x; idx < L.n; idx += NT) {
            L.K[idx] = P.k[t] ? P.k[t][idx] : 1.f;
            L.DI[idx] = P.dinv[t] ? P.dinv[t][idx] : P.dinv_const[t];
            if (t == 0) { L.X[idx] = P.x[idx]; L.B[idx] = P.b[idx]; }
        }
    }
    __syncthreads();
    const float omega = P.omega;
    const int last = P.nlev - 1;
    // ---- down leg ----
    for (int t = 0; t < last; ++t) {
        Lv& L = lv[t];
        Lv& C = lv[t + 1];
        const int done = (t == 0) ? P.first_done : ((P.nu_pre >= 1) ? 1 : 0);
        sweeps(L, s, omega, max(0, P.nu_pre - done));
        stencil_pass<1>(L, s, omega);                  // residual into Y
        __syncthreads();
        const int first = (t + 1 == last) ? (P.coarse_sweeps >= 1) : (P.nu_pre >= 1);
        for (int idx = threadIdx.x; idx < C.n; idx += NT) {
            const int i = idx % C.nx, q = idx / C.nx, j = q % C.ny, k = q / C.ny;
            float sum = 0.f;
#pragma unroll
            for (int dk = 0; dk < 2; ++dk)
#pragma unroll
                for (int dj = 0; dj < 2; ++dj) {
                    const int row = ((2 * k + dk) * L.ny + 2 * j + dj) * L.nx + 2 * i;
                    sum += L.Y[row] + L.Y[row + 1];
                }
            const float bc = 0.125f * sum;
            C.B[idx] = bc;
            C.X[idx] = first ? omega * C.DI[idx] * bc : 0.f;
        }
        __syncthreads();
    }
    // ---- coarsest ----
    {
        const int done = (last == 0) ? P.first_done : ((P.coarse_sweeps >= 1) ? 1 : 0);
        sweeps(lv[last], s, omega, max(0, P.coarse_sweeps - done));
    }
    // ---- up leg ----
    for (int t = last - 1; t >= 0; --t) {
        Lv& L = lv[t];
        Lv& C = lv[t + 1];
        for (int idx = threadIdx.x; idx < L.n; idx += NT) {
            const int i = idx % L.nx, q = idx / L.nx, j = q % L.ny, k = q / L.ny;
            L.X[idx] += C.X[((k >> 1) * C.ny + (j >> 1)) * C.nx + (i >> 1)];
        }
        __syncthreads();
        sweeps(L, s, omega, P.nu_post);
    }
    for (int idx = threadIdx.x; idx < lv[0].n; idx += NT) P.x[idx] = lv[0].X[idx];
}

}  // namespace tk
}  // namespace mgb
