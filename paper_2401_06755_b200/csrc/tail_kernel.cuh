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
__device__ __forceinline__ void stencil_pass(const Lv& Lr, const float* __restrict__ sfac, float omega) {
    // local copies: the level descriptors live in a dynamically indexed (local-memory) array
    const int nx = Lr.nx, ny = Lr.ny, nz = Lr.nz, n = Lr.n;
    const float ce = Lr.ce, cc = Lr.cc;
    const float* __restrict__ X = Lr.X; const float* __restrict__ K = Lr.K;
    const float* __restrict__ B = Lr.B; const float* __restrict__ DI = Lr.DI;
    float* __restrict__ Y = Lr.Y;
    const float s0 = sfac[0], s1 = sfac[1], s2 = sfac[2], s3 = sfac[3], s4 = sfac[4], s5 = sfac[5];
    for (int idx = threadIdx.x; idx < n; idx += NT) {
        const int i = idx % nx, t = idx / nx, j = t % ny, k = t / ny;
        const float xi = X[idx], ki = K[idx];
        float ax0 = 0.f, ax1 = 0.f;
#pragma unroll
        for (int c = -1; c <= 1; ++c) {
            int kk = k + c; float fz = 1.f;
            if (kk < 0) { kk = 0; fz = s4; } else if (kk >= nz) { kk = nz - 1; fz = s5; }
#pragma unroll
            for (int b = -1; b <= 1; ++b) {
                int jj = j + b; float fy = fz;
                if (jj < 0) { jj = 0; fy *= s2; } else if (jj >= ny) { jj = ny - 1; fy *= s3; }
                const int row = (kk * ny + jj) * nx;
#pragma unroll
                for (int a = -1; a <= 1; ++a) {
                    const int m = (a != 0) + (b != 0) + (c != 0);
                    if (m < 2) continue;
                    int ii = i + a; float f = fy;
                    if (ii < 0) { ii = 0; f *= s0; } else if (ii >= nx) { ii = nx - 1; f *= s1; }
                    const float w = (m == 2) ? ce : cc;
                    if ((a + b + c) & 1) ax1 = fmaf(w * (ki + K[row + ii]), xi - f * X[row + ii], ax1);
                    else ax0 = fmaf(w * (ki + K[row + ii]), xi - f * X[row + ii], ax0);
                }
            }
        }
        const float r = B[idx] - (ax0 + ax1);
        Y[idx] = MODE == 0 ? fmaf(omega * DI[idx], r, xi) : r;
    }
}

// ---- strip path for levels with several points per thread (n > NT, nx % 4 == 0) ----------------
// One thread updates a strip of 4 consecutive x points from the 8 neighbouring rows (dy, dz) != (0, 0)
// read as float4 plus the two end neighbours.  Eq. 13 form with integer weights (stream_kernel.cuh):
//   S(f) = sum over the 4 rows with |dy| + |dz| = 1 of 2 R  +  sum over the 4 rows with |dy| = |dz| = 1 of (R + 2 f),
//   R(c) = f(c-1) + f(c+1);   A x = x / DI - cc (k S(x) + S(k x)),  1/DI = D precomputed per level.
template <int MODE>
__device__ __forceinline__ void strip_pass(const Lv& Lr, const float* __restrict__ sfac, float omega) {
    const int nx = Lr.nx, ny = Lr.ny, nz = Lr.nz, sx = nx >> 2, ns = Lr.n >> 2;
    const float cc = Lr.cc;
    const float* __restrict__ X = Lr.X; const float* __restrict__ K = Lr.K;
    const float* __restrict__ B = Lr.B; const float* __restrict__ DI = Lr.DI;
    float* __restrict__ Y = Lr.Y;
    const float s0 = sfac[0], s1 = sfac[1], s2 = sfac[2], s3 = sfac[3], s4 = sfac[4], s5 = sfac[5];
    for (int sidx = threadIdx.x; sidx < ns; sidx += NT) {
        const int i0 = 4 * (sidx % sx), t = sidx / sx, j = t % ny, k = t / ny;
        const bool lin = i0 > 0, rin = i0 + 4 < nx;
        float Sx[4] = {0.f, 0.f, 0.f, 0.f}, Sz[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
        for (int c = -1; c <= 1; ++c) {
            int kk = k + c; float fz = 1.f;
            if (kk < 0) { kk = 0; fz = s4; } else if (kk >= nz) { kk = nz - 1; fz = s5; }
#pragma unroll
            for (int b = -1; b <= 1; ++b) {
                if (b == 0 && c == 0) continue;
                int jj = j + b; float f = fz;
                if (jj < 0) { jj = 0; f *= s2; } else if (jj >= ny) { jj = ny - 1; f *= s3; }
                const int row = (kk * ny + jj) * nx + i0;
                const float4 v4 = *reinterpret_cast<const float4*>(X + row);
                const float4 q4 = *reinterpret_cast<const float4*>(K + row);
                float v[6] = {0.f, v4.x, v4.y, v4.z, v4.w, 0.f}, q[6] = {0.f, q4.x, q4.y, q4.z, q4.w, 0.f};
                v[0] = lin ? X[row - 1] : s0 * v4.x; v[5] = rin ? X[row + 4] : s1 * v4.w;
                q[0] = lin ? K[row - 1] : q4.x;      q[5] = rin ? K[row + 4] : q4.w;
                float z[6];
#pragma unroll
                for (int e = 0; e < 6; ++e) { v[e] *= f; z[e] = q[e] * v[e]; }
                const bool corner = (b != 0) && (c != 0);
#pragma unroll
                for (int e = 0; e < 4; ++e) {
                    const float Rx = v[e] + v[e + 2], Rz = z[e] + z[e + 2];
                    if (corner) { Sx[e] += fmaf(2.f, v[e + 1], Rx); Sz[e] += fmaf(2.f, z[e + 1], Rz); }
                    else { Sx[e] = fmaf(2.f, Rx, Sx[e]); Sz[e] = fmaf(2.f, Rz, Sz[e]); }
                }
            }
        }
        const int idx = (k * ny + j) * nx + i0;
        const float4 x4 = *reinterpret_cast<const float4*>(X + idx), k4 = *reinterpret_cast<const float4*>(K + idx);
        const float4 b4 = *reinterpret_cast<const float4*>(B + idx), d4 = *reinterpret_cast<const float4*>(DI + idx);
        const float xv[4] = {x4.x, x4.y, x4.z, x4.w}, kv[4] = {k4.x, k4.y, k4.z, k4.w};
        const float bv[4] = {b4.x, b4.y, b4.z, b4.w}, dv[4] = {d4.x, d4.y, d4.z, d4.w};
        float o[4];
#pragma unroll
        for (int e = 0; e < 4; ++e) {
            const float u = fmaf(cc, fmaf(kv[e], Sx[e], Sz[e]), bv[e]);          // b + cc (k S(x) + S(k x))
            o[e] = MODE == 0 ? fmaf(omega * dv[e], u, (1.f - omega) * xv[e]) : u - __fdividef(xv[e], dv[e]);
        }
        *reinterpret_cast<float4*>(Y + idx) = make_float4(o[0], o[1], o[2], o[3]);
    }
}

template <int MODE>
__device__ __forceinline__ void level_pass(const Lv& L, const float* s, float omega) {
    if ((L.nx & 3) == 0) strip_pass<MODE>(L, s, omega); else stencil_pass<MODE>(L, s, omega);
}

// ---- register-resident path for levels with at most one point per thread (n <= NT) ----------
// Each thread keeps the 20 folded neighbour weights w^_j = omega/D c_j (k_i + k_j) f_j (f_j = product of
// the halo factors of the ghost neighbour) and the neighbours' shared-memory indices of ITS point, so a
// sweep is 20 shared loads and 21 FMAs:  t = omega/D (b - A x) = sc b - dh x_i + sum_j w^_j x_j,  x' = x + t,
// and the residual is t / sc.  Only the warps that own points take part (named barrier 1).
struct RegPt { float w[20]; int i[20]; float dh, sc; };

__device__ __forceinline__ void reg_setup(const Lv& L, const float* __restrict__ s, float omega, RegPt& R) {
    const int idx = threadIdx.x < L.n ? threadIdx.x : 0;
    const int i = idx % L.nx, t = idx / L.nx, j = t % L.ny, k = t / L.ny;
    const float ki = L.K[idx], od = omega * L.DI[idx];
    float dsum = 0.f;
    int q = 0;
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
                const float w = ((m == 2) ? L.ce : L.cc) * (ki + L.K[row + ii]);
                dsum += w;
                R.w[q] = od * w * f;
                R.i[q] = row + ii;
                ++q;
            }
        }
    }
    R.dh = od * dsum;
    R.sc = od;
}

__device__ __forceinline__ float reg_t(const RegPt& R, const float* __restrict__ X, float xi, float bi) {
    float t0 = fmaf(-R.dh, xi, R.sc * bi), t1 = 0.f, t2 = 0.f, t3 = 0.f;
#pragma unroll
    for (int q = 0; q < 20; q += 4) {
        t0 = fmaf(R.w[q], X[R.i[q]], t0); t1 = fmaf(R.w[q + 1], X[R.i[q + 1]], t1);
        t2 = fmaf(R.w[q + 2], X[R.i[q + 2]], t2); t3 = fmaf(R.w[q + 3], X[R.i[q + 3]], t3);
    }
    return (t0 + t1) + (t2 + t3);
}

__device__ __forceinline__ void bar_part(int nthreads) {
    asm volatile("bar.sync 1, %0;" ::"r"(nthreads) : "memory");
}

// `n` sweeps on a small level, then (RES) the residual into Y.  Ends with a block-wide barrier.
template <bool RES>
__device__ __forceinline__ void reg_level(Lv& L, const float* s, float omega, int n) {
    const int nact = ((L.n + 31) / 32) * 32;
    if ((int)threadIdx.x < nact) {
        RegPt R;
        reg_setup(L, s, omega, R);
        const bool on = (int)threadIdx.x < L.n;
        const int idx = on ? threadIdx.x : 0;
        const float bi = L.B[idx];
        float xi = L.X[idx];
        float* X = L.X; float* Y = L.Y;
        for (int it = 0; it < n; ++it) {
            xi += reg_t(R, X, xi, bi);
            if (on) Y[idx] = xi;
            bar_part(nact);
            float* t = X; X = Y; Y = t;
        }
        if (RES) {
            const float r = reg_t(R, X, xi, bi) / R.sc;
            if (on) Y[idx] = r;
        }
    }
    if (n & 1) { float* t = L.X; L.X = L.Y; L.Y = t; }
    __syncthreads();
}

__device__ __forceinline__ void sweeps(Lv& L, const float* s, float omega, int n) {
    if (L.n <= NT) { reg_level<false>(L, s, omega, n); return; }
    for (int it = 0; it < n; ++it) {
        level_pass<0>(L, s, omega);
        __syncthreads();
        float* t = L.X; L.X = L.Y; L.Y = t;
    }
}

// nu sweeps followed by the residual into Y
__device__ __forceinline__ void sweeps_residual(Lv& L, const float* s, float omega, int n) {
    if (L.n <= NT) { reg_level<true>(L, s, omega, n); return; }
    sweeps(L, s, omega, n);
    level_pass<1>(L, s, omega);
    __syncthreads();
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
        }
    }
    // Programmatic dependent launch: the coefficient data above is static during a cycle; x and b of the tail's finest
    // level come from the previous kernel.
    asm volatile("griddepcontrol.wait;" ::: "memory");
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    for (int idx = threadIdx.x; idx < lv[0].n; idx += NT) { lv[0].X[idx] = P.x[idx]; lv[0].B[idx] = P.b[idx]; }
    __syncthreads();
    const float omega = P.omega;
    const int last = P.nlev - 1;
    // ---- down leg ----
    for (int t = 0; t < last; ++t) {
        Lv& L = lv[t];
        Lv& C = lv[t + 1];
        const int done = (t == 0) ? P.first_done : ((P.nu_pre >= 1) ? 1 : 0);
        sweeps_residual(L, s, omega, max(0, P.nu_pre - done));   // residual into Y
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
