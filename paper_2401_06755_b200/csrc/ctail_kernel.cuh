// ctail_kernel.cuh -- the coarse tail of the V-cycle on one thread-block CLUSTER (8 blocks, distributed shared
// memory): every level from 16^3-sized grids down is smoothed, restricted, solved and prolonged without leaving
// the chip and without a kernel boundary (north_star: "small coarse levels run as single-CTA or cooperative
// kernels"; SURVEY hard part 6).  It spreads the work tail_kernel.cuh does in ONE block over 8 SMs: 29 us instead of
// 41 us for 16^3 + 8^3 + 4^3 at V(2,2) with 50 coarse sweeps.  (It can hold a 32^3 level too, but five lean_kernel
// launches are faster for that; the host picks.)
//
// Distribution.  A "distributed" level (nz a multiple of 8) is cut into 8 z slabs, one per block of the cluster.
// Each block keeps its slab of x (two buffers), k, b, 1/D in shared memory; x and k carry one halo plane below and
// above.  After every pass that changes x the blocks store their first / last plane into the neighbours' halo
// planes through distributed shared memory and meet at a cluster barrier; the blocks at the domain faces fill
// their outer halo with the boundary rule ghost = s * mirror.  Restriction and prolongation between
// distributed levels are local to a block (the 2:1 coarsening maps slab to slab).  Levels with nz < 8 ("solo"
// levels, e.g. 4^3) live in block 0 and run the single-block code of tail_kernel.cuh; the last distributed level
// sends its in-plane child sums there and fetches the correction back through distributed shared memory.
//
// Arithmetic: the integer-weight form of Eq. 13 on a uniform grid (as lean_kernel.cuh / tail_kernel.cuh strip_pass):
//   S(f) = 2 E(f) + Cn(f),   A x = x / DI - cc (k S(x) + S(k x)),   DI = 1 / D precomputed per level.
#pragma once
#include <cooperative_groups.h>
#include <cuda_runtime.h>

#include "tail_kernel.cuh"

namespace mgb {
namespace ck {

namespace cg = cooperative_groups;

constexpr int NC = 8;        // blocks per cluster
constexpr int NT = tk::NT;   // 512 threads per block
constexpr int MAXD = 3;      // distributed levels
constexpr int MAXS = 2;      // solo levels

struct CParams {
    int nd, ns;                               // distributed / solo level counts (ns >= 1)
    int nx[MAXD + MAXS], ny[MAXD + MAXS], nz[MAXD + MAXS];
    const float* k[MAXD + MAXS];              // NULL: constant coefficient
    const float* dinv[MAXD + MAXS];           // 1/D per point (variable k)
    float ce[MAXD + MAXS], cc[MAXD + MAXS], dinv_const[MAXD + MAXS];
    float s[6];
    float omega;
    int nu_pre, nu_post, coarse_sweeps;
    int first_done;                           // the parent already applied the first sweep to x (level 0 of the tail)
    float* x;                                 // level-0 iterate of the tail (in / out)
    const float* b;                           // level-0 right-hand side
    // The coarsest solve (coarse_sweeps Jacobi sweeps from a zero guess) is a fixed linear map x = M b of the n_c coarsest
    // points; when the host has tabulated it (n_c <= 64; cmat[j * n_c + i] = M_ij, rebuilt when the coefficient or the
    // parameters change) one n_c x n_c product replaces the serial chain of sweeps.  NULL: run the sweeps.
    const float* cmat;
};

// one block's slab of a distributed level
struct Slab {
    int nx, ny, nzl, ps;        // ps = nx * ny; nzl local planes
    float cc;
    float *X, *Y;               // (nzl + 2) planes each: plane 0 / nzl + 1 are the halos
    float *K;                   // (nzl + 2) planes
    float *B, *DI;              // nzl planes
};

// MODE 0: Y = weighted-Jacobi sweep of X;  MODE 1: Y = B - A X.  Strips of 4 x points; z neighbours come from the
// halo planes, x / y ghosts by clamping with the face factor.
template <int MODE>
__device__ __forceinline__ void slab_pass(const Slab& L, const float* __restrict__ sfac, float omega) {
    const int nx = L.nx, ny = L.ny, sx = nx >> 2, ns = (L.nzl * L.ps) >> 2;
    const float cc = L.cc;
    const float* __restrict__ X = L.X; const float* __restrict__ K = L.K;
    float* __restrict__ Y = L.Y;
    const float s0 = sfac[0], s1 = sfac[1], s2 = sfac[2], s3 = sfac[3];
    for (int sidx = threadIdx.x; sidx < ns; sidx += NT) {
        const int i0 = 4 * (sidx % sx), t = sidx / sx, j = t % ny, zl = t / ny + 1;
        const bool lin = i0 > 0, rin = i0 + 4 < nx;
        float Sx[4] = {0.f, 0.f, 0.f, 0.f}, Sz[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
        for (int c = -1; c <= 1; ++c) {
#pragma unroll
            for (int b = -1; b <= 1; ++b) {
                if (b == 0 && c == 0) continue;
                int jj = j + b; float f = 1.f;
                if (jj < 0) { jj = 0; f = s2; } else if (jj >= ny) { jj = ny - 1; f = s3; }
                const int row = (zl + c) * L.ps + jj * nx + i0;
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
        const int idx = zl * L.ps + j * nx + i0, idb = idx - L.ps;
        const float4 x4 = *reinterpret_cast<const float4*>(X + idx), k4 = *reinterpret_cast<const float4*>(K + idx);
        const float4 b4 = *reinterpret_cast<const float4*>(L.B + idb), d4 = *reinterpret_cast<const float4*>(L.DI + idb);
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

// Halo exchange of the current iterate X of a distributed level: first / last own plane into the neighbours' halo
// planes (distributed shared memory), boundary rule at the domain faces, then a cluster barrier.
__device__ __forceinline__ void exchange(cg::cluster_group& cl, const Slab& L, int rank, const float* __restrict__ sfac) {
    float* X = L.X;
    const int ps = L.ps, top = (L.nzl + 1) * ps;
    float* below = rank > 0 ? cl.map_shared_rank(X, rank - 1) : nullptr;
    float* above = rank < NC - 1 ? cl.map_shared_rank(X, rank + 1) : nullptr;
    const float s4 = sfac[4], s5 = sfac[5];
    for (int e = 4 * threadIdx.x; e < ps; e += 4 * NT) {
        const float4 lo = *reinterpret_cast<const float4*>(X + ps + e), hi = *reinterpret_cast<const float4*>(X + L.nzl * ps + e);
        if (below) *reinterpret_cast<float4*>(below + top + e) = lo;
        else *reinterpret_cast<float4*>(X + e) = make_float4(s4 * lo.x, s4 * lo.y, s4 * lo.z, s4 * lo.w);
        if (above) *reinterpret_cast<float4*>(above + e) = hi;
        else *reinterpret_cast<float4*>(X + top + e) = make_float4(s5 * hi.x, s5 * hi.y, s5 * hi.z, s5 * hi.w);
    }
    cl.sync();
}

__device__ __forceinline__ void cpa4(float* dst, const float* src) {      // 4-byte asynchronous copy global -> shared
    asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"((uint32_t)__cvta_generic_to_shared(dst)), "l"(src) : "memory");
}

__device__ __forceinline__ void swap_xy(Slab& L) { float* t = L.X; L.X = L.Y; L.Y = t; }

__global__ void __cluster_dims__(NC, 1, 1) __launch_bounds__(NT, 1) ctail_kernel(const CParams P) {
    cg::cluster_group cl = cg::this_cluster();
    const int rank = (int)cl.block_rank(), tid = threadIdx.x;
    extern __shared__ __align__(16) float sm[];
    __shared__ float s[6];
    Slab sl[MAXD];
    tk::Lv lv[MAXS];
    if (tid < 6) s[tid] = P.s[tid];
    const int nd = P.nd, ns = P.ns;

    // ---- identical shared-memory layout in every block of the cluster ----
    float* p = sm;
#pragma unroll
    for (int t = 0; t < MAXD; ++t) {
        if (t >= nd) break;
        Slab& L = sl[t];
        L.nx = P.nx[t]; L.ny = P.ny[t]; L.nzl = P.nz[t] / NC; L.ps = L.nx * L.ny; L.cc = P.cc[t];
        L.X = p; p += (L.nzl + 2) * L.ps; L.Y = p; p += (L.nzl + 2) * L.ps; L.K = p; p += (L.nzl + 2) * L.ps;
        L.B = p; p += L.nzl * L.ps; L.DI = p; p += L.nzl * L.ps;
    }
#pragma unroll
    for (int u = 0; u < MAXS; ++u) {
        if (u >= ns) break;
        tk::Lv& L = lv[u];
        L.nx = P.nx[nd + u]; L.ny = P.ny[nd + u]; L.nz = P.nz[nd + u]; L.n = L.nx * L.ny * L.nz;
        L.ce = P.ce[nd + u]; L.cc = P.cc[nd + u];
        L.X = p; L.Y = p + L.n; L.B = p + 2 * L.n; L.K = p + 3 * L.n; L.DI = p + 4 * L.n;
        p += 5 * L.n;
    }
    const int cps = (sl[nd - 1].nx >> 1) * (sl[nd - 1].ny >> 1);     // in-plane size of the first solo level
    float* part = p; p += NC * cps;                                   // block 0: in-plane child sums of every block's plane
    float* sres = p;                                                  // block 0: result of the solo cycle (lv[0].n floats)

    // ---- static data: coefficient slabs with copy halos, 1/D; solo levels in block 0 ----
    // All of it by asynchronous copies (cp.async, 4 bytes each) with ONE wait at the end: as plain loads the five loops below were five
    // dependent round trips to L2 / HBM (4.4 us, most of it exposed: the predecessor in the stream is a 3 us kernel).
#pragma unroll
    for (int t = 0; t < MAXD; ++t) {
        if (t >= nd) break;
        const Slab& L = sl[t];
        const int nzg = P.nz[t];
        for (int e = tid; e < (L.nzl + 2) * L.ps; e += NT) {
            const int zl = e / L.ps, r = e - zl * L.ps;
            const int zg = min(max(rank * L.nzl + zl - 1, 0), nzg - 1);
            if (P.k[t]) cpa4(L.K + e, P.k[t] + (size_t)zg * L.ps + r); else L.K[e] = 1.f;
        }
        for (int e = tid; e < L.nzl * L.ps; e += NT) {
            if (P.dinv[t]) cpa4(L.DI + e, P.dinv[t] + (size_t)rank * L.nzl * L.ps + e); else L.DI[e] = P.dinv_const[t];
        }
    }
    if (rank == 0) {
#pragma unroll
        for (int u = 0; u < MAXS; ++u) {
            if (u >= ns) break;
            const tk::Lv& L = lv[u];
            for (int idx = tid; idx < L.n; idx += NT) {
                if (P.k[nd + u]) cpa4(L.K + idx, P.k[nd + u] + idx); else L.K[idx] = 1.f;
                if (P.dinv[nd + u]) cpa4(L.DI + idx, P.dinv[nd + u] + idx); else L.DI[idx] = P.dinv_const[nd + u];
            }
        }
    }
    // Programmatic dependent launch: x and b of the tail's finest level come from the previous kernel
    asm volatile("griddepcontrol.wait;" ::: "memory");
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    {
        const Slab& L = sl[0];
        const int nzg = P.nz[0];
        for (int e = tid; e < (L.nzl + 2) * L.ps; e += NT) {          // x with its halo planes straight from global memory
            const int zl = e / L.ps, r = e - zl * L.ps;
            const int z = rank * L.nzl + zl - 1;
            if (z >= 0 && z < nzg) cpa4(L.X + e, P.x + (size_t)z * L.ps + r);
            else L.X[e] = (z < 0 ? P.s[4] : P.s[5]) * P.x[(size_t)(z < 0 ? 0 : nzg - 1) * L.ps + r];      // ghost plane = s * mirror
        }
        for (int e = tid; e < L.nzl * L.ps; e += NT) cpa4(L.B + e, P.b + (size_t)rank * L.nzl * L.ps + e);
    }
    asm volatile("cp.async.wait_all;" ::: "memory");
    cl.sync();       // every block of the cluster is running and has its data: distributed shared memory may be used from here

    const float omega = P.omega;
    const int nlev = nd + ns;
    // ---- down leg over the distributed levels ----
    for (int t = 0; t < nd; ++t) {
        Slab& L = sl[t];
        const int done = (t == 0) ? P.first_done : ((P.nu_pre >= 1) ? 1 : 0);
        for (int it = 0; it < max(0, P.nu_pre - done); ++it) {
            slab_pass<0>(L, s, omega);
            __syncthreads();
            swap_xy(L);
            exchange(cl, L, rank, s);
        }
        slab_pass<1>(L, s, omega);                                  // residual into Y
        __syncthreads();
        const int first = (t + 1 == nlev - 1) ? (P.coarse_sweeps >= 1) : (P.nu_pre >= 1);
        if (t + 1 < nd) {                                           // 8-child mean: slab to slab, local
            Slab& C = sl[t + 1];
            for (int idx = tid; idx < C.nzl * C.ps; idx += NT) {
                const int i = idx % C.nx, q = idx / C.nx, j = q % C.ny, zc = q / C.ny;       // zc = 0 .. nzl_c - 1
                float sum = 0.f;
#pragma unroll
                for (int dk = 0; dk < 2; ++dk)
#pragma unroll
                    for (int dj = 0; dj < 2; ++dj) {
                        const int row = (2 * zc + 1 + dk) * L.ps + (2 * j + dj) * L.nx + 2 * i;
                        sum += L.Y[row] + L.Y[row + 1];
                    }
                const float bc = 0.125f * sum;
                C.B[idx] = bc;
                C.X[C.ps + idx] = first ? omega * C.DI[idx] * bc : 0.f;
            }
            __syncthreads();
            exchange(cl, C, rank, s);
        } else {                                                    // children live in block 0: send in-plane sums of the own plane
            float* part0 = cl.map_shared_rank(part, 0);
            const int cnx = L.nx >> 1;
            for (int idx = tid; idx < cps; idx += NT) {
                const int i = idx % cnx, j = idx / cnx;
                const int row = L.ps + (2 * j) * L.nx + 2 * i;
                part0[rank * cps + idx] = (L.Y[row] + L.Y[row + 1]) + (L.Y[row + L.nx] + L.Y[row + L.nx + 1]);
            }
            cl.sync();
        }
    }

    // ---- solo levels: the single-block cycle of tail_kernel.cuh in block 0 ----
    if (rank == 0) {
        const int last = ns - 1;
        {
            tk::Lv& C = lv[0];
            const int first = (nd == nlev - 1) ? (P.coarse_sweeps >= 1) : (P.nu_pre >= 1);
            for (int idx = tid; idx < C.n; idx += NT) {
                const int k = idx / cps, r = idx - k * cps;
                const float bc = 0.125f * (part[(2 * k) * cps + r] + part[(2 * k + 1) * cps + r]);
                C.B[idx] = bc;
                C.X[idx] = first ? omega * C.DI[idx] * bc : 0.f;
            }
        }
        __syncthreads();
        for (int u = 0; u < last; ++u) {                            // down leg
            tk::Lv& L = lv[u];
            tk::Lv& C = lv[u + 1];
            const int done = (P.nu_pre >= 1) ? 1 : 0;
            tk::sweeps_residual(L, s, omega, max(0, P.nu_pre - done));
            const int first = (u + 1 == last) ? (P.coarse_sweeps >= 1) : (P.nu_pre >= 1);
            for (int idx = tid; idx < C.n; idx += NT) {
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
        if (P.cmat) {                                               // coarsest: x = M b
            tk::Lv& L = lv[last];
            if (tid < L.n) {
                const float* __restrict__ m = P.cmat + tid;
                float a0 = 0.f, a1 = 0.f, a2 = 0.f, a3 = 0.f;
#pragma unroll 4
                for (int j = 0; j < L.n; j += 4) {
                    a0 = fmaf(m[(j + 0) * L.n], L.B[j + 0], a0); a1 = fmaf(m[(j + 1) * L.n], L.B[j + 1], a1);
                    a2 = fmaf(m[(j + 2) * L.n], L.B[j + 2], a2); a3 = fmaf(m[(j + 3) * L.n], L.B[j + 3], a3);
                }
                L.X[tid] = (a0 + a1) + (a2 + a3);
            }
            __syncthreads();
        } else {
            tk::sweeps(lv[last], s, omega, max(0, P.coarse_sweeps - ((P.coarse_sweeps >= 1) ? 1 : 0)));   // coarsest
        }
        for (int u = last - 1; u >= 0; --u) {                       // up leg
            tk::Lv& L = lv[u];
            tk::Lv& C = lv[u + 1];
            for (int idx = tid; idx < L.n; idx += NT) {
                const int i = idx % L.nx, q = idx / L.nx, j = q % L.ny, k = q / L.ny;
                L.X[idx] += C.X[((k >> 1) * C.ny + (j >> 1)) * C.nx + (i >> 1)];
            }
            __syncthreads();
            tk::sweeps(L, s, omega, P.nu_post);
        }
        for (int idx = tid; idx < lv[0].n; idx += NT) sres[idx] = lv[0].X[idx];
    }
    cl.sync();

    // ---- up leg over the distributed levels ----
    for (int t = nd - 1; t >= 0; --t) {
        Slab& L = sl[t];
        if (t == nd - 1) {                                          // correction from block 0 (own plane = global plane `rank`)
            const float* src = cl.map_shared_rank(sres, 0);
            const int cnx = L.nx >> 1, cny = L.ny >> 1;
            for (int idx = tid; idx < L.ps; idx += NT) {
                const int i = idx % L.nx, j = idx / L.nx;
                L.X[L.ps + idx] += src[((rank >> 1) * cny + (j >> 1)) * cnx + (i >> 1)];
            }
        } else {
            const Slab& C = sl[t + 1];
            for (int idx = tid; idx < L.nzl * L.ps; idx += NT) {
                const int i = idx % L.nx, q = idx / L.nx, j = q % L.ny, zl = q / L.ny;         // zl = 0 .. nzl - 1
                L.X[L.ps + idx] += C.X[((zl >> 1) + 1) * C.ps + (j >> 1) * C.nx + (i >> 1)];
            }
        }
        __syncthreads();
        if (P.nu_post > 0) exchange(cl, L, rank, s);
        for (int it = 0; it < P.nu_post; ++it) {
            slab_pass<0>(L, s, omega);
            __syncthreads();
            swap_xy(L);
            if (it + 1 < P.nu_post) exchange(cl, L, rank, s);
        }
    }
    cl.sync();       // no block may exit while another still reads its shared memory
    {
        const Slab& L = sl[0];
        for (int e = tid; e < L.nzl * L.ps; e += NT) P.x[(size_t)rank * L.nzl * L.ps + e] = L.X[L.ps + e];
    }
}

}  // namespace ck
}  // namespace mgb
