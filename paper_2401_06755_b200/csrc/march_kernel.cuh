// march_kernel.cuh -- z-marching residual kernel for uniform grids in any precision (sm_100a):
//   r = b - A x  (optionally stored; y = A x when b is NULL) and sum r^2 accumulated in fp64,
// used by the solve loops: TX = double, TB = float is the fp64 defect of the
// mixed-precision loop (reading C6 "fp32 reading", C8), TX = TB = double / float the plain loops.
//
// Same arithmetic as lean_kernel.cuh (reading C1/C2, Eqs. 8, 12-13 P:109-114, 146-159; uniform spacing:
// the face weights vanish, edge neighbours carry 2 cc, corner neighbours cc, cc = 1/(24 h^2)):
//   S(f)_i = 2 E(f)_i + Cn(f)_i,   r = b + cc (k S(x) + S(k x) - (32 k + S(k)) x)
//   constant coefficient: r = b + cc (2 S(x) - 64 x).
// A block owns a TX x TY column and marches along z.  Each plane of x and k is copied once into a
// 4-deep ring of shared tiles WITH its halo already evaluated (ghost = s * mirror; k ghosts are
// plain copies), so the arithmetic has no boundary cases.  Each thread owns 4 consecutive x points of one
// row, reads its 3 rows, forms the row sums R(c) = f(c-1) + f(c+1), T = R + 2 f and the in-plane sums
//   Dg = R_0 + R_2,  Pp = T_0 + T_2 + 2 R_1,   S[z] = Pp[z-1] + 2 Dg[z] + Pp[z+1]
// with two rolling accumulators per point and field.  One __syncthreads per plane; three planes are in flight (cp.async)
// while one is consumed.
#pragma once
#include <cuda_runtime.h>
#include <cstdint>

namespace mgb {
namespace mk {

struct MParams {
    int nx, ny, nz;
    int zchunk;
    double s[6];     // halo factors x-, x+, y-, y+, z-, z+
    double cc;       // 1 / (24 h^2)
    int dotx;        // accumulate sum out * x instead of sum out^2 (b = NULL: <x, A x>)
};

constexpr int LX = 16, LY = 16, NT = LX * LY;
constexpr int NSTG = 4;                       // ring of staged planes: 3 planes are in flight while one is consumed
constexpr int NBS = 8;                        // ring of staged right-hand-side rows (consumed one plane after x: > NSTG slots)
constexpr int TX = 4 * LX, TY = LY;
constexpr int PYS = TY + 2;
// Layout of one staged row (own columns 0 .. TX - 1, halo columns -1 and TX), chosen so that the 16-byte loads of a warp are
// bank-conflict free.  fp32: linear, [pad x3, halo, TX own, halo, pad x3]: a thread's 4 floats are one aligned 16-byte word
// and lanes are contiguous.  fp64: a thread's 4 doubles are two 16-byte pairs 32 bytes apart, a 4-way conflict if stored
// linearly (measured: 58 % of the shared-memory wavefronts were conflicts); so pairs are numbered pp = (col + 2) / 2 and the
// odd pairs (a thread's first pair, and its right neighbour) go to the first half of the row, the even pairs (second pair,
// left neighbour) to the second half -- each load of a warp then touches consecutive 16-byte slots.
template <typename T> struct Lay;
template <> struct Lay<float> {
    static constexpr int ROW = TX + 8;
    __host__ __device__ static constexpr int off(int col) { return 4 + col; }
    __host__ __device__ static constexpr int own0(int lx) { return 4 + 4 * lx; }       // columns c0, c0 + 1 (and c0 + 2, c0 + 3: same word)
    __host__ __device__ static constexpr int own1(int lx) { return 4 + 4 * lx + 2; }
};
template <> struct Lay<double> {
    static constexpr int HB = 2 * (LX + 1);          // start of the second half (even pairs), in elements
    static constexpr int ROW = HB + 2 * (LX + 2);
    __host__ __device__ static constexpr int off(int col) { return (((col + 2) >> 1) & 1 ? 0 : HB) + 2 * ((col + 2) >> 2) + ((col + 2) & 1); }
    __host__ __device__ static constexpr int own0(int lx) { return 2 * lx; }
    __host__ __device__ static constexpr int own1(int lx) { return HB + 2 * lx + 2; }
};

template <typename T> struct Vec4;
template <> struct Vec4<float> { typedef float4 type; };
template <> struct Vec4<double> { typedef double4 type; };

template <typename T>
__device__ __forceinline__ void load4(const T* p, T (&v)[4]) {
    if (sizeof(T) == 4) {
        const float4 t = *reinterpret_cast<const float4*>(p);
        v[0] = (T)t.x; v[1] = (T)t.y; v[2] = (T)t.z; v[3] = (T)t.w;
    } else {
        const double2 a = *reinterpret_cast<const double2*>(p), b = *reinterpret_cast<const double2*>(p + 2);
        v[0] = (T)a.x; v[1] = (T)a.y; v[2] = (T)b.x; v[3] = (T)b.y;
    }
}

// 4 own values from the staged row: one 16-byte word (fp32; p1 = p0 + 2 is the same word) or two 16-byte pairs (fp64)
template <typename T>
__device__ __forceinline__ void load22(const T* p0, const T* p1, T* v) {
    if (sizeof(T) == 4) {
        const float4 t = *reinterpret_cast<const float4*>(p0);
        v[0] = (T)t.x; v[1] = (T)t.y; v[2] = (T)t.z; v[3] = (T)t.w;
    } else {
        const double2 a = *reinterpret_cast<const double2*>(p0), b = *reinterpret_cast<const double2*>(p1);
        v[0] = (T)a.x; v[1] = (T)a.y; v[2] = (T)b.x; v[3] = (T)b.y;
    }
}

// in-plane sums of one field for the thread's 4 points from its 3 staged rows (each: l, v0..v3, r)
template <typename T>
__device__ __forceinline__ void plane_sums(const T (&f)[3][6], T (&Dg)[4], T (&Pp)[4]) {
    T R[3][4];
#pragma unroll
    for (int q = 0; q < 3; ++q)
#pragma unroll
        for (int c = 0; c < 4; ++c) R[q][c] = f[q][c] + f[q][c + 2];
#pragma unroll
    for (int c = 0; c < 4; ++c) {
        Dg[c] = R[0][c] + R[2][c];
        Pp[c] = (Dg[c] + T(2) * (f[0][c + 1] + f[2][c + 1])) + T(2) * R[1][c];
    }
}

template <typename TXT, typename TB, bool VAR, bool HASB>
__global__ void __launch_bounds__(NT, (sizeof(TXT) == 8 ? 1 : 2))
march_residual_kernel(const MParams P, const TXT* __restrict__ x, const TXT* __restrict__ kc, const TB* __restrict__ b,
                      TB* __restrict__ r, double* __restrict__ acc, float* __restrict__ yout = nullptr) {
    typedef TXT T;
    extern __shared__ __align__(16) unsigned char smraw[];
    T* sm = reinterpret_cast<T*>(smraw);
    constexpr int ROW = Lay<T>::ROW, PLANE = ROW * PYS;
    T* const xs = sm;                  // x planes [NSTG], then k planes [NSTG]
    T* const ks = sm + NSTG * PLANE;
    // right-hand side: every thread copies the 4 values of its own points (plane p rides in the commit group of x plane p)
    // and reads them back itself one plane later, so the global-load latency is off the critical path
    TB* const bs = reinterpret_cast<TB*>(sm + 2 * NSTG * PLANE);
    __shared__ double red[NT / 32];

    const int tid = threadIdx.x, lx = tid % LX, ly = tid / LX;
    const int nx = P.nx, ny = P.ny, nz = P.nz;
    const int x0 = blockIdx.x * TX, y0 = blockIdx.y * TY;
    const int zc0 = blockIdx.z * P.zchunk, zc1 = min(zc0 + P.zchunk, nz);
    const int gi0 = x0 + 4 * lx, gj = y0 + ly;
    const bool active = gi0 < nx && gj < ny;

    // staging: row rr of the tile <- global row y0 - 1 + rr (mirrored at the faces), in UNITS: the left halo cell (column -1),
    // TX / V aligned chunks of V elements (fp32: 16 bytes; fp64: single cells), the right halo cell (column TX).  nx is a multiple of 4, so the domain ends
    // on a chunk boundary: a chunk lies inside the domain or outside; of the chunks outside only the first element of the one
    // that starts at column nx is ever read (the ghost of column nx - 1) and is staged as a single cell.  Each thread stages
    // the same NE units of every plane: shared offsets, in-plane global offsets and the unit kinds are z-invariant.  The copy
    // is asynchronous (cp.async, global -> shared without registers) and overlaps the arithmetic of the current plane; ghost
    // cells are scaled in place by their owner afterwards.
    // fp64 stages every cell on its own (V = 1, no unit kinds: the code below compiles to the plain per-cell loop): 16-byte
    // chunks of two doubles were measured slower there (12.4 vs 11.2 ms for 20 solve cycles at 256^3, and 11.6 ms with the
    // unit bookkeeping alone), while fp32 gains (residual 106 -> 94 us)
    constexpr bool CHUNKED = sizeof(T) == 4;
    constexpr int V = CHUNKED ? 4 : 1, U = TX / V + 2, NUNIT = U * PYS, NE = (NUNIT + NT - 1) / NT;
    int soff[NE], goff[NE];
    unsigned lmask = 0;                  // bit e: unit e is staged at all
    unsigned cmask = 0;                  // bit e: unit e is a 16-byte chunk (else one cell)
    unsigned gmask = 0;                  // bit e: unit e is an x / y ghost (factor may differ from 1)
    auto xyfac = [&](int e) {            // halo factor of unit e (rare path)
        const int unit = tid + e * NT, rr = unit / U, u = unit - rr * U;
        const int gy = y0 - 1 + rr;
        T f = T(1);
        if (gy < 0) f *= (T)P.s[2]; else if (gy >= ny) f *= (T)P.s[3];
        if constexpr (!CHUNKED) {
            const int gx = x0 - 1 + u;
            if (gx < 0) f *= (T)P.s[0]; else if (gx >= nx) f *= (T)P.s[1];
        } else if (!((cmask >> e) & 1u)) {
            const int gx = u == 0 ? x0 - 1 : x0 + (u - 1) * V;     // a cell: the left halo, or the first column outside the domain
            if (gx < 0) f *= (T)P.s[0]; else if (gx >= nx) f *= (T)P.s[1];
        }
        return f;
    };
#pragma unroll
    for (int e = 0; e < NE; ++e) {
        if constexpr (!CHUNKED) {
            const int cell = min(tid + e * NT, NUNIT - 1);          // the surplus threads of the last round repeat the last cell
            const int rr = cell / U, cq = cell - rr * U;
            int gy = y0 - 1 + rr, gx = x0 - 1 + cq;
            bool gh = false;
            if (gy < 0) { gy = -1 - gy; gh = true; } else if (gy >= ny) { gy = 2 * ny - 1 - gy; gh = true; }
            if (gx < 0) { gx = -1 - gx; gh = true; } else if (gx >= nx) { gx = 2 * nx - 1 - gx; gh = true; }
            gy = min(max(gy, 0), ny - 1); gx = min(max(gx, 0), nx - 1);          // cells beyond a partial tile: any valid address
            soff[e] = rr * ROW + Lay<T>::off(cq - 1);
            goff[e] = gy * nx + gx;
            if (gh && tid + e * NT < NUNIT) gmask |= 1u << e;
            continue;
        }
        const int unit = tid + e * NT, rr = min(unit / U, PYS - 1), u = unit - (unit / U) * U;
        int gy = y0 - 1 + rr;
        bool gh = false;
        if (gy < 0) { gy = -1 - gy; gh = true; } else if (gy >= ny) { gy = 2 * ny - 1 - gy; gh = true; }
        gy = min(max(gy, 0), ny - 1);                                         // rows beyond a partial tile: any valid address
        const int col = u == 0 ? -1 : (u - 1) * V;                            // first column of the unit
        int gx = x0 + col;
        bool live = unit < NUNIT, chunk = CHUNKED && u != 0 && u != U - 1;
        if (gx < 0) { gx = 0; gh = true; }                                    // left halo at the domain face: mirror of column 0
        else if (gx == nx) { gx = nx - 1; gh = true; chunk = false; }         // first column outside: mirror of column nx - 1
        else if (gx > nx) { gx = 0; live = false; }                           // never read
        soff[e] = rr * ROW + Lay<T>::off(col);
        goff[e] = gy * nx + gx;
        if (live) lmask |= 1u << e;
        if (live && chunk) cmask |= 1u << e;
        if (live && gh) gmask |= 1u << e;
    }
    const uint32_t xs_a = (uint32_t)__cvta_generic_to_shared(xs), ks_a = (uint32_t)__cvta_generic_to_shared(ks);
    const uint32_t bs_a = (uint32_t)__cvta_generic_to_shared(bs + 4 * tid);
    const TB* const bcol = HASB ? b + (size_t)gj * nx + gi0 : nullptr;
    auto stage = [&](int p) {            // issue the copies of plane p
        const int zs = p < 0 ? -1 - p : (p >= nz ? 2 * nz - 1 - p : p);
        const size_t zoff = (size_t)zs * ny * nx;
        const uint32_t bo = (uint32_t)((p & (NSTG - 1)) * PLANE);
#pragma unroll
        for (int e = 0; e < NE; ++e) {
            if (CHUNKED && !((lmask >> e) & 1u)) continue;
            const uint32_t so = (bo + (uint32_t)soff[e]) * (uint32_t)sizeof(T);
            if (CHUNKED && ((cmask >> e) & 1u)) {
                asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(xs_a + so), "l"(x + zoff + goff[e]) : "memory");
                if (VAR) asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(ks_a + so), "l"(kc + zoff + goff[e]) : "memory");
            } else if (sizeof(T) == 4) {
                asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(xs_a + so), "l"(x + zoff + goff[e]) : "memory");
                if (VAR) asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(ks_a + so), "l"(kc + zoff + goff[e]) : "memory");
            } else {
                asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(xs_a + so), "l"(x + zoff + goff[e]) : "memory");
                if (VAR) asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(ks_a + so), "l"(kc + zoff + goff[e]) : "memory");
            }
        }
        if (HASB && active && p >= zc0 && p < zc1) {
            const uint32_t so = bs_a + (uint32_t)((p & (NBS - 1)) * NT * 4 * sizeof(TB));
            const TB* src = bcol + zoff;
            asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(so), "l"(src) : "memory");
            if (sizeof(TB) == 8) asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(so + 16), "l"(src + 2) : "memory");
        }
        asm volatile("cp.async.commit_group;" ::: "memory");
    };
    auto stage_finish = [&](int p) {     // wait for this thread's copies of plane p and scale its ghost cells
        asm volatile("cp.async.wait_group %0;" ::"n"(NSTG - 2) : "memory");     // every group but the NSTG - 2 newest has landed
        const bool zg = p < 0 || p >= nz;
        if (gmask || zg) {
            const T fz = p < 0 ? (T)P.s[4] : (p >= nz ? (T)P.s[5] : T(1));
            T* xd = xs + (p & (NSTG - 1)) * PLANE;
#pragma unroll
            for (int e = 0; e < NE; ++e)
                if ((CHUNKED ? ((lmask >> e) & 1u) != 0u : tid + e * NT < NUNIT) && (zg || ((gmask >> e) & 1u))) {
                    const T f = fz * xyfac(e);
                    if ((cmask >> e) & 1u) {
#pragma unroll
                        for (int c = 0; c < V; ++c) xd[soff[e] + c] *= f;
                    } else xd[soff[e]] *= f;
                }
        }
    };

    T xA[4], xB[4], zA[4], zB[4], kA[4], kB[4], xo[4], ko[4];
#pragma unroll
    for (int c = 0; c < 4; ++c) { xA[c] = xB[c] = zA[c] = zB[c] = kA[c] = kB[c] = xo[c] = T(0); ko[c] = T(1); }
    double sq = 0.0;
    const T cc = (T)P.cc;

    // one commit group per plane, empty past the end of the chunk, so that "all but the NSTG - 2 newest" always means
    // "up to the plane needed next"
    auto stage_or_skip = [&](int p) { if (p <= zc1) stage(p); else asm volatile("cp.async.commit_group;" ::: "memory"); };
#pragma unroll
    for (int d = 0; d < NSTG - 1; ++d) stage_or_skip(zc0 - 1 + d);
    stage_finish(zc0 - 1);
#pragma unroll 2
    for (int p = zc0 - 1; p <= zc1; ++p) {
        __syncthreads();                       // plane p is staged; everyone is done reading the other buffer
        stage_or_skip(p + NSTG - 1);           // asynchronous copy into the buffer plane p - 1 has just left
        T bv[4] = {T(0), T(0), T(0), T(0)};
        const int qc = p - 1;
        if (HASB && qc >= zc0 && active) {
            TB t4[4];
            load4<TB>(bs + ((qc & (NBS - 1)) * NT + tid) * 4, t4);
#pragma unroll
            for (int c = 0; c < 4; ++c) bv[c] = (T)t4[c];
        }
        const T* xr = xs + (p & (NSTG - 1)) * PLANE + ly * ROW;      // row ly - 1 of the tile = staged row ly
        const T* kr = ks + (p & (NSTG - 1)) * PLANE + ly * ROW;
        const int o0 = Lay<T>::own0(lx), o1 = Lay<T>::own1(lx), ol = Lay<T>::off(4 * lx - 1), orr = Lay<T>::off(4 * lx + 4);
        T fx[3][6], fk[3][6], fz[3][6];
#pragma unroll
        for (int q = 0; q < 3; ++q) {
            fx[q][0] = xr[q * ROW + ol]; fx[q][5] = xr[q * ROW + orr];
            load22<T>(xr + q * ROW + o0, xr + q * ROW + o1, &fx[q][1]);
            if (VAR) {
                fk[q][0] = kr[q * ROW + ol]; fk[q][5] = kr[q * ROW + orr];
                load22<T>(kr + q * ROW + o0, kr + q * ROW + o1, &fk[q][1]);
#pragma unroll
                for (int c = 0; c < 6; ++c) fz[q][c] = fk[q][c] * fx[q][c];
            }
        }
        T Dg[4], Pp[4], Sx[4], Sz[4], Sk[4];
        plane_sums<T>(fx, Dg, Pp);
#pragma unroll
        for (int c = 0; c < 4; ++c) { Sx[c] = xA[c] + Pp[c]; xA[c] = xB[c] + T(2) * Dg[c]; xB[c] = Pp[c]; }
        if (VAR) {
            plane_sums<T>(fz, Dg, Pp);
#pragma unroll
            for (int c = 0; c < 4; ++c) { Sz[c] = zA[c] + Pp[c]; zA[c] = zB[c] + T(2) * Dg[c]; zB[c] = Pp[c]; }
            plane_sums<T>(fk, Dg, Pp);
#pragma unroll
            for (int c = 0; c < 4; ++c) { Sk[c] = kA[c] + Pp[c]; kA[c] = kB[c] + T(2) * Dg[c]; kB[c] = Pp[c]; }
        }
        if (qc >= zc0 && active) {
            T rv[4];
#pragma unroll
            for (int c = 0; c < 4; ++c) {
                if (VAR) rv[c] = bv[c] + cc * ((ko[c] * Sx[c] + Sz[c]) - (T(32) * ko[c] + Sk[c]) * xo[c]);
                else rv[c] = bv[c] + cc * (T(2) * Sx[c] - T(64) * xo[c]);
                if (!HASB) rv[c] = -rv[c];       // no right-hand side: the output is y = A x
                sq += (double)rv[c] * (!HASB && P.dotx ? (double)xo[c] : (double)rv[c]);
            }
            if (yout) {                // r / D, D = cc (32 k + S(k)): the Jacobi seed of the next correction cycle
                float yv[4];
#pragma unroll
                for (int c = 0; c < 4; ++c) {
                    double rd;    // approximate reciprocal (as lean_kernel's own 1 / D): the seed feeds a smoother, not the iterate
                    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(rd) : "d"((double)(cc * (VAR ? T(32) * ko[c] + Sk[c] : T(64)))));
                    yv[c] = (float)((double)rv[c] * rd);
                }
                *reinterpret_cast<float4*>(yout + ((size_t)qc * ny + gj) * nx + gi0) = make_float4(yv[0], yv[1], yv[2], yv[3]);
            }
            if (r) {
                TB* dst = r + ((size_t)qc * ny + gj) * nx + gi0;
                if (sizeof(TB) == 4) *reinterpret_cast<float4*>(dst) = make_float4((float)rv[0], (float)rv[1], (float)rv[2], (float)rv[3]);
                else { *reinterpret_cast<double2*>(dst) = make_double2((double)rv[0], (double)rv[1]);
                       *reinterpret_cast<double2*>(dst + 2) = make_double2((double)rv[2], (double)rv[3]); }
            }
        }
#pragma unroll
        for (int c = 0; c < 4; ++c) { xo[c] = fx[1][c + 1]; if (VAR) ko[c] = fk[1][c + 1]; }
        if (p < zc1) stage_finish(p + 1);
    }
    // block sum of sq -> one atomic per block
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) sq += __shfl_xor_sync(0xffffffffu, sq, o);
    if ((tid & 31) == 0) red[tid >> 5] = sq;
    __syncthreads();
    if (tid == 0 && acc) {
        double t = 0.0;
#pragma unroll
        for (int w = 0; w < NT / 32; ++w) t += red[w];
        atomicAdd(acc, t);
    }
}

}  // namespace mk
}  // namespace mgb
