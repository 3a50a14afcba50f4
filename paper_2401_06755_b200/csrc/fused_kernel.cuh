// fused_kernel.cuh -- the tuned fp32 smoother / transfer kernel for uniform grids (sm_100a).
//
// One kernel template covers the three fused passes of the V-cycle:
//   <NS sweeps>                      temporally fused weighted-Jacobi sweeps            x -> x'
//   <PRO, NS sweeps>                 prolongation + correction + NS post-sweeps        x + P x_c -> x'
//   <NS sweeps, RR>                  NS sweeps, residual, 8-child-mean restriction and the coarse
//                                    level's first sweep from a zero guess             x -> x', b_c, x_c
//
// Arithmetic (uniform spacing h; reading C1/C2, Eqs. 8, 12-13 P:109-114, 146-159): with the
// off-diagonal neighbour sum  S(f)_i = ce E(f)_i + cc Cn(f)_i  (E = 12 edge neighbours, Cn = 8
// corner neighbours; the 6 face weights of the trilinear-FE Laplacian vanish on a uniform grid),
//   ce = 1/(12 h^2), cc = 1/(24 h^2), cdiag = 4/(3 h^2):
//   D_i    = cdiag k_i + S(k)_i
//   (A x)_i = D_i x_i - k_i S(x)_i - S(k x)_i            [Eq. 13 with sum_j w_ij = 0]
//   sweep:  x' = (1 - omega) x + (omega / D) (b + k S(x) + S(k x))
//   resid:  r  = b + k S(x) + S(k x) - D x
// Constant coefficient: A x = w0 x - S1(x), S1 = 2 S, w0 = 8/(3 h^2).
//
// Data flow: the block owns a TX x TY column of the grid and streams along z.  Each z plane of
// x, k, b (tile + halo) is staged in shared memory by TMA (cp.async.bulk.tensor.3d, out-of-bounds
// zero fill) NPF planes ahead, completion on mbarriers.  Halo cells outside the domain are filled
// once per plane with the boundary rule ghost = s * mirror -- for s = +-1 the mirror
// symmetry is then preserved by every later stage, so ghost cells are simply computed like real
// cells; s = 0 faces re-zero them per stage.  The 27-point sum is factorised into in-plane cross
// and diagonal sums of ONE plane (X, Dg) that are scattered into per-thread register accumulators
// of the plane below, the plane itself and the plane above, so every plane of every stage is read
// from shared memory exactly once.  Each thread owns a 4 (x) by 2 (y) patch of columns.  Stages
// are skewed by one plane in z and exchange one plane of x^s and k x^s through shared memory.
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <cstdint>

namespace mgb {
namespace fk {

struct FParams {
    int nx, ny, nz;
    int zchunk;                 // output planes per block (even)
    float sx0, sx1, sy0, sy1, sz0, sz1;
    float ce, cc, cdiag;        // variable k
    float w0;                   // constant k: centre weight; S1 uses 2 ce, 2 cc
    float omega;
    int any_s0;                 // some face has s = 0 (MG_BC_DIRICHLET_HALO)
    float* out;                 // x' (may be NULL when only the restriction is wanted)
    const float* xc;            // PRO: coarse correction (nx/2 * ny/2 * nz/2)
    float* bc_out;              // RR: restricted residual
    float* xc_out;              // RR: coarse first sweep  omega b_c / D_c  (or zeros)
    const float* dinv_c;        // RR, variable k: 1 / D_c on the coarse level
    float gc_const;             // RR, constant k: omega / w0_c  (0 => x_c = 0)
    int first_sweep;            // RR: write x_c = omega b_c / D_c (1) or zeros (0)
};

template <int NS_, bool RR_, bool PRO_, bool VAR_, int TX_, int TY_>
struct Cfg {
    static constexpr int NS = NS_;
    static constexpr bool RR = RR_, PRO = PRO_, VAR = VAR_;
    static constexpr int TX = TX_, TY = TY_;
    static constexpr int RY = 2;
    static constexpr int NST = NS + (RR ? 1 : 0);            // stencil stages
    static constexpr int HX = 4;
    static constexpr int HY = ((NST + 1) / 2) * 2;
    static constexpr int PX = TX + 2 * HX, PY = TY + 2 * HY;
    static constexpr int LX = PX / 4, LY = PY / RY, NT = LX * LY;
    static constexpr int PLANE = PX * PY;
    static constexpr int NPF = (NST == 1) ? 3 : 2;           // TMA prefetch distance in planes
    static constexpr int DXR = NPF;                          // raw x ring
    static constexpr int DK = NPF + NST + 1;                 // k and b rings (own-point reads lag by up to NST)
    static constexpr int DG = (VAR && NST >= 2) ? NST : 0;   // omega/D (or D) ring for the lagged stages
    static constexpr int NPLANES = DXR + (VAR ? DK : 0) + DK + 2 * NST + (VAR ? NST : 0) + DG;
    static constexpr int BAR_FLOATS = 32;                    // mbarriers live in the first 128 bytes
    static constexpr size_t SMEM = (size_t)NPLANES * PLANE * sizeof(float) + BAR_FLOATS * sizeof(float);
    static_assert(NST >= 1 && NST <= 2, "one or two stencil stages per pass");
    static_assert(LX == 16 || LX == 32, "a tile row must be a half warp or a warp (x neighbours come by shuffle)");
    static_assert(TX % 4 == 0 && TY % 2 == 0 && PY % RY == 0, "tile shape");
    static_assert((PLANE * 4) % 128 == 0, "TMA destination alignment");
};

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t* bar, int count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
    asm volatile(
        "{\n"
        ".reg .pred P1;\n"
        "LAB_WAIT:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n"
        "@P1 bra DONE;\n"
        "bra LAB_WAIT;\n"
        "DONE:\n"
        "}" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
__device__ __forceinline__ void tma_load_plane(float* dst, const CUtensorMap* tm, uint64_t* bar, int cx, int cy, int cz) {
    asm volatile(
        "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5}], [%2];"
        ::"r"(smem_u32(dst)), "l"(reinterpret_cast<uint64_t>(tm)), "r"(smem_u32(bar)), "r"(cx), "r"(cy), "r"(cz)
        : "memory");
}

__device__ __forceinline__ float4 ld4(const float* p) { return *reinterpret_cast<const float4*>(p); }
__device__ __forceinline__ void st4(float* p, float4 v) { *reinterpret_cast<float4*>(p) = v; }
__device__ __forceinline__ float4 rev4(float4 v) { return make_float4(v.w, v.z, v.y, v.x); }
__device__ __forceinline__ float4 mul4(float4 v, float f) { return make_float4(v.x * f, v.y * f, v.z * f, v.w * f); }

// In-plane sums of one staged plane for the thread's 4 x RY patch: for every own point,
//   X = f(i-1,j) + f(i+1,j) + f(i,j-1) + f(i,j+1),  Dg = f(i-1,j-1) + f(i+1,j-1) + f(i-1,j+1) + f(i+1,j+1),
// returned as P = ce X + cc Dg (contribution to the planes below and above) and Q = ce Dg (to the plane itself).
template <int RY, int PX>
__device__ __forceinline__ void plane_sums(const float* __restrict__ F, const int (&roff)[RY + 2], float ce, float cc,
                                           float (&P)[RY][4], float (&Q)[RY][4]) {
    float v[RY + 2][4], R[RY + 2][4];
#pragma unroll
    for (int q = 0; q < RY + 2; ++q) {
        const float4 c = ld4(F + roff[q]);
        // x neighbours of the patch ends come from the adjacent lanes (same row); the two lanes at
        // the row ends receive junk, which only reaches the outermost halo column
        const float l = __shfl_up_sync(0xffffffffu, c.w, 1), r = __shfl_down_sync(0xffffffffu, c.x, 1);
        v[q][0] = c.x; v[q][1] = c.y; v[q][2] = c.z; v[q][3] = c.w;
        R[q][0] = l + c.y; R[q][1] = c.x + c.z; R[q][2] = c.y + c.w; R[q][3] = c.z + r;
    }
#pragma unroll
    for (int j = 0; j < RY; ++j)
#pragma unroll
        for (int c = 0; c < 4; ++c) {
            const float X = R[j + 1][c] + (v[j][c] + v[j + 2][c]);
            const float Dg = R[j][c] + R[j + 2][c];
            P[j][c] = fmaf(cc, Dg, ce * X);
            Q[j][c] = ce * Dg;
        }
}

template <class C>
__global__ void __launch_bounds__(C::NT, 1)
fused_kernel(const __grid_constant__ CUtensorMap tmx, const __grid_constant__ CUtensorMap tmk,
             const __grid_constant__ CUtensorMap tmb, const FParams P) {
    constexpr int NS = C::NS, NST = C::NST, RY = C::RY, PX = C::PX, PY = C::PY, PLANE = C::PLANE;
    constexpr int NPF = C::NPF, DXR = C::DXR, DK = C::DK, DG = C::DG, HX = C::HX, HY = C::HY;
    constexpr bool RR = C::RR, PRO = C::PRO, VAR = C::VAR;

    extern __shared__ __align__(1024) float smf[];
    uint64_t* bars = reinterpret_cast<uint64_t*>(smf);
    float* XR = smf + C::BAR_FLOATS;                  // [DXR] raw x planes (TMA)
    float* KR = XR + DXR * PLANE;                     // [DK]  k planes (TMA + ghost fill)       (VAR)
    float* BR = KR + (VAR ? DK : 0) * PLANE;          // [DK]  b planes (TMA + ghost fill)
    float* XS = BR + DK * PLANE;                      // [NST][2] stage inputs x^s
    float* ZS = XS + 2 * NST * PLANE;                 // [NST] k x^s                             (VAR)
    float* GR = ZS + (VAR ? NST : 0) * PLANE;         // [DG]  omega/D (sweep) or D (residual) of lagged planes

    const int tid = threadIdx.x, lx = tid % C::LX, ly = tid / C::LX;
    const int x0 = blockIdx.x * C::TX, y0 = blockIdx.y * C::TY;
    const int zc0 = blockIdx.z * P.zchunk, zc1 = min(zc0 + P.zchunk, P.nz);
    const int pbeg = zc0 - NST, pend = zc1 + NST;
    const int c0 = 4 * lx, r0 = RY * ly;
    const int gi0 = x0 - HX + c0, gj0 = y0 - HY + r0;
    const int nx = P.nx, ny = P.ny, nz = P.nz;

    // ---- z-invariant per-thread set-up -------------------------------------------------------
    int roff[RY + 2];
#pragma unroll
    for (int q = 0; q < RY + 2; ++q) roff[q] = min(max(r0 - 1 + q, 0), PY - 1) * PX + c0;
    int own[RY];
#pragma unroll
    for (int j = 0; j < RY; ++j) own[j] = (r0 + j) * PX + c0;

    // ghost fill: source patch (mirrored cell) and factor for every own row
    int src[RY]; float fxy[RY]; bool ghost[RY], indom[RY]; bool rev = false;
    int gis = gi0; float fx = 1.f; bool xok = true;
    if (gi0 < 0) { gis = -4 - gi0; fx = P.sx0; rev = true; xok = (gi0 >= -4); }             // cells -4..-1 <- 3..0
    else if (gi0 >= nx) { gis = 2 * nx - 4 - gi0; fx = P.sx1; rev = true; xok = (gi0 < nx + 4) && gis >= 0; }
    int gjs[RY];
#pragma unroll
    for (int j = 0; j < RY; ++j) {
        const int gj = gj0 + j;
        int g2 = gj; float fy = 1.f; bool yok = true;
        if (gj < 0) { g2 = -1 - gj; fy = P.sy0; yok = (gj >= -NST) && g2 < ny; }
        else if (gj >= ny) { g2 = 2 * ny - 1 - gj; fy = P.sy1; yok = (gj < ny + NST) && g2 >= 0; }
        gjs[j] = g2;
        const int sr = r0 + j + (g2 - gj), sc = c0 + (gis - gi0);
        const bool inside = sr >= 0 && sr < PY && sc >= 0 && sc + 3 < PX;
        indom[j] = (gi0 >= 0 && gi0 < nx && gj >= 0 && gj < ny);
        ghost[j] = !indom[j] && xok && yok && inside;
        src[j] = inside ? sr * PX + sc : own[j];
        fxy[j] = fx * fy;
    }
    // cells that must be re-zeroed after every sweep stage: ghosts of a face with s = 0
    bool zero_row[RY];
#pragma unroll
    for (int j = 0; j < RY; ++j) {
        const int gj = gj0 + j;
        zero_row[j] = P.any_s0 && ((gi0 < 0 && P.sx0 == 0.f) || (gi0 >= nx && P.sx1 == 0.f) || (gj < 0 && P.sy0 == 0.f) ||
                                   (gj >= ny && P.sy1 == 0.f));
    }
    // which own cells are outputs of this block
    const bool xvalid = gi0 >= x0 && gi0 < x0 + C::TX && gi0 < nx;
    bool valid[RY];
#pragma unroll
    for (int j = 0; j < RY; ++j) {
        const int gj = gj0 + j;
        valid[j] = xvalid && gj >= y0 && gj < y0 + C::TY && gj < ny;
    }

    const float ce = VAR ? P.ce : 2.f * P.ce, cc = VAR ? P.cc : 2.f * P.cc;
    const float omega = P.omega, om1 = 1.f - P.omega;
    const float gconst = VAR ? 0.f : P.omega / P.w0;

    // ---- accumulators --------------------------------------------------------------------------
    float dA[RY][4], dB[RY][4];                       // S(k)
    float sxA[NST][RY][4], sxB[NST][RY][4];           // S(x^s)
    float szA[NST][RY][4], szB[NST][RY][4];           // S(k x^s)
    float hold[2] = {0.f, 0.f};                       // restriction: partial sums of the even plane
#pragma unroll
    for (int j = 0; j < RY; ++j)
#pragma unroll
        for (int c = 0; c < 4; ++c) {
            dA[j][c] = dB[j][c] = 0.f;
#pragma unroll
            for (int s = 0; s < NST; ++s) sxA[s][j][c] = sxB[s][j][c] = szA[s][j][c] = szB[s][j][c] = 0.f;
        }

    auto zsrc = [&](int p) { return p < 0 ? -1 - p : (p >= nz ? 2 * nz - 1 - p : p); };
    auto zfac = [&](int p) { return p < 0 ? P.sz0 : (p >= nz ? P.sz1 : 1.f); };
    constexpr uint32_t TX_BYTES = (uint32_t)(PLANE * sizeof(float)) * (VAR ? 3u : 2u);
    auto issue = [&](int p) {   // one thread: TMA of planes x, k, b for plane index p
        const int itp = p - pbeg;
        uint64_t* bar = &bars[itp % NPF];
        mbar_expect_tx(bar, TX_BYTES);
        const int z = zsrc(p);
        tma_load_plane(XR + (itp % DXR) * PLANE, &tmx, bar, x0 - HX, y0 - HY, z);
        if (VAR) tma_load_plane(KR + (itp % DK) * PLANE, &tmk, bar, x0 - HX, y0 - HY, z);
        tma_load_plane(BR + (itp % DK) * PLANE, &tmb, bar, x0 - HX, y0 - HY, z);
    };

    if (tid == 0) {
#pragma unroll
        for (int q = 0; q < NPF; ++q) mbar_init(&bars[q], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    }
    __syncthreads();
    if (tid == 0)
        for (int q = 0; q < NPF && pbeg + q < pend; ++q) issue(pbeg + q);

    const int nxc = nx >> 1, nyc = ny >> 1;

    // ring slots, advanced incrementally (all warp-uniform)
    int xcur = 0, kcur = 0, bpar = 0;                 // raw-x slot / barrier index, k-b slot, barrier parity
    int kcs[NST], gcs[NST];                           // k-b slot and g slot of the plane each stage finalises
#pragma unroll
    for (int s = 0; s < NST; ++s) { kcs[s] = (8 * DK - s - 1) % DK; gcs[s] = DG > 0 ? (8 * DG - s - 1) % DG : 0; }

    for (int p = pbeg; p < pend; ++p) {
        const int it = p - pbeg;
        // ---- prolongation operands (global loads issued before the TMA wait) ------------------
        float2 pc[RY];
        if (PRO) {
            const int ck = zsrc(p) >> 1;
#pragma unroll
            for (int j = 0; j < RY; ++j) {
                pc[j] = make_float2(0.f, 0.f);
                if ((indom[j] || ghost[j]) && gis >= 0 && gis < nx)
                    pc[j] = *reinterpret_cast<const float2*>(P.xc + ((size_t)ck * nyc + (gjs[j] >> 1)) * nxc + (gis >> 1));
            }
        }
        mbar_wait(&bars[xcur], bpar);

        // ---- prep: ghost fill of k and b, stage-0 input x^0 (+ prolongation, z factor) and k x^0 ----
        {
            const float fzp = zfac(p);
            const float* xr = XR + xcur * PLANE;
            float* kr = KR + kcur * PLANE;
            float* br = BR + kcur * PLANE;
            float* x0w = XS + (it & 1) * PLANE;
            float* z0w = ZS;
#pragma unroll
            for (int j = 0; j < RY; ++j) {
                float4 xv, kv = make_float4(1.f, 1.f, 1.f, 1.f);
                if (!ghost[j]) {
                    xv = ld4(xr + own[j]);
                    if (VAR) kv = ld4(kr + own[j]);
                    if (PRO) { xv.x += pc[j].x; xv.y += pc[j].x; xv.z += pc[j].y; xv.w += pc[j].y; }
                } else {
                    xv = ld4(xr + src[j]);
                    if (PRO) { xv.x += pc[j].x; xv.y += pc[j].x; xv.z += pc[j].y; xv.w += pc[j].y; }
                    float4 bv = ld4(br + src[j]);
                    if (rev) { xv = rev4(xv); bv = rev4(bv); }
                    xv = mul4(xv, fxy[j]);
                    st4(br + own[j], mul4(bv, fxy[j]));
                    if (VAR) {
                        kv = ld4(kr + src[j]);
                        if (rev) kv = rev4(kv);
                        st4(kr + own[j], kv);
                    }
                }
                if (fzp != 1.f) xv = mul4(xv, fzp);
                st4(x0w + own[j], xv);
                if (VAR) st4(z0w + own[j], make_float4(kv.x * xv.x, kv.y * xv.y, kv.z * xv.z, kv.w * xv.w));
            }
        }
        __syncthreads();
        if (tid == 0 && p + NPF < pend) {
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
            issue(p + NPF);
        }

        // ---- stages ---------------------------------------------------------------------------
#pragma unroll
        for (int s = 0; s < NST; ++s) {
            const int qc = p - s - 1;                          // plane finalised by this stage
            const float* Xin = XS + (2 * s + ((it - s) & 1)) * PLANE;
            const float* Xc = XS + (2 * s + ((it - s - 1) & 1)) * PLANE;
            const float* Kc = KR + kcs[s] * PLANE;
            const float* Bc = BR + kcs[s] * PLANE;
            const float fzc = zfac(qc);
            const bool zero_plane = P.any_s0 && ((qc < 0 && P.sz0 == 0.f) || (qc >= nz && P.sz1 == 0.f));

            float Px[RY][4], Qx[RY][4];
            plane_sums<RY, PX>(Xin, roff, ce, cc, Px, Qx);
            float Sx[RY][4], Sz[RY][4], Dv[RY][4];
#pragma unroll
            for (int j = 0; j < RY; ++j)
#pragma unroll
                for (int c = 0; c < 4; ++c) {
                    Sx[j][c] = sxA[s][j][c] + Px[j][c];
                    sxA[s][j][c] = sxB[s][j][c] + Qx[j][c];
                    sxB[s][j][c] = Px[j][c];
                }
            if (VAR) {
                float Pz[RY][4], Qz[RY][4];
                plane_sums<RY, PX>(ZS + s * PLANE, roff, ce, cc, Pz, Qz);
#pragma unroll
                for (int j = 0; j < RY; ++j)
#pragma unroll
                    for (int c = 0; c < 4; ++c) {
                        Sz[j][c] = szA[s][j][c] + Pz[j][c];
                        szA[s][j][c] = szB[s][j][c] + Qz[j][c];
                        szB[s][j][c] = Pz[j][c];
                    }
                if (s == 0) {   // diagonal of the plane finalised by stage 0: D = cdiag k + S(k)
                    float Pk[RY][4], Qk[RY][4];
                    plane_sums<RY, PX>(KR + kcur * PLANE, roff, ce, cc, Pk, Qk);
#pragma unroll
                    for (int j = 0; j < RY; ++j)
#pragma unroll
                        for (int c = 0; c < 4; ++c) {
                            Dv[j][c] = dA[j][c] + Pk[j][c];
                            dA[j][c] = dB[j][c] + Qk[j][c];
                            dB[j][c] = Pk[j][c];
                        }
                }
            }
            const bool last_sweep = (s == NS - 1);
            const bool is_rr = RR && (s == NS);
            const bool plane_out = (qc >= zc0 && qc < zc1);
            float rs0 = 0.f, rs1 = 0.f;
#pragma unroll
            for (int j = 0; j < RY; ++j) {
                const float4 xc4 = ld4(Xc + own[j]);
                const float4 b4 = ld4(Bc + own[j]);
                const float xcv[4] = {xc4.x, xc4.y, xc4.z, xc4.w}, bv[4] = {b4.x, b4.y, b4.z, b4.w};
                float kv[4] = {1.f, 1.f, 1.f, 1.f}, gv[4];
                if (VAR) {
                    const float4 k4 = ld4(Kc + own[j]);
                    kv[0] = k4.x; kv[1] = k4.y; kv[2] = k4.z; kv[3] = k4.w;
                    if (s == 0) {
#pragma unroll
                        for (int c = 0; c < 4; ++c) {
                            const float D = fmaf(P.cdiag, kv[c], Dv[j][c]);
                            gv[c] = is_rr ? D : __fdividef(omega, D);
                            if (DG > 0) Dv[j][c] = (RR && NS == 1) ? D : gv[c];      // what the lagged stage needs
                        }
                        if (DG > 0) st4(GR + gcs[0] * PLANE + own[j], make_float4(Dv[j][0], Dv[j][1], Dv[j][2], Dv[j][3]));
                    } else {
                        const float4 g4 = ld4(GR + gcs[s] * PLANE + own[j]);
                        gv[0] = g4.x; gv[1] = g4.y; gv[2] = g4.z; gv[3] = g4.w;
                    }
                }
                float outv[4];
#pragma unroll
                for (int c = 0; c < 4; ++c) {
                    const float t = VAR ? fmaf(fzc, bv[c], fmaf(kv[c], Sx[j][c], Sz[j][c])) : fmaf(fzc, bv[c], Sx[j][c]);
                    if (is_rr) {
                        outv[c] = VAR ? fmaf(-gv[c], xcv[c], t) : fmaf(-P.w0, xcv[c], t);      // residual
                    } else {
                        outv[c] = VAR ? fmaf(gv[c], t, om1 * xcv[c]) : fmaf(gconst, t, om1 * xcv[c]);
                        if (zero_row[j] || zero_plane) outv[c] = 0.f;
                    }
                }
                if (is_rr) {
                    rs0 += outv[0] + outv[1];
                    rs1 += outv[2] + outv[3];
                } else {
                    if (s + 1 < NST) {   // hand the plane to the next stage
                        st4(XS + (2 * (s + 1) + ((it - s - 1) & 1)) * PLANE + own[j], make_float4(outv[0], outv[1], outv[2], outv[3]));
                        if (VAR) st4(ZS + (s + 1) * PLANE + own[j],
                                     make_float4(kv[0] * outv[0], kv[1] * outv[1], kv[2] * outv[2], kv[3] * outv[3]));
                    }
                    if (last_sweep && P.out && plane_out && valid[j])
                        st4(P.out + ((size_t)qc * ny + (gj0 + j)) * nx + gi0, make_float4(outv[0], outv[1], outv[2], outv[3]));
                }
            }
            if (is_rr) {
                if (qc & 1) {
                    if (plane_out && valid[0]) {
                        const size_t ci = ((size_t)(qc >> 1) * nyc + (gj0 >> 1)) * nxc + (gi0 >> 1);
                        const float2 bcv = make_float2(0.125f * (hold[0] + rs0), 0.125f * (hold[1] + rs1));
                        *reinterpret_cast<float2*>(P.bc_out + ci) = bcv;
                        float2 xcv2 = make_float2(0.f, 0.f);
                        if (P.first_sweep) {
                            if (VAR) {
                                const float2 di = *reinterpret_cast<const float2*>(P.dinv_c + ci);
                                xcv2 = make_float2(omega * di.x * bcv.x, omega * di.y * bcv.y);
                            } else {
                                xcv2 = make_float2(P.gc_const * bcv.x, P.gc_const * bcv.y);
                            }
                        }
                        *reinterpret_cast<float2*>(P.xc_out + ci) = xcv2;
                    }
                } else {
                    hold[0] = rs0; hold[1] = rs1;
                }
            }
            if (s + 1 < NST || NST == 1) __syncthreads();
        }
        if (++xcur == NPF) { xcur = 0; bpar ^= 1; }
        if (++kcur == DK) kcur = 0;
#pragma unroll
        for (int s = 0; s < NST; ++s) {
            if (++kcs[s] == DK) kcs[s] = 0;
            if (DG > 0 && ++gcs[s] == DG) gcs[s] = 0;
        }
    }
}

}  // namespace fk
}  // namespace mgb
