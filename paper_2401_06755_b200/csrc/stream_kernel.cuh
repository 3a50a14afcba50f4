// stream_kernel.cuh -- the fp32 streaming smoother / transfer kernel for uniform grids (sm_100a).
//
// One stencil stage per pass, three variants:
//   MODE_SWEEP   weighted-Jacobi sweep                                   x            -> x'
//   MODE_PRO     prolongation + correction + sweep                      x + P x_c    -> x'
//   MODE_RR      residual, 8-child-mean restriction and the coarse level's first sweep from a
//                zero guess                                              x            -> b_c, x_c
//
// Arithmetic (uniform spacing h; reading C1/C2, Eqs. 8, 12-13 P:109-114, 146-159).  The 6 face
// weights of the trilinear-FE Laplacian vanish on a uniform grid; the 12 edge neighbours carry
// -w = 2 cc and the 8 corner neighbours cc, cc = 1/(24 h^2).  With the integer-weight neighbour sum
//   S(f)_i = 2 E(f)_i + Cn(f)_i            (E = sum over edge neighbours, Cn = over corner neighbours)
// Eq. 13 with sum_j w_ij = 0 reads
//   D_i     = cc (32 k_i + S(k)_i)
//   (A x)_i = D_i x_i - cc (k_i S(x)_i + S(k x)_i)
//   sweep:  x' = (1 - omega) x + omega / (32 k + S(k)) * (b / cc + k S(x) + S(k x))
//   resid:  r  = b + cc (k S(x) + S(k x) - (32 k + S(k)) x)
// Constant coefficient (k = 1): S(k) = 32, S(k x) = S(x).
//
// Data flow.  A block owns a TX x TY column of the grid and streams along z.  The z planes of x and
// k (tile + one halo row / 4 halo columns per side) are staged in shared memory by TMA
// (cp.async.bulk.tensor.3d, out-of-bounds zero fill) into an NS-deep ring, completion on mbarriers;
// the slot of plane p also receives the tile of b of plane p - 1 (no halo), the plane that iteration
// finalises; x' is written straight from registers with 128-bit stores.  Each thread owns a 4 (x) by RY (y) patch of columns: it
// reads its RY + 2 rows of the plane from shared memory as float4, takes the x neighbours of the
// patch ends from the adjacent lanes by shuffle (the two lanes at the ends of a tile row read the
// halo column from shared memory instead), forms k x for those rows in registers, and reduces
// each plane to the in-plane sums
//   Dg = 4 diagonal neighbours,   Pp = 2 (4 cross neighbours) + Dg,
// so that  S[z] = Pp[z-1] + 2 Dg[z] + Pp[z+1]  is accumulated in two registers per point and field
// and every plane is read from shared memory once.  Boundary halos (ghost = s * mirror)
// cost nothing in shared memory: a ghost row is the mirrored row read with the factor s, a ghost
// column is s times the patch's own end value, a ghost plane is the mirrored plane loaded again.
// There is one __syncthreads per plane (ring-slot hand-back to the TMA producer thread).
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <cstdint>

namespace mgb {
namespace sk {

enum { MODE_SWEEP = 0, MODE_PRO = 1, MODE_RR = 2 };

struct SParams {
    int nx, ny, nz;
    int zchunk;                 // output planes per block (even)
    float sx0, sx1, sy0, sy1, sz0, sz1;
    float cc, icc;              // 1/(24 h^2) and its inverse
    float omega;
    float* out;                 // x' (sweep modes)
    const float* xc;            // PRO: coarse correction (nx/2 * ny/2 * nz/2)
    float* bc_out;              // RR: restricted residual
    float* xc_out;              // RR: coarse first sweep  omega b_c / D_c  (or zeros)
    const float* dinv_c;        // RR, variable k: 1 / D_c on the coarse level
    float gc_const;             // RR, constant k: omega / w0_c
    int first_sweep;            // RR: write x_c = omega b_c / D_c (1) or zeros (0)
};

template <int LX_, int LY_, bool VAR_, int MODE_, int MINB_>
struct SCfg {
    static constexpr int LX = LX_, LY = LY_, MODE = MODE_, MINB = MINB_;
    static constexpr bool VAR = VAR_;
    static constexpr int RY = 2;
    static constexpr int TX = 4 * LX, TY = RY * LY, NT = LX * LY;
    static constexpr int PX = TX + 8, PY = TY + 2;
    static constexpr int NS = 3;                                          // ring depth = planes in flight
    static constexpr int PLANE = ((PX * PY + 31) / 32) * 32;              // floats per staged x / k plane (128-byte multiple)
    static constexpr int BPLANE = ((TX * TY + 31) / 32) * 32;             // floats per staged b tile
    static constexpr int SLOT = PLANE * (VAR ? 2 : 1) + BPLANE;           // floats per ring slot: x, (k,) b
    static constexpr uint32_t BOX_BYTES = (uint32_t)(PX * PY * sizeof(float));
    static constexpr uint32_t BBOX_BYTES = (uint32_t)(TX * TY * sizeof(float));
    static constexpr int BAR_FLOATS = 32;
    static constexpr size_t SMEM = (size_t)(BAR_FLOATS + NS * SLOT) * sizeof(float);
    static_assert(LX <= 32 && 32 % LX == 0, "a tile row is a warp or a power-of-two fraction of one");
    static_assert(NT % 32 == 0, "whole warps");
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
        "SK_WAIT:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n"
        "@P1 bra SK_DONE;\n"
        "bra SK_WAIT;\n"
        "SK_DONE:\n"
        "}" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
__device__ __forceinline__ void tma_load_plane(float* dst, const CUtensorMap* tm, uint64_t* bar, int cx, int cy, int cz) {
    asm volatile(
        "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5}], [%2];"
        ::"r"(smem_u32(dst)), "l"(reinterpret_cast<uint64_t>(tm)), "r"(smem_u32(bar)), "r"(cx), "r"(cy), "r"(cz)
        : "memory");
}

// One staged row of a thread's patch: its 4 values and the x neighbours of the patch ends.
struct Row { float l, v0, v1, v2, v3, r; };

// In-plane sums of one field for the thread's 4 x RY patch from its RY + 2 rows:
//   R_q(c) = f(c-1, q) + f(c+1, q),  T_q = R_q + 2 f(c, q)
//   Dg_j = R_{j-1} + R_{j+1},  Pp_j = T_{j-1} + T_{j+1} + 2 R_j   (= 2 cross + diagonal)
// scattered into the z accumulators:  S = A + Pp (plane below is complete), A <- B + 2 Dg, B <- Pp.
template <int RY>
__device__ __forceinline__ void plane_accumulate(const Row (&w)[RY + 2], float (&A)[RY][4], float (&B)[RY][4],
                                                 float (&S)[RY][4]) {
    float R[RY + 2][4], T[RY + 2][4];
#pragma unroll
    for (int q = 0; q < RY + 2; ++q) {
        R[q][0] = w[q].l + w[q].v1; R[q][1] = w[q].v0 + w[q].v2; R[q][2] = w[q].v1 + w[q].v3; R[q][3] = w[q].v2 + w[q].r;
        T[q][0] = fmaf(2.f, w[q].v0, R[q][0]); T[q][1] = fmaf(2.f, w[q].v1, R[q][1]);
        T[q][2] = fmaf(2.f, w[q].v2, R[q][2]); T[q][3] = fmaf(2.f, w[q].v3, R[q][3]);
    }
#pragma unroll
    for (int j = 0; j < RY; ++j)
#pragma unroll
        for (int c = 0; c < 4; ++c) {
            const float Dg = R[j][c] + R[j + 2][c];
            const float Pp = fmaf(2.f, R[j + 1][c], T[j][c] + T[j + 2][c]);
            S[j][c] = A[j][c] + Pp;
            A[j][c] = fmaf(2.f, Dg, B[j][c]);
            B[j][c] = Pp;
        }
}

template <class C>
__global__ void __launch_bounds__(C::NT, C::MINB)
stream_kernel(const __grid_constant__ CUtensorMap tmx, const __grid_constant__ CUtensorMap tmk,
              const __grid_constant__ CUtensorMap tmb, const SParams P) {
    constexpr int RY = C::RY, PX = C::PX, PY = C::PY, PLANE = C::PLANE, NS = C::NS, LX = C::LX, SLOT = C::SLOT;
    constexpr bool VAR = C::VAR;
    constexpr int MODE = C::MODE;
    constexpr int KOFF = PLANE, BOFF = PLANE * (VAR ? 2 : 1);      // k and b inside a ring slot

    extern __shared__ __align__(1024) float smf[];
    uint64_t* bars = reinterpret_cast<uint64_t*>(smf);
    float* ring = smf + C::BAR_FLOATS;

    const int tid = threadIdx.x, lx = tid % LX, ly = tid / LX;
    const int nx = P.nx, ny = P.ny, nz = P.nz;
    const int x0 = blockIdx.x * C::TX, y0 = blockIdx.y * C::TY;
    const int zc0 = blockIdx.z * P.zchunk, zc1 = min(zc0 + P.zchunk, nz);
    const int pbeg = zc0 - 1, niter = zc1 - zc0 + 2;
    const int c0 = 4 * lx, gi0 = x0 + c0, gj0 = y0 + RY * ly;
    const bool active = gi0 < nx && gj0 < ny;

    // ---- z-invariant per-thread set-up: row offsets / factors, patch-end neighbour sources ----
    int roff[RY + 2];
#pragma unroll
    for (int q = 0; q < RY + 2; ++q) {
        const int gq = gj0 - 1 + q;
        const int m = gq < 0 ? -1 - gq : (gq >= ny ? 2 * ny - 1 - gq : gq);
        roff[q] = min(max(m - (y0 - 1), 0), PY - 1) * PX + 4 + c0;
    }
    // only the first and the last staged row of a patch can be ghost rows (factor s of the y faces)
    const float fy_lo = (gj0 - 1 < 0) ? P.sy0 : 1.f, fy_hi = (gj0 + RY >= ny) ? P.sy1 : 1.f;
    // left / right neighbour of the patch: adjacent lane (default), ghost = s * own end value, or the halo column
    const bool lghost = gi0 == 0, rghost = gi0 + 4 >= nx;
    const bool lhalo = !lghost && lx == 0, rhalo = !rghost && lx == LX - 1;
    const int boff = BOFF + (RY * ly) * C::TX + c0;

    auto zsrc = [&](int p) { return p < 0 ? -1 - p : (p >= nz ? 2 * nz - 1 - p : p); };
    auto zfac = [&](int p) { return p < 0 ? P.sz0 : (p >= nz ? P.sz1 : 1.f); };
    auto issue = [&](int it) {   // one thread: TMA of the x, k planes of iteration `it` and of the b tile it finalises
        uint64_t* bar = &bars[it % NS];
        float* dst = ring + (it % NS) * SLOT;
        const bool wb = it >= 2;                                   // plane pbeg + it - 1 >= zc0
        mbar_expect_tx(bar, C::BOX_BYTES * (VAR ? 2u : 1u) + (wb ? C::BBOX_BYTES : 0u));
        const int z = zsrc(pbeg + it);
        tma_load_plane(dst, &tmx, bar, x0 - 4, y0 - 1, z);
        if (VAR) tma_load_plane(dst + KOFF, &tmk, bar, x0 - 4, y0 - 1, z);
        if (wb) tma_load_plane(dst + BOFF, &tmb, bar, x0, y0, pbeg + it - 1);
    };

    if (tid == 0) {
#pragma unroll
        for (int q = 0; q < NS; ++q) mbar_init(&bars[q], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    }
    __syncthreads();
    if (tid == 0)
        for (int q = 0; q < NS && q < niter; ++q) issue(q);

    // ---- per-point state carried along z ---------------------------------------------------------
    float xA[RY][4], xB[RY][4], zA[RY][4], zB[RY][4], kA[RY][4], kB[RY][4];   // S accumulators of x, k x, k
    float xp[RY][4], kp[RY][4];                                               // own values of the previous plane
    float hold0 = 0.f, hold1 = 0.f;                                           // restriction: sums of the even plane
#pragma unroll
    for (int j = 0; j < RY; ++j)
#pragma unroll
        for (int c = 0; c < 4; ++c) {
            xA[j][c] = xB[j][c] = zA[j][c] = zB[j][c] = kA[j][c] = kB[j][c] = 0.f;
            xp[j][c] = 0.f; kp[j][c] = 1.f;
        }
    const float omega = P.omega, om1 = 1.f - P.omega, icc = P.icc, cc = P.cc;
    const int nxc = nx >> 1, nyc = ny >> 1;
    int slot = 0; uint32_t par = 0;

    for (int it = 0; it < niter; ++it) {
        const int p = pbeg + it;
        // ---- PRO: coarse correction of the staged rows, issued before the barrier wait ----
        float2 pc[3]; float pl[3], pr[3];
        if (MODE == MODE_PRO) {
            // rows (-1), (0, 1), (2) of the patch lie in 3 coarse rows; halo columns in the neighbouring coarse cells
            const size_t cplane = (size_t)(zsrc(p) >> 1) * nyc;
#pragma unroll
            for (int q = 0; q < 3; ++q) {
                pc[q] = make_float2(0.f, 0.f); pl[q] = 0.f; pr[q] = 0.f;
                const int gq = gj0 - 1 + (q == 0 ? 0 : (q == 1 ? 1 : 3));
                const int m = gq < 0 ? -1 - gq : (gq >= ny ? 2 * ny - 1 - gq : gq);
                const float* crow = P.xc + (cplane + (m >> 1)) * nxc;
                if (active) {
                    pc[q] = __ldg(reinterpret_cast<const float2*>(crow + (gi0 >> 1)));
                    if (lhalo) pl[q] = __ldg(crow + ((gi0 - 1) >> 1));
                    if (rhalo) pr[q] = __ldg(crow + ((gi0 + 4) >> 1));
                }
            }
        }
        // ---- ring hand-back: everyone has finished iteration it - 1, so its slot can be refilled ----
        __syncthreads();
        if (tid == 0 && it >= 1 && it - 1 + NS < niter) {
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
            issue(it - 1 + NS);
        }
        mbar_wait(&bars[slot], par);

        // ---- stage the RY + 2 rows of x (and k) in registers ----
        const float* xs = ring + slot * SLOT;
        const float fz = zfac(p);
        Row xw[RY + 2], kw[RY + 2];
#pragma unroll
        for (int q = 0; q < RY + 2; ++q) {
            const float* xr = xs + roff[q];
            float4 c = *reinterpret_cast<const float4*>(xr);
            float el = 0.f, er = 0.f;
            if (lhalo) el = xr[-1];
            if (rhalo) er = xr[4];
            if (MODE == MODE_PRO) {
                const int a = q == 0 ? 0 : (q == RY + 1 ? 2 : 1);
                c.x += pc[a].x; c.y += pc[a].x; c.z += pc[a].y; c.w += pc[a].y;
                el += pl[a]; er += pr[a];
            }
            if (q == 0 || q == RY + 1) {
                const float f = (q == 0 ? fy_lo : fy_hi) * fz;
                c.x *= f; c.y *= f; c.z *= f; c.w *= f; el *= f; er *= f;
            } else if (fz != 1.f) {
                c.x *= fz; c.y *= fz; c.z *= fz; c.w *= fz; el *= fz; er *= fz;
            }
            float l = __shfl_up_sync(0xffffffffu, c.w, 1), r = __shfl_down_sync(0xffffffffu, c.x, 1);
            if (lhalo) l = el;
            if (rhalo) r = er;
            if (lghost) l = P.sx0 * c.x;
            if (rghost) r = P.sx1 * c.w;
            xw[q].l = l; xw[q].v0 = c.x; xw[q].v1 = c.y; xw[q].v2 = c.z; xw[q].v3 = c.w; xw[q].r = r;
            if (VAR) {
                const float* kr_ = xr + KOFF;
                const float4 d = *reinterpret_cast<const float4*>(kr_);
                float kl = __shfl_up_sync(0xffffffffu, d.w, 1), kr = __shfl_down_sync(0xffffffffu, d.x, 1);
                if (lhalo) kl = kr_[-1];
                if (rhalo) kr = kr_[4];
                if (lghost) kl = d.x;
                if (rghost) kr = d.w;
                kw[q].l = kl; kw[q].v0 = d.x; kw[q].v1 = d.y; kw[q].v2 = d.z; kw[q].v3 = d.w; kw[q].r = kr;
            }
        }

        // ---- plane sums, z accumulation ----
        float Sx[RY][4], Sz[RY][4], Sk[RY][4];
        if (VAR) {
            Row zw[RY + 2];
#pragma unroll
            for (int q = 0; q < RY + 2; ++q) {
                zw[q].l = kw[q].l * xw[q].l; zw[q].v0 = kw[q].v0 * xw[q].v0; zw[q].v1 = kw[q].v1 * xw[q].v1;
                zw[q].v2 = kw[q].v2 * xw[q].v2; zw[q].v3 = kw[q].v3 * xw[q].v3; zw[q].r = kw[q].r * xw[q].r;
            }
            plane_accumulate<RY>(zw, zA, zB, Sz);
            plane_accumulate<RY>(kw, kA, kB, Sk);
        }
        plane_accumulate<RY>(xw, xA, xB, Sx);

        // ---- finalise plane p - 1 ----
        const int qc = p - 1;
        if (qc >= zc0) {
            float rs0 = 0.f, rs1 = 0.f;
#pragma unroll
            for (int j = 0; j < RY; ++j) {
                const float4 b4 = *reinterpret_cast<const float4*>(xs + boff + j * C::TX);
                const float bv[4] = {b4.x, b4.y, b4.z, b4.w};
                float o[4];
#pragma unroll
                for (int c = 0; c < 4; ++c) {
                    const float xv = xp[j][c];
                    if (VAR) {
                        const float kv = kp[j][c];
                        const float Dp = fmaf(32.f, kv, Sk[j][c]);
                        const float t = fmaf(kv, Sx[j][c], Sz[j][c]);
                        if (MODE == MODE_RR) o[c] = fmaf(cc, fmaf(-Dp, xv, t), bv[c]);
                        else o[c] = fmaf(__fdividef(omega, Dp), fmaf(icc, bv[c], t), om1 * xv);
                    } else {
                        if (MODE == MODE_RR) o[c] = fmaf(cc, fmaf(-64.f, xv, 2.f * Sx[j][c]), bv[c]);
                        else o[c] = fmaf(omega * (1.f / 64.f), fmaf(icc, bv[c], 2.f * Sx[j][c]), om1 * xv);
                    }
                }
                if (MODE == MODE_RR) { rs0 += o[0] + o[1]; rs1 += o[2] + o[3]; }
                else if (active)
                    *reinterpret_cast<float4*>(P.out + ((size_t)qc * ny + (gj0 + j)) * nx + gi0) = make_float4(o[0], o[1], o[2], o[3]);
            }
            if (MODE == MODE_RR) {
                if (qc & 1) {
                    if (active) {
                        const size_t ci = ((size_t)(qc >> 1) * nyc + (gj0 >> 1)) * nxc + (gi0 >> 1);
                        const float2 bcv = make_float2(0.125f * (hold0 + rs0), 0.125f * (hold1 + rs1));
                        *reinterpret_cast<float2*>(P.bc_out + ci) = bcv;
                        float2 xcv = make_float2(0.f, 0.f);
                        if (P.first_sweep) {
                            if (VAR) {
                                const float2 di = __ldg(reinterpret_cast<const float2*>(P.dinv_c + ci));
                                xcv = make_float2(omega * di.x * bcv.x, omega * di.y * bcv.y);
                            } else {
                                xcv = make_float2(P.gc_const * bcv.x, P.gc_const * bcv.y);
                            }
                        }
                        *reinterpret_cast<float2*>(P.xc_out + ci) = xcv;
                    }
                } else {
                    hold0 = rs0; hold1 = rs1;
                }
            }
        }
        // ---- roll the per-plane state ----
#pragma unroll
        for (int j = 0; j < RY; ++j) {
            xp[j][0] = xw[j + 1].v0; xp[j][1] = xw[j + 1].v1; xp[j][2] = xw[j + 1].v2; xp[j][3] = xw[j + 1].v3;
            if (VAR) { kp[j][0] = kw[j + 1].v0; kp[j][1] = kw[j + 1].v1; kp[j][2] = kw[j + 1].v2; kp[j][3] = kw[j + 1].v3; }
        }
        if (++slot == NS) { slot = 0; par ^= 1; }
    }
}

}  // namespace sk
}  // namespace mgb
