// lean_kernel.cuh -- the fp32 streaming smoother / transfer kernel for uniform grids (sm_100a).
//
// One stencil stage per pass, three variants:
//   MODE_SWEEP   weighted-Jacobi sweep                                   x            -> x'
//   MODE_PRO     prolongation + correction + sweep                      x + P x_c    -> x'   (x_c tile staged by TMA too)
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
// k (tile + one halo row / 4 halo columns per side, out-of-bounds cells zero-filled) and the tile of
// b are staged in shared memory by TMA (cp.async.bulk.tensor.3d) into an NS-deep ring, completion on
// mbarriers; x' goes from registers to HBM with 128-bit stores.  Each thread owns a 4 (x) by 2 (y)
// patch of columns.  Per plane it reads its 4 rows as one 128-bit and two 32-bit shared loads per
// row and field (rows 0 and 2 first, then 1 and 3, to keep few values live) and reduces the plane to
// the in-plane sums
//   Dg = 4 diagonal neighbours,   Pp = 2 (4 cross neighbours) + Dg,
// so that  S[z] = Pp[z-1] + 2 Dg[z] + Pp[z+1]  is accumulated in two registers per point and field
// and every plane is read from shared memory once.
//
// The kernel is bound by instruction issue unless written tightly (profiles/r01_ncu_stream_v1.md:
// 83 instructions per point), so the arithmetic runs on the packed fp32 pipe (FADD2 / FMUL2 / FFMA2,
// two columns per instruction: a 128-bit shared load delivers the aligned pairs directly), halo
// factors are folded into FMAs that are needed anyway, and the plane loop is unrolled by two so that
// the rolling accumulators and the "own values of the previous plane" are renamed, not moved.
// Boundary halos (ghost = s * mirror): a ghost row is the mirrored row, its factor s folded
// into the row combination; a ghost column is the zero-filled halo cell plus s times the patch's own
// end value (one FMA); a ghost plane is the mirrored plane loaded again, its factor folded into the z
// accumulation.
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <cstdint>
#include <type_traits>

namespace mgb {
namespace lk {

enum { MODE_SWEEP = 0, MODE_PRO = 1, MODE_RR = 2, MODE_SEED = 3 };

struct LParams {
    int nx, ny, nz;
    int zchunk;                 // output planes per block (even)
    int dir;                    // +1: blocks march towards larger z, -1: towards smaller z (one-stage launches: +1; alternating the
                                // direction between consecutive passes was measured: no L2 reuse to be had, 51.3 vs 51.3 us)
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
    int zero_x;                 // SWEEP: the iterate is zero whatever `src` holds: its planes are not read (12 B/point, not 16)
    // MODE_SEED: the first TWO sweeps of a cycle from a zero guess in one pass over y = b / D (written by the defect kernel):
    // x_2 = omega (2 - omega) y + (omega^2 / D) cc (k S(y) + S(k y)) -- the sweep formula x' = om_x x + (om_g / D)(b + cc (..))
    // with om_g = omega^2, om_x = omega (2 - omega) and no b term (the b tiles are not fetched, their ring slots are cleared;
    // 12 B/point).  A mode of its own so that the code of the other modes is untouched.
    float om_g, om_x;
};

template <int LX_, int LY_, bool VAR_, int MODE_, int MINB_>
struct LCfg {
    static constexpr int LX = LX_, LY = LY_, MODE = MODE_, MINB = MINB_;
    static constexpr bool VAR = VAR_;
    static constexpr int RY = 2;
    static constexpr int TX = 4 * LX, TY = RY * LY, NT = LX * LY;
    static constexpr int PX = TX + 8, PY = TY + 2;
    static constexpr int NS = 4;                                          // ring depth = planes in flight + 1
    static constexpr int PLANE = ((PX * PY + 31) / 32) * 32;              // floats per staged x / k plane (128-byte multiple)
    static constexpr int BPLANE = ((TX * TY + 31) / 32) * 32;             // floats per staged b tile
    static constexpr int CPX = TX / 2 + 8, CPY = TY / 2 + 2;              // PRO: staged tile of the coarse correction
    static constexpr int CPLANE_PRO = ((CPX * CPY + 31) / 32) * 32;
    static constexpr int CPLANE = MODE == 1 ? CPLANE_PRO : 0;
    static constexpr int SLOT = PLANE * (VAR ? 2 : 1) + BPLANE + CPLANE;  // floats per ring slot: x, (k,) b, (x_c)
    static constexpr uint32_t CBOX_BYTES = (uint32_t)(CPX * CPY * sizeof(float));
    static constexpr uint32_t BOX_BYTES = (uint32_t)(PX * PY * sizeof(float));
    static constexpr uint32_t BBOX_BYTES = (uint32_t)(TX * TY * sizeof(float));
    static constexpr int BAR_FLOATS = 32;
    static constexpr size_t SMEM = (size_t)(BAR_FLOATS + NS * SLOT) * sizeof(float);
    static_assert(NT % 32 == 0, "whole warps");
};

typedef unsigned long long u64;   // two packed floats {lo, hi} = columns {c, c + 1}

__device__ __forceinline__ u64 pk(float lo, float hi) { u64 r; asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi)); return r; }
__device__ __forceinline__ float lo(u64 v) { float a, b; asm("mov.b64 {%0, %1}, %2;" : "=f"(a), "=f"(b) : "l"(v)); return a; }
__device__ __forceinline__ float hi(u64 v) { float a, b; asm("mov.b64 {%0, %1}, %2;" : "=f"(a), "=f"(b) : "l"(v)); return b; }
__device__ __forceinline__ u64 add2(u64 a, u64 b) { u64 r; asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }
__device__ __forceinline__ u64 mul2(u64 a, u64 b) { u64 r; asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }
__device__ __forceinline__ u64 fma2(u64 a, u64 b, u64 c) { u64 r; asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c)); return r; }
__device__ __forceinline__ u64 bc2(float s) { return pk(s, s); }
__device__ __forceinline__ float rcpa(float a) { float r; asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(a)); return r; }
// shared-memory loads by 32-bit shared-space address (no generic-address arithmetic in the plane loop)
__device__ __forceinline__ float lds32(uint32_t a) { float r; asm volatile("ld.shared.f32 %0, [%1];" : "=f"(r) : "r"(a)); return r; }
__device__ __forceinline__ u64 lds64(uint32_t a) { u64 r; asm volatile("ld.shared.b64 %0, [%1];" : "=l"(r) : "r"(a)); return r; }
__device__ __forceinline__ void lds128(uint32_t a, u64& p, u64& q) { asm volatile("ld.shared.v2.b64 {%0, %1}, [%2];" : "=l"(p), "=l"(q) : "r"(a)); }

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
        "LK_WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n"
        "@P1 bra LK_DONE_%=;\n"
        "bra LK_WAIT_%=;\n"
        "LK_DONE_%=:\n"
        "}" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
__device__ __forceinline__ void tma_load_plane(float* dst, const CUtensorMap* tm, uint64_t* bar, int cx, int cy, int cz) {
    asm volatile(
        "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5}], [%2];"
        ::"r"(smem_u32(dst)), "l"(reinterpret_cast<uint64_t>(tm)), "r"(smem_u32(bar)), "r"(cx), "r"(cy), "r"(cz)
        : "memory");
}

// One staged row of a thread's patch: columns (c0, c0+1) = p, (c0+2, c0+3) = q and the x neighbours of the patch ends.
struct Row { u64 p, q; float l, r; };
// Row-wise x sums of one row:  R(c) = f(c-1) + f(c+1),  T(c) = R(c) + 2 f(c)
struct RT { u64 rp, rq, tp, tq; };

__device__ __forceinline__ RT row_sums(const Row& w, u64 two) {
    RT o;
    o.rp = pk(w.l + hi(w.p), lo(w.p) + lo(w.q));
    o.rq = pk(hi(w.p) + hi(w.q), lo(w.q) + w.r);
    o.tp = fma2(w.p, two, o.rp);
    o.tq = fma2(w.q, two, o.rq);
    return o;
}

// row at shared address `a` (its column c0): halo cell (zero outside the domain) + g * own end value
__device__ __forceinline__ Row load_row(uint32_t a, float gl, float gr) {
    Row w;
    lds128(a, w.p, w.q);
    w.l = lds32(a - 4); w.r = lds32(a + 16);
    w.l = fmaf(gl, lo(w.p), w.l); w.r = fmaf(gr, hi(w.q), w.r);
    return w;
}

// z accumulators of one field for the thread's 2 rows x 2 column pairs
struct Acc { u64 v[2][2]; };

// In-plane sums of one output row j from its three staged rows (a = row j, m = row j + 1, c = row j + 2; fa / fc
// are halo factors of a / c, 1 except for a ghost row):
//   Dg = fa R_a + fc R_c,  Pp = fa T_a + fc T_c + 2 R_m          (FAC: which of a, c can be a ghost row)
// scattered into the z accumulators with the plane factor fz (1 except for a ghost plane):
//   S = A + fz Pp (the plane below is complete),  A <- Bin + 2 fz Dg,  Bout <- Pp (the caller scales it by fz).
template <int FAC>   // 0: no factor, 1: factor on row a, 2: factor on row c
__device__ __forceinline__ void out_row(const RT& a, const RT& m, const RT& c, u64 f, u64 two, u64 fz2, u64 twofz,
                                        u64 (&A)[2], const u64 (&Bin)[2], u64 (&Bout)[2], u64 (&S)[2]) {
    u64 dgp, dgq, ppp, ppq;
    if (FAC == 1) { dgp = fma2(a.rp, f, c.rp); dgq = fma2(a.rq, f, c.rq); ppp = fma2(a.tp, f, c.tp); ppq = fma2(a.tq, f, c.tq); }
    else if (FAC == 2) { dgp = fma2(c.rp, f, a.rp); dgq = fma2(c.rq, f, a.rq); ppp = fma2(c.tp, f, a.tp); ppq = fma2(c.tq, f, a.tq); }
    else { dgp = add2(a.rp, c.rp); dgq = add2(a.rq, c.rq); ppp = add2(a.tp, c.tp); ppq = add2(a.tq, c.tq); }
    ppp = fma2(m.rp, two, ppp); ppq = fma2(m.rq, two, ppq);
    if (FAC == 0) {           // the coefficient: ghost = plain copy
        S[0] = add2(A[0], ppp); S[1] = add2(A[1], ppq);
        A[0] = fma2(dgp, two, Bin[0]); A[1] = fma2(dgq, two, Bin[1]);
    } else {
        S[0] = fma2(ppp, fz2, A[0]); S[1] = fma2(ppq, fz2, A[1]);
        A[0] = fma2(dgp, twofz, Bin[0]); A[1] = fma2(dgq, twofz, Bin[1]);
    }
    Bout[0] = ppp; Bout[1] = ppq;
}

// ---- wave scheduling (wave_kernel.cuh): several dependent stages of one level in ONE launch -------------------------
// A block of stage s + 1 reads the planes that the blocks of stage s (its own tile and the 8 tiles around it) have already
// written; the intermediate iterate travels through L2, not HBM.  Each block publishes in `my_prog` how many planes of
// its z chunk are complete and visible; a consumer polls the flags of its producers before it asks TMA for a plane.
// Chunks march in alternating directions (even chunks upwards, odd ones downwards) so that the two chunks that meet at a
// boundary both start or both end there: the halo plane a consumer needs from the neighbouring chunk is produced at the
// same point of the march as its own, and an output plane is only overwritten (the iterate ping-pongs between two
// buffers) after every block that reads its old contents has moved past it.  Producers always have lower block indices
// than their consumers and blocks are dispatched in index order, so a waiting block never keeps its producer off the SMs.
struct WaveCtx {
    int dir;               // +1: the chunk marches towards larger z, -1: towards smaller z
    int tx, ty, chunk;     // this block's tile and z chunk
    int gx, gy, nch;       // tiles and chunks of the level
    int zchunk;            // planes per chunk (the last chunk may be shorter)
    int* my_prog;          // this block's progress flag (nullptr: nobody waits for this stage)
    const int* dep_prog;   // progress flags [nch][gy][gx] of the stage that produces this stage's iterate (nullptr: none)
    int* err;              // set to 1 if a wait timed out (the result is then garbage, but the kernel ends)
};

__device__ __forceinline__ int ld_acquire_gpu(const int* p) {
    int v; asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory"); return v;
}
__device__ __forceinline__ void st_release_gpu(int* p, int v) {
    asm volatile("st.release.gpu.global.s32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}

template <class C, int MODE, bool WAVE>
__device__ __forceinline__ void lean_body(const CUtensorMap& tmx, const CUtensorMap& tmk, const CUtensorMap& tmb,
                                          const CUtensorMap& tmc, const LParams& P, const int bx, const int by, const int bz,
                                          const WaveCtx& wc) {
    constexpr int RY = C::RY, PX = C::PX, PY = C::PY, PLANE = C::PLANE, NS = C::NS, LX = C::LX;
    constexpr bool VAR = C::VAR;
    constexpr int CPLANE = MODE == MODE_PRO ? C::CPLANE_PRO : 0;
    constexpr int SLOT = PLANE * (VAR ? 2 : 1) + C::BPLANE + CPLANE;
    constexpr int KOFF = PLANE, BOFF = PLANE * (VAR ? 2 : 1);      // k and b inside a ring slot
    constexpr int COFF = BOFF + C::BPLANE;                         // PRO: coarse tile
    static_assert(RY == 2, "2 output rows per thread");

    extern __shared__ __align__(1024) float smf[];
    uint64_t* bars = reinterpret_cast<uint64_t*>(smf);
    float* ring = smf + C::BAR_FLOATS;

    const int tid = threadIdx.x, lx = tid % LX, ly = tid / LX;
    const int nx = P.nx, ny = P.ny, nz = P.nz;
    const int x0 = bx * C::TX, y0 = by * C::TY;
    const int zc0 = bz * P.zchunk, zc1 = min(zc0 + P.zchunk, nz);
    const int niter = zc1 - zc0 + 2;                               // even: zchunk and nz are even
    // iteration `it` stages plane pfirst + dir * it and finalises the plane staged one iteration earlier
    const int dir = WAVE ? wc.dir : P.dir;
    const int pfirst = dir > 0 ? zc0 - 1 : zc1;
    const int c0 = 4 * lx, gi0 = x0 + c0, gj0 = y0 + RY * ly;
    const bool active = gi0 < nx && gj0 < ny;

    // ---- z-invariant per-thread set-up ----------------------------------------------------------
    const uint32_t ring_a = smem_u32(ring);
    uint32_t raddr[4];                                             // shared address of the 4 staged rows in slot 0
#pragma unroll
    for (int q = 0; q < 4; ++q) {
        const int gq = gj0 - 1 + q;
        const int m = gq < 0 ? -1 - gq : (gq >= ny ? 2 * ny - 1 - gq : gq);     // ghost row -> mirrored row
        raddr[q] = ring_a + 4u * (uint32_t)(min(max(m - (y0 - 1), 0), PY - 1) * PX + 4 + c0);
    }
    const uint32_t baddr = ring_a + 4u * (uint32_t)(BOFF + (RY * ly) * C::TX + c0);
    // PRO: the staged coarse tile starts at coarse cell (x0/2 - 4, y0/2 - 1): the first coordinate of a TMA box has to be
    // 16-byte aligned like the x planes' x0 - 4 (a box starting at x0/2 - 1 raised an illegal-instruction fault on B200); rows (-1), (0, 1), (2) of the patch lie in 3
    // coarse rows, the patch and its x neighbours in the 4 coarse cells gi0/2 - 1 .. gi0/2 + 2 (zero outside the domain)
    uint32_t caddr[3] = {0u, 0u, 0u};
    if (MODE == MODE_PRO) {
#pragma unroll
        for (int e = 0; e < 3; ++e) {
            const int gq = gj0 - 1 + (e == 0 ? 0 : (e == 1 ? 1 : 3));
            const int m = gq < 0 ? -1 - gq : (gq >= ny ? 2 * ny - 1 - gq : gq);
            caddr[e] = ring_a + 4u * (uint32_t)(COFF + min(max((m >> 1) - ((y0 >> 1) - 1), 0), C::CPY - 1) * C::CPX + 3 + (c0 >> 1));
        }
    }
    // only the first and the last staged row of a patch can be ghost rows (factor s of the y faces)
    const u64 f0 = bc2((gj0 - 1 < 0) ? P.sy0 : 1.f), f3 = bc2((gj0 + RY >= ny) ? P.sy1 : 1.f);
    // x neighbours of the patch ends: halo cell (zero-filled outside the domain) + s * own end value at a domain face
    const bool lghost = gi0 == 0, rghost = gi0 + 4 >= nx;
    const float glx = lghost ? P.sx0 : 0.f, grx = rghost ? P.sx1 : 0.f;
    const float glk = lghost ? 1.f : 0.f, grk = rghost ? 1.f : 0.f;

    auto zsrc = [&](int p) { return p < 0 ? -1 - p : (p >= nz ? 2 * nz - 1 - p : p); };
    auto issue = [&](int it) {   // one thread: TMA of the x, k planes of iteration `it` and of the b tile it finalises
        uint64_t* bar = &bars[it % NS];
        float* dst = ring + (it % NS) * SLOT;
        const bool wb = it >= 2 && MODE != MODE_SEED;              // the plane finalised in iteration `it` lies in the chunk
        const bool zx = MODE == MODE_SWEEP && P.zero_x;            // x planes stay the zeros written below
        mbar_expect_tx(bar, C::BOX_BYTES * ((VAR ? 1u : 0u) + (zx ? 0u : 1u)) + (wb ? C::BBOX_BYTES : 0u) + (MODE == MODE_PRO ? C::CBOX_BYTES : 0u));
        const int z = zsrc(pfirst + dir * it);
        if (!zx) tma_load_plane(dst, &tmx, bar, x0 - 4, y0 - 1, z);
        if (VAR) tma_load_plane(dst + KOFF, &tmk, bar, x0 - 4, y0 - 1, z);
        if (wb) tma_load_plane(dst + BOFF, &tmb, bar, x0, y0, pfirst + dir * (it - 1));
        if (MODE == MODE_PRO) tma_load_plane(dst + COFF, &tmc, bar, (x0 >> 1) - 4, (y0 >> 1) - 1, z >> 1);
    };
    // ---- wave scheduling: wait until the producers of this stage's iterate have written the plane of iteration `it` ----
    // (warp 0, converged).  `known` caches the progress of the producers in this block's own chunk.
    int known = 0;
    auto wait_dep = [&](int it) {
        if (!WAVE || wc.dep_prog == nullptr) return;
        // the plane of iteration `it` in march order: position it - 1 of this chunk; position -1 is the last-but-first plane
        // of the chunk behind the start, position len the plane beyond the end -- both lie in a neighbouring chunk that
        // marches the other way (or are ghost planes: the mirrored plane is this chunk's own first / last plane)
        const int len = zc1 - zc0;
        int c = wc.chunk, need = it;                                // own chunk: positions 0 .. it - 1 complete
        if (it == 0) {
            const int cn = wc.chunk - dir;                          // chunk behind the start; it starts at the same boundary
            if (cn >= 0 && cn < wc.nch) { c = cn; need = 1; } else need = 1;
        } else if (it == len + 1) {
            const int cn = wc.chunk + dir;                          // chunk beyond the end; it ends at the same boundary
            if (cn >= 0 && cn < wc.nch) { c = cn; need = min(wc.zchunk, nz - cn * wc.zchunk); } else need = len;
        }
        if (c == wc.chunk && known >= need) return;
        const int lane = tid & 31;
        const int ddx = lane % 3 - 1, ddy = (lane / 3) % 3 - 1;
        const int ux = wc.tx + ddx, uy = wc.ty + ddy;
        const bool valid = lane < 9 && ux >= 0 && ux < wc.gx && uy >= 0 && uy < wc.gy;
        const int* fp = wc.dep_prog + ((size_t)c * wc.gy + (valid ? uy : wc.ty)) * wc.gx + (valid ? ux : wc.tx);
        int m = 0;
        for (long long spin = 0;; ++spin) {
            const int v = valid ? ld_acquire_gpu(fp) : 0x7fffffff;
            m = __reduce_min_sync(0xffffffffu, v);
            if (m >= need) break;
            if (spin > (1ll << 22)) { if (lane == 0) atomicExch(wc.err, 1); break; }   // ~ seconds: give up, flag the error
            __nanosleep(64);
        }
        __syncwarp();
        if (c == wc.chunk) known = m;
    };
    // publish: `count` planes of this chunk are complete (called by thread 0 after a block barrier that follows their stores)
    auto publish = [&](int count) {
        if (!WAVE || wc.my_prog == nullptr) return;
        // the consumers read these planes through TMA (async proxy); the release makes the block's stores (ordered before
        // this thread by the block barrier) visible at gpu scope before the flag
        asm volatile("fence.proxy.async.global;" ::: "memory");
        st_release_gpu(wc.my_prog, count);
    };

    if (tid == 0) {
#pragma unroll
        for (int q = 0; q < NS; ++q) mbar_init(&bars[q], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    }
    if (MODE == MODE_SWEEP && P.zero_x)
        for (int e = tid; e < NS * PLANE; e += C::NT) ring[(e / PLANE) * SLOT + (e % PLANE)] = 0.f;
    if (MODE == MODE_SEED)
        for (int e = tid; e < NS * C::BPLANE; e += C::NT) ring[(e / C::BPLANE) * SLOT + BOFF + (e % C::BPLANE)] = 0.f;
    __syncthreads();
    // Programmatic dependent launch: everything above touched only kernel parameters; the fields written by the previous
    // kernel of the cycle are first read below.  The next kernel may begin its own prologue from here on.
    asm volatile("griddepcontrol.wait;" ::: "memory");
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    if (WAVE) {
        if (tid < 32)
            for (int q = 0; q < NS && q < niter; ++q) {
                wait_dep(q);
                if (tid == 0) {
                    if (wc.dep_prog) asm volatile("fence.proxy.async.global;" ::: "memory");
                    issue(q);
                }
            }
    } else if (tid == 0)
        for (int q = 0; q < NS && q < niter; ++q) issue(q);

    // ---- per-point state carried along z ---------------------------------------------------------
    u64 xA[2][2], zA[2][2], kA[2][2];        // S accumulators [row][column pair] of x, k x, k ...
    u64 xB[2][2][2], zB[2][2][2], kB[2][2][2];   // ... B double-buffered by plane parity [parity][row][pair]
    u64 xo[2][2][2], ko[2][2][2];            // own values [plane parity][row][column pair]
    float hold0 = 0.f, hold1 = 0.f;          // restriction: sums of the even plane
#pragma unroll
    for (int j = 0; j < 2; ++j)
#pragma unroll
        for (int c = 0; c < 2; ++c) {
            xA[j][c] = zA[j][c] = kA[j][c] = 0ull;
            xB[0][j][c] = zB[0][j][c] = kB[0][j][c] = xB[1][j][c] = zB[1][j][c] = kB[1][j][c] = 0ull;
            xo[0][j][c] = xo[1][j][c] = ko[0][j][c] = ko[1][j][c] = 0ull;
        }
    const u64 two = bc2(2.f);
    const float omega = P.omega;
    const int nxc = nx >> 1, nyc = ny >> 1;

    // one plane: PAR = parity of the iteration index
    auto body = [&](auto par_tag, const int it) {
        constexpr int PAR = decltype(par_tag)::value;
        const int p = pfirst + dir * it;
        const int slot = it & (NS - 1);
        // ---- ring hand-back: everyone has finished iteration it - 1, so its slot can be refilled ----
        __syncthreads();
        if (WAVE) {
            if (tid < 32) {
                if (it >= 1 && it - 1 + NS < niter) {
                    wait_dep(it - 1 + NS);
                    if (tid == 0) {
                        // slot reuse: generic reads of the slot before the TMA write; and the producers' stores (acquired in
                        // wait_dep) before the TMA read of global memory.  (A plain fence.proxy.async is a full MEMBAR.GPU.)
                        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
                        if (wc.dep_prog) asm volatile("fence.proxy.async.global;" ::: "memory");
                        issue(it - 1 + NS);
                    }
                }
                // iterations <= it - 1 are complete: they finalised the chunk positions 0 .. it - 3
                if (tid == 0 && PAR == 0 && it >= 4) publish(it - 2);
            }
        } else if (tid == 0 && it >= 1 && it - 1 + NS < niter) {
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
            issue(it - 1 + NS);
        }
        mbar_wait(&bars[slot], (uint32_t)((it / NS) & 1));

        const uint32_t so = (uint32_t)(slot * SLOT * 4);
        const bool zghost = p < 0 || p >= nz;
        const float fz = zghost ? (p < 0 ? P.sz0 : P.sz1) : 1.f;
        const u64 fz2 = bc2(fz), twofz = bc2(2.f * fz);
        u64 Sx[2][2], Sz[2][2], Sk[2][2];

        // staged row q of x (with the PRO correction), of k, and their product; x sums of the three
        auto stage = [&](int q, RT& sx, RT& sk, RT& sz) {
            const uint32_t a = raddr[q] + so;
            Row w;
            lds128(a, w.p, w.q);
            w.l = lds32(a - 4); w.r = lds32(a + 16);
            if (MODE == MODE_PRO) {
                const uint32_t ca = caddr[q == 0 ? 0 : (q == 3 ? 2 : 1)] + so;
                const u64 c12 = lds64(ca + 4);                       // coarse cells gi0/2, gi0/2 + 1
                w.p = add2(w.p, bc2(lo(c12))); w.q = add2(w.q, bc2(hi(c12)));
                w.l += lds32(ca); w.r += lds32(ca + 12);             // gi0/2 - 1, gi0/2 + 2
            }
            w.l = fmaf(glx, lo(w.p), w.l); w.r = fmaf(grx, hi(w.q), w.r);
            if (q == 1) { xo[PAR][0][0] = w.p; xo[PAR][0][1] = w.q; }
            if (q == 2) { xo[PAR][1][0] = w.p; xo[PAR][1][1] = w.q; }
            sx = row_sums(w, two);
            if (VAR) {
                const Row kw = load_row(a + KOFF * 4, glk, grk);
                if (q == 1) { ko[PAR][0][0] = kw.p; ko[PAR][0][1] = kw.q; }
                if (q == 2) { ko[PAR][1][0] = kw.p; ko[PAR][1][1] = kw.q; }
                sk = row_sums(kw, two);
                Row zw; zw.p = mul2(kw.p, w.p); zw.q = mul2(kw.q, w.q); zw.l = kw.l * w.l; zw.r = kw.r * w.r;
                sz = row_sums(zw, two);
            }
        };
        {
            RT sx0, sk0, sz0, sx1, sk1, sz1, sx2, sk2, sz2, sx3, sk3, sz3;
            stage(0, sx0, sk0, sz0);
            stage(1, sx1, sk1, sz1);
            stage(2, sx2, sk2, sz2);
            out_row<1>(sx0, sx1, sx2, f0, two, fz2, twofz, xA[0], xB[PAR ^ 1][0], xB[PAR][0], Sx[0]);
            if (VAR) {
                out_row<1>(sz0, sz1, sz2, f0, two, fz2, twofz, zA[0], zB[PAR ^ 1][0], zB[PAR][0], Sz[0]);
                out_row<0>(sk0, sk1, sk2, f0, two, fz2, twofz, kA[0], kB[PAR ^ 1][0], kB[PAR][0], Sk[0]);
            }
            stage(3, sx3, sk3, sz3);
            out_row<2>(sx1, sx2, sx3, f3, two, fz2, twofz, xA[1], xB[PAR ^ 1][1], xB[PAR][1], Sx[1]);
            if (VAR) {
                out_row<2>(sz1, sz2, sz3, f3, two, fz2, twofz, zA[1], zB[PAR ^ 1][1], zB[PAR][1], Sz[1]);
                out_row<0>(sk1, sk2, sk3, f3, two, fz2, twofz, kA[1], kB[PAR ^ 1][1], kB[PAR][1], Sk[1]);
            }
        }

        if (PAR == 0 && it == 0 && zghost) {   // the ghost plane below the domain: its Pp enters the plane above scaled
#pragma unroll
            for (int j = 0; j < 2; ++j)
#pragma unroll
                for (int c = 0; c < 2; ++c) {
                    xB[PAR][j][c] = mul2(xB[PAR][j][c], fz2);
                    if (VAR) zB[PAR][j][c] = mul2(zB[PAR][j][c], fz2);
                }
        }

        // ---- finalise plane p - 1 ----
        const int qc = p - dir;
        if (it >= 2) {
            const u64 icc2 = bc2(P.icc), cc2 = bc2(P.cc), om12 = bc2(MODE == MODE_SEED ? P.om_x : 1.f - omega);
            const float om_g = MODE == MODE_SEED ? P.om_g : omega;
            float rs0 = 0.f, rs1 = 0.f;
#pragma unroll
            for (int j = 0; j < RY; ++j) {
                u64 b4[2];
                lds128(baddr + so + j * (C::TX * 4), b4[0], b4[1]);
                u64 o[2];
#pragma unroll
                for (int c = 0; c < 2; ++c) {
                    const u64 bv = b4[c];
                    const u64 xv = xo[PAR ^ 1][j][c];
                    if (VAR) {
                        const u64 kv = ko[PAR ^ 1][j][c];
                        const u64 Dp = fma2(kv, bc2(32.f), Sk[j][c]);
                        const u64 t = fma2(kv, Sx[j][c], Sz[j][c]);
                        if (MODE == MODE_RR) {
                            o[c] = fma2(mul2(Dp, bc2(-P.cc)), xv, fma2(t, cc2, bv));
                        } else {
                            const u64 g = mul2(pk(rcpa(lo(Dp)), rcpa(hi(Dp))), bc2(om_g));
                            o[c] = fma2(g, fma2(bv, icc2, t), mul2(xv, om12));
                        }
                    } else {
                        const u64 s2 = add2(Sx[j][c], Sx[j][c]);
                        if (MODE == MODE_RR) o[c] = fma2(fma2(xv, bc2(-64.f), s2), cc2, bv);
                        else o[c] = fma2(bc2(om_g * (1.f / 64.f)), fma2(bv, icc2, s2), mul2(xv, om12));
                    }
                }
                if (MODE == MODE_RR) { rs0 += lo(o[0]) + hi(o[0]); rs1 += lo(o[1]) + hi(o[1]); }
                else if (active)
                    *reinterpret_cast<ulonglong2*>(P.out + ((size_t)qc * ny + (gj0 + j)) * nx + gi0) = make_ulonglong2(o[0], o[1]);
            }
            if (MODE == MODE_RR) {
                if (PAR == 0) {     // first plane of a pair {2m, 2m + 1} in march order (zc0, zc1 are even)
                    hold0 = rs0; hold1 = rs1;
                } else if (active) {
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
            }
        }
    };

    for (int it = 0; it < niter; it += 2) {
        body(std::integral_constant<int, 0>{}, it);
        body(std::integral_constant<int, 1>{}, it + 1);
    }
    if (WAVE && wc.my_prog != nullptr) {     // the whole chunk is complete
        __syncthreads();
        if (tid == 0) publish(zc1 - zc0);
    }
}

template <class C>
__global__ void __launch_bounds__(C::NT, C::MINB)
lean_kernel(const __grid_constant__ CUtensorMap tmx, const __grid_constant__ CUtensorMap tmk,
            const __grid_constant__ CUtensorMap tmb, const __grid_constant__ CUtensorMap tmc, const LParams P) {
    const WaveCtx none = {};
    lean_body<C, C::MODE, false>(tmx, tmk, tmb, tmc, P, blockIdx.x, blockIdx.y, blockIdx.z, none);
}

}  // namespace lk
}  // namespace mgb
