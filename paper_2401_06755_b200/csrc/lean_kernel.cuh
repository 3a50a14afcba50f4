// lean_kernel.cuh -- the fp32 streaming smoother / transfer kernel for uniform grids (sm_100a).
//
// One stencil stage per pass, three variants:
//   MODE_SWEEP   weighted-Jacobi sweep                                   x            -> x'
//   MODE_PRO     prolongation + correction + sweep                      x + P x_c    -> x'   (x_c tile staged by TMA too)
//   MODE_RES     residual r = b - A x (or y = A x) at full resolution, optionally with ||r||^2 in fp64    x            -> r
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

enum { MODE_SWEEP = 0, MODE_PRO = 1, MODE_RR = 2, MODE_SEED = 3, MODE_RES = 4 };

struct LParams {
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
    int zero_x;                 // SWEEP: the iterate is zero whatever `src` holds: its planes are not read (12 B/point, not 16)
    // MODE_SEED: the first TWO sweeps of a cycle from a zero guess in one pass over y = b / D (written by the defect kernel):
    // x_2 = omega (2 - omega) y + (omega^2 / D) cc (k S(y) + S(k y)) -- the sweep formula x' = om_x x + (om_g / D)(b + cc (..))
    // with om_g = omega^2, om_x = omega (2 - omega) and no b term (the b tiles are not fetched, their ring slots are cleared;
    // 12 B/point).  A mode of its own so that the code of the other modes is untouched.
    float om_g, om_x;
    // MODE_RES: out = rsign (b - A x) (out may be NULL); zero_b: b is absent (its tiles are not fetched), so with rsign = -1
    // out = A x; acc (may be NULL): sum of out^2 over the grid, accumulated in fp64, one atomic per block
    float rsign;
    int zero_b;
    double* acc;
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

template <class C>
__global__ void __launch_bounds__(C::NT, C::MINB)
lean_kernel(const __grid_constant__ CUtensorMap tmx, const __grid_constant__ CUtensorMap tmk,
            const __grid_constant__ CUtensorMap tmb, const __grid_constant__ CUtensorMap tmc, const LParams P) {
    constexpr int MODE = C::MODE;
    constexpr bool WAVE = false;
    const int bx = blockIdx.x, by = blockIdx.y, bz = blockIdx.z;
    const WaveCtx wc = {};
#include "lean_body.inc"
}

// the same body as a device function, one per mode, for wave_kernel.cuh
template <class C, int MODE, bool WAVE>
__device__ __forceinline__ void lean_body(const CUtensorMap& tmx, const CUtensorMap& tmk, const CUtensorMap& tmb,
                                          const CUtensorMap& tmc, const LParams& P, const int bx, const int by, const int bz,
                                          const WaveCtx& wc) {
#include "lean_body.inc"
}

}  // namespace lk
}  // namespace mgb
