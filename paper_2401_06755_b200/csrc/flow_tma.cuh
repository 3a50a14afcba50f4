// flow_tma.cuh -- the explicit stencil kernels of flow_march.cuh with their inputs STAGED BY TMA (fp32, nx % 4 == 0, 16-byte
// aligned fields; included by flow.cu inside its namespace, after flow_march.cuh).
//
// Same arithmetic, same thread geometry (32 x 4 threads, W = 4 points per thread, 16 output planes per block, march along z),
// same helpers (in_plane, ZAcc, GradRoll) -- only where the 3 x 3 neighbourhoods come from differs.  The marching kernels read
// them with plain global loads and wait for each plane (3-17 long-scoreboard stall cycles per issued instruction at 28-45 %
// occupancy, profiles/r02_ncu_flow.md); here one thread asks TMA for the planes three iterations ahead
// (cp.async.bulk.tensor.3d into a 4-deep shared-memory ring, mbarrier completion, as lean_kernel.cuh), and the threads read
// shared memory: one 128-bit and two 32-bit loads per row.  Stencil fields are staged with one halo row and four halo columns
// per side (TMA boxes start at multiples of 16 bytes); fields used at the centre only are staged as plain tiles, one plane
// behind (they are needed when a plane is finalised).  Halos are the zero-derivative copies of flow_march.cuh: rows and planes
// by clamped indices, columns by the thread's own end value.
#pragma once

namespace ft {

constexpr int W = 4, TX = W * MBX, TY = MBY, NT = MBX * MBY;
constexpr int PX = TX + 8, PY = TY + 2;
constexpr int SPLANE = ((PX * PY + 31) / 32) * 32;        // floats per staged stencil plane
constexpr int CPLANE = TX * TY;                            // floats per staged centre tile
constexpr int NS = 4;                                      // default ring depth (3 where the slots are large: blocks per SM matter more)
constexpr int MAXF = 6;
constexpr uint32_t SBYTES = PX * PY * 4, CBYTES = TX * TY * 4;

struct alignas(64) Maps { CUtensorMap m[MAXF]; };          // stencil fields first, then centre fields

template <int NSF, int NCF, int ND = NS>
struct Ring {
    static constexpr int SLOT = NSF * SPLANE + NCF * CPLANE;
    static constexpr size_t SMEM = (size_t)(32 + ND * SLOT) * sizeof(float);
};

typedef Pk<float, W> V4;

// the thread's view of the staged tiles
struct View {
    uint32_t row[3];      // byte offset of the thread's first column in staged rows j - 1, j, j + 1 (clamped) of a stencil plane
    uint32_t cen;         // byte offset of the thread's 4 values in a centre tile
    bool lin, rin;        // the left / right x neighbour exists (otherwise: copy of the own end value)
};

__device__ __forceinline__ View make_view(const Geo<float>& G, int x0, int y0, int lx, int ly) {
    View v;
    const int gj = y0 + ly, gi = x0 + W * lx;
#pragma unroll
    for (int b = 0; b < 3; ++b) {
        const int r = min(max(gj - 1 + b, 0), G.ny - 1) - (y0 - 1);                 // 0 .. PY - 1 for rows inside the domain
        v.row[b] = 4u * (uint32_t)(min(max(r, 0), PY - 1) * PX + 4 + W * lx);
    }
    v.cen = 4u * (uint32_t)(ly * TX + W * lx);
    v.lin = gi > 0; v.rin = gi + W < G.nx;
    return v;
}

// 3 x 3 neighbourhood of the thread's 4 points from a staged stencil plane at shared address `a`
__device__ __forceinline__ void load9s(uint32_t a, const View& vw, V4 (&v)[3][3]) {
#pragma unroll
    for (int b = 0; b < 3; ++b) {
        const uint32_t r = a + vw.row[b];
        lk::u64 p, q;
        lk::lds128(r, p, q);
        const float l = lk::lds32(r - 4), rr = lk::lds32(r + 16);
        V4& c = v[b][1];
        c[0] = lk::lo(p); c[1] = lk::hi(p); c[2] = lk::lo(q); c[3] = lk::hi(q);
        v[b][0][0] = vw.lin ? l : c[0]; v[b][2][3] = vw.rin ? rr : c[3];
#pragma unroll
        for (int e = 1; e < W; ++e) { v[b][0][e] = c[e - 1]; v[b][2][e - 1] = c[e]; }
    }
}
__device__ __forceinline__ V4 ldc(uint32_t a, const View& vw) {
    lk::u64 p, q;
    lk::lds128(a + vw.cen, p, q);
    V4 c; c[0] = lk::lo(p); c[1] = lk::hi(p); c[2] = lk::lo(q); c[3] = lk::hi(q);
    return c;
}

// The staging pipeline of one block.  Iteration `it` (0 .. niter - 1) works on stencil plane z0 - 1 + it and finalises output
// plane q = z0 - 2 + it, whose centre tiles arrive in the same slot.
template <int NSF, int NCF, int ND = NS>
struct Pipe {
    typedef Ring<NSF, NCF, ND> R;
    uint64_t* bars; float* ring; uint32_t ring_a;
    const Maps* maps;
    int x0, y0, z0, nz, niter;

    __device__ __forceinline__ void issue(int it) const {            // one thread
        uint64_t* bar = &bars[it % ND];
        float* dst = ring + (it % ND) * R::SLOT;
        const int z = min(max(z0 - 1 + it, 0), nz - 1), q = z0 - 2 + it;
        const bool wc = NCF > 0 && it >= 2;                            // q lies in the chunk
        lk::mbar_expect_tx(bar, NSF * SBYTES + (wc ? NCF * CBYTES : 0u));
#pragma unroll
        for (int f = 0; f < NSF; ++f) lk::tma_load_plane(dst + f * SPLANE, &maps->m[f], bar, x0 - 4, y0 - 1, z);
        if (wc) {
#pragma unroll
            for (int f = 0; f < NCF; ++f) lk::tma_load_plane(dst + NSF * SPLANE + f * CPLANE, &maps->m[NSF + f], bar, x0, y0, q);
        }
    }
    __device__ __forceinline__ void start(const Maps& M, int bx, int by, int bz, int nz_, int z1) {
        extern __shared__ __align__(1024) float smf[];
        bars = reinterpret_cast<uint64_t*>(smf); ring = smf + 32; ring_a = lk::smem_u32(ring);
        maps = &M; x0 = bx * TX; y0 = by * TY; z0 = bz * MZC; nz = nz_; niter = z1 - z0 + 2;
        if (threadIdx.x == 0 && threadIdx.y == 0) {
#pragma unroll
            for (int f = 0; f < NSF + NCF; ++f) asm volatile("prefetch.tensormap [%0];" ::"l"(reinterpret_cast<uint64_t>(&M.m[f])) : "memory");
#pragma unroll
            for (int s = 0; s < ND; ++s) lk::mbar_init(&bars[s], 1);
            asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        }
        __syncthreads();
        if (threadIdx.x == 0 && threadIdx.y == 0)
            for (int s = 0; s < ND && s < niter; ++s) issue(s);
    }
    // top of iteration `it`: hand the slot of iteration it - 1 back to TMA, wait for this iteration's planes;
    // returns the shared address of the slot
    __device__ __forceinline__ uint32_t acquire(int it) const {
        __syncthreads();
        if (threadIdx.x == 0 && threadIdx.y == 0 && it >= 1 && it - 1 + ND < niter) {
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
            issue(it - 1 + ND);
        }
        lk::mbar_wait(&bars[it % ND], (uint32_t)((it / ND) & 1));
        return ring_a + 4u * (uint32_t)((it % ND) * R::SLOT);
    }
    __device__ __forceinline__ uint32_t sfield(uint32_t slot, int f) const { return slot + 4u * (uint32_t)(f * SPLANE); }
    __device__ __forceinline__ uint32_t cfield(uint32_t slot, int f) const { return slot + 4u * (uint32_t)(NSF * SPLANE + f * CPLANE); }
};

// steps 1-2 of reading C9: adv = u psi_x + v psi_y + w psi_z      (maps: psi | u, v, w)
__global__ void __launch_bounds__(NT) advection_tma(const __grid_constant__ Maps M, const Geo<float> G, float* __restrict__ adv) {
    Pipe<1, 3> P;
    const Col<float, W> c = make_col<float, W>(G);
    P.start(M, blockIdx.x, blockIdx.y, blockIdx.z, G.nz, c.z1);
    const View vw = make_view(G, P.x0, P.y0, threadIdx.x, threadIdx.y);
    GradRoll<float, V4> g; g.init();
    for (int it = 0; it < P.niter; ++it) {
        const uint32_t slot = P.acquire(it);
        V4 n9[3][3];
        load9s(P.sfield(slot, 0), vw, n9);
        g.add(G, in_plane<float, true, false>(G, n9));
        const int q = c.z0 - 2 + it;
        if (q >= c.z0 && c.ok) {
            V4 gx, gy, gz; g.grad(G, gx, gy, gz);
            stv(adv + at(c, q), ldc(P.cfield(slot, 0), vw) * gx + ldc(P.cfield(slot, 1), vw) * gy + ldc(P.cfield(slot, 2), vw) * gz);
        }
    }
}

// steps 11-12 (vof_diffusion_march): sC = adv + sum_d diff_d, Cnew = C - dt sC      (maps: C, k^x, k^y, k^z | adv)
__global__ void __launch_bounds__(NT) vof_diffusion_tma(const __grid_constant__ Maps M, const Geo<float> G, float dt, float* __restrict__ sC,
                                                        float* __restrict__ Cnew) {
    typedef V4 V;
    Pipe<4, 1> P;
    const Col<float, W> c = make_col<float, W>(G);
    P.start(M, blockIdx.x, blockIdx.y, blockIdx.z, G.nz, c.z1);
    const View vw = make_view(G, P.x0, P.y0, threadIdx.x, threadIdx.y);
    Diff3<V> dx, dy, dz; dx.init(); dy.init(); dz.init();
    V C0 = {}, C0n = {}, k0[3] = {}, k0n[3] = {};
    for (int it = 0; it < P.niter; ++it) {
        const uint32_t slot = P.acquire(it);
        V nc[3][3], nk[3][3], nz9[3][3];
        load9s(P.sfield(slot, 0), vw, nc);
        const InPlane<V> rc = in_plane<float, false, true>(G, nc);
        C0 = C0n; C0n = nc[1][1];
        V pk[3], pz[3];
#pragma unroll
        for (int d = 0; d < 3; ++d) {
            load9s(P.sfield(slot, 1 + d), vw, nk);
#pragma unroll
            for (int b = 0; b < 3; ++b)
#pragma unroll
                for (int a = 0; a < 3; ++a) nz9[b][a] = nk[b][a] * nc[b][a];
            k0[d] = k0n[d]; k0n[d] = nk[1][1];
            if (d == 2) {
                pk[d] = in_plane<float, false, false>(G, nk).mm; pz[d] = in_plane<float, false, false>(G, nz9).mm;
            } else {
                const InPlane<V> rk = in_plane<float, false, true>(G, nk), rz = in_plane<float, false, true>(G, nz9);
                pk[d] = d == 0 ? rk.km : rk.mk; pz[d] = d == 0 ? rz.km : rz.mk;
            }
        }
        const V xf = dx.f.stepM(G, rc.km), xk = dx.k.stepM(G, pk[0]), xz = dx.z.stepM(G, pz[0]);
        const V yf = dy.f.stepM(G, rc.mk), yk = dy.k.stepM(G, pk[1]), yz = dy.z.stepM(G, pz[1]);
        const V zf = dz.f.stepK(G, rc.mm), zk = dz.k.stepK(G, pk[2]), zz = dz.z.stepK(G, pz[2]);
        const int q = c.z0 - 2 + it;
        if (q >= c.z0 && c.ok) {
            const V ddx = 0.5f * (xz + k0[0] * xf - C0 * xk);
            const V ddy = 0.5f * (yz + k0[1] * yf - C0 * yk);
            const V ddz = 0.5f * (zz + k0[2] * zf - C0 * zk);
            const size_t c0 = at(c, q);
            const V sv = ldc(P.cfield(slot, 0), vw) + ddx + ddy + ddz;
            if (sC) stv(sC + c0, sv);
            if (Cnew) stv(Cnew + c0, C0 - dt * sv);
        }
    }
}

// steps 3-10 (vof_coeff_march with the 3-point detectors of Eq. 33): k^x, k^y, k^z      (maps: C, adv | u, v, w)
__global__ void __launch_bounds__(NT) vof_coeff_tma(const __grid_constant__ Maps M, const Geo<float> G, float k_min, float k_max,
                                                    float* __restrict__ kx, float* __restrict__ ky, float* __restrict__ kz) {
    typedef V4 V;
    typedef float T;
    Pipe<2, 3> P;
    const Col<float, W> c = make_col<float, W>(G);
    P.start(M, blockIdx.x, blockIdx.y, blockIdx.z, G.nz, c.z1);
    const View vw = make_view(G, P.x0, P.y0, threadIdx.x, threadIdx.y);
    const T Kp = T(300), Km = T(300);        // K+, K- 
    const T beta = T(0.1), eps_x = T(1e-4);  // Eq. 36
    const T Kcal = T(3);                     // Eq. 39
    const T ih[3] = {T(1) / G.h[0], T(1) / G.h[1], T(1) / G.h[2]};
    GradRoll<T, V> g; g.init();
    ZAcc<V> am; am.init();
    V a0 = {}, a0n = {};
    V Cc[3] = {};
    V Sx = {}, Sxn = {}, Sy = {}, Syn = {};
    for (int it = 0; it < P.niter; ++it) {
        const uint32_t slot = P.acquire(it);
        V n9[3][3];
        load9s(P.sfield(slot, 0), vw, n9);
        g.add(G, in_plane<T, true, false>(G, n9));
        push(Cc, n9[1][1]);
        Sx = Sxn; Sy = Syn;
        Sxn = (n9[1][1] - n9[1][0]) * (n9[1][2] - n9[1][1]);
        Syn = (n9[1][1] - n9[0][1]) * (n9[2][1] - n9[1][1]);
        load9s(P.sfield(slot, 1), vw, n9);
        const V madv = am.stepM(G, in_plane<T, false, false>(G, n9).mm);
        a0 = a0n; a0n = n9[1][1];
        const int q = c.z0 - 2 + it;
        if (q >= c.z0 && c.ok) {
            V Cx, Cy, Cz; g.grad(G, Cx, Cy, Cz);
            const V a = T(2) * (madv - a0);
            const V kabs = k_abs_pk(G, a, Cx, Cy, Cz);
            const V C0 = Cc[1];
            V S[3] = {Sx, Sy, (C0 - Cc[0]) * (Cc[2] - C0)};
#pragma unroll
            for (int e = 0; e < W; ++e)
                if (C0[e] > T(0.95) || C0[e] < T(0.05)) S[0][e] = S[1][e] = S[2][e] = T(-1);
            const size_t c0 = at(c, q);
            const V uu = ldc(P.cfield(slot, 0), vw), vv = ldc(P.cfield(slot, 1), vw), ww = ldc(P.cfield(slot, 2), vw);
            const V g2 = Cx * Cx + Cy * Cy + Cz * Cz;
            const V gq = pdiv(uu * Cx + vv * Cy + ww * Cz, eps_x + g2);
            const V us = gq * Cx, vs = gq * Cy, ws = gq * Cz;
            const V kneg = pdiv(-beta * (uu * uu + vv * vv + ww * ww), eps_x + g2 * (pabs(us) + pabs(vs) + pabs(ws)) * T(1.0 / 3.0));
            T* const out[3] = {kx, ky, kz};
#pragma unroll
            for (int d = 0; d < 3; ++d) {
                const V wp = -pmax(T(-1), pmin(T(0), Kp * S[d]));
                const V wm = pmin(T(1), pmax(T(0), Km * S[d]));
                const V kk = wp * (Kcal * kabs) + wm * (kneg * ih[d]);
                stv(out[d] + c0, pmax(-k_min, pmin(k_max, kk)));
            }
        }
    }
}

// The advection terms of the three momentum components in one pass (advection3_march)      (maps: u, v, w | -)
template <bool BC>
__global__ void __launch_bounds__(NT) advection3_tma(const __grid_constant__ Maps M, const Geo<float> G, float* __restrict__ au,
                                                     float* __restrict__ av, float* __restrict__ aw, const Halo6<float> Hu,
                                                     const Halo6<float> Hv, const Halo6<float> Hw) {
    typedef V4 V;
    Pipe<3, 0> P;
    const Col<float, W> c = make_col<float, W>(G);
    P.start(M, blockIdx.x, blockIdx.y, blockIdx.z, G.nz, c.z1);
    const View vw = make_view(G, P.x0, P.y0, threadIdx.x, threadIdx.y);
    HaloFac<float> hu = {}, hv = {}, hw = {};
    if (BC) { hu = halo_fac(G, c, Hu); hv = halo_fac(G, c, Hv); hw = halo_fac(G, c, Hw); }
    GradRoll<float, V> gu, gv, gw; gu.init(); gv.init(); gw.init();
    V cu = {}, cv = {}, cw = {};
    for (int it = 0; it < P.niter; ++it) {
        const uint32_t slot = P.acquire(it);
        const int z = c.z0 - 1 + it;
        V n9[3][3];
        load9s(P.sfield(slot, 0), vw, n9);
        if (BC) halo_scale(G, Hu, hu, z, n9);
        gu.add(G, in_plane<float, true, false>(G, n9));
        const V nu = n9[1][1];
        load9s(P.sfield(slot, 1), vw, n9);
        if (BC) halo_scale(G, Hv, hv, z, n9);
        gv.add(G, in_plane<float, true, false>(G, n9));
        const V nv = n9[1][1];
        load9s(P.sfield(slot, 2), vw, n9);
        if (BC) halo_scale(G, Hw, hw, z, n9);
        gw.add(G, in_plane<float, true, false>(G, n9));
        const V nw = n9[1][1];
        const int q = z - 1;
        if (q >= c.z0 && c.ok) {
            const size_t c0 = at(c, q);
            V gx, gy, gz;
            gu.grad(G, gx, gy, gz); stv(au + c0, cu * gx + cv * gy + cw * gz);
            gv.grad(G, gx, gy, gz); stv(av + c0, cu * gx + cv * gy + cw * gz);
            gw.grad(G, gx, gy, gz); stv(aw + c0, cu * gx + cv * gy + cw * gz);
        }
        cu = nu; cv = nv; cw = nw;
    }
}

// k_c = rho min{k_max, k_abs(c)} + mu (mom_coeff_march)      (maps: comp, adv | C, u, v, w)
template <bool BC>
__global__ void __launch_bounds__(NT) mom_coeff_tma(const __grid_constant__ Maps M, const Geo<float> G, float rho_l, float rho_g, float mu_l,
                                                    float mu_g, float* __restrict__ kc, const Halo6<float> H) {
    typedef V4 V;
    typedef float T;
    Pipe<2, 4, 3> P;
    const Col<float, W> c = make_col<float, W>(G);
    P.start(M, blockIdx.x, blockIdx.y, blockIdx.z, G.nz, c.z1);
    const View vw = make_view(G, P.x0, P.y0, threadIdx.x, threadIdx.y);
    HaloFac<T> hf = {};
    if (BC) hf = halo_fac(G, c, H);
    GradRoll<T, V> g; g.init();
    ZAcc<V> am; am.init();
    V a0 = {}, a0n = {};
    for (int it = 0; it < P.niter; ++it) {
        const uint32_t slot = P.acquire(it);
        const int z = c.z0 - 1 + it;
        V n9[3][3];
        load9s(P.sfield(slot, 0), vw, n9);
        if (BC) halo_scale(G, H, hf, z, n9);
        g.add(G, in_plane<T, true, false>(G, n9));
        load9s(P.sfield(slot, 1), vw, n9);
        const V madv = am.stepM(G, in_plane<T, false, false>(G, n9).mm);
        a0 = a0n; a0n = n9[1][1];
        const int q = z - 1;
        if (q >= c.z0 && c.ok) {
            V px, py, pz; g.grad(G, px, py, pz);
            const V a = T(2) * (madv - a0);
            const V Cc = ldc(P.cfield(slot, 0), vw);
            const V rho = mix01(rho_l, rho_g, Cc);
            const V mu = mix01(mu_l, mu_g, Cc);
            const V kmax = G.h[0] * pabs(ldc(P.cfield(slot, 1), vw)) + G.h[1] * pabs(ldc(P.cfield(slot, 2), vw)) + G.h[2] * pabs(ldc(P.cfield(slot, 3), vw));
            stv(kc + at(c, q), rho * pmin(kmax, k_abs_pk(G, a, px, py, pz)) + mu);
        }
    }
}

// s = rho adv + f^lap(c, k_c), q~ = q_n - dt s / rho, q_half' = (q_n + q~) / 2 (mom_update_march)      (maps: comp, k_c | C, adv, q_n)
template <bool BC>
__global__ void __launch_bounds__(NT) mom_update_tma(const __grid_constant__ Maps M, const Geo<float> G, float rho_l, float rho_g, float dt,
                                                     float* __restrict__ qt, float* __restrict__ qhn, const Halo6<float> H) {
    typedef V4 V;
    typedef float T;
    Pipe<2, 3, 3> P;
    const Col<float, W> c = make_col<float, W>(G);
    P.start(M, blockIdx.x, blockIdx.y, blockIdx.z, G.nz, c.z1);
    const View vw = make_view(G, P.x0, P.y0, threadIdx.x, threadIdx.y);
    HaloFac<T> hf = {};
    if (BC) hf = halo_fac(G, c, H);
    Diff3<V> L; L.init();
    V x0 = {}, x0n = {}, k0 = {}, k0n = {};
    for (int it = 0; it < P.niter; ++it) {
        const uint32_t slot = P.acquire(it);
        const int z = c.z0 - 1 + it;
        V nx9[3][3], nk9[3][3], nz9[3][3];
        load9s(P.sfield(slot, 0), vw, nx9);
        if (BC) halo_scale(G, H, hf, z, nx9);
        load9s(P.sfield(slot, 1), vw, nk9);
#pragma unroll
        for (int b = 0; b < 3; ++b)
#pragma unroll
            for (int a = 0; a < 3; ++a) nz9[b][a] = nk9[b][a] * nx9[b][a];
        const InPlane<V> rx = in_plane<T, false, true>(G, nx9), rk = in_plane<T, false, true>(G, nk9), rz = in_plane<T, false, true>(G, nz9);
        auto lap = [&](ZAcc<V>& a, const InPlane<V>& r) {
            const V p1 = r.km + r.mk, t = G.M[0] * p1 + G.K[2][0] * r.mm;
            return a.step(t, G.M[1] * p1 + G.K[2][1] * r.mm, t);
        };
        const V Lx = lap(L.f, rx), Lk = lap(L.k, rk), Lz = lap(L.z, rz);
        x0 = x0n; x0n = nx9[1][1]; k0 = k0n; k0n = nk9[1][1];
        const int q = z - 1;
        if (q >= c.z0 && c.ok) {
            const V diff = T(0.5) * (Lz + k0 * Lx - x0 * Lk);
            const size_t c0 = at(c, q);
            const V rho = mix01(rho_l, rho_g, ldc(P.cfield(slot, 0), vw));
            const V sv = rho * ldc(P.cfield(slot, 1), vw) + diff;
            const V qv = ldc(P.cfield(slot, 2), vw);
            const V t = qv - dt * sv / rho;
            stv(qt + c0, t);
            if (qhn) stv(qhn + c0, T(0.5) * (qv + t));
        }
    }
}

// b = -(1/dt) (f(u; w_x) + f(v; w_y) + f(w; w_z)) (pressure_rhs_march)      (maps: u, v, w | -)
template <bool BC>
__global__ void __launch_bounds__(NT) pressure_rhs_tma(const __grid_constant__ Maps M, const Geo<float> G, float inv_dt, float* __restrict__ bout,
                                                       const Halo6<float> Hu, const Halo6<float> Hv, const Halo6<float> Hw) {
    typedef V4 V;
    Pipe<3, 0, 3> P;
    const Col<float, W> c = make_col<float, W>(G);
    P.start(M, blockIdx.x, blockIdx.y, blockIdx.z, G.nz, c.z1);
    const View vw = make_view(G, P.x0, P.y0, threadIdx.x, threadIdx.y);
    HaloFac<float> fu = {}, fv = {}, fw = {};
    if (BC) { fu = halo_fac(G, c, Hu); fv = halo_fac(G, c, Hv); fw = halo_fac(G, c, Hw); }
    ZAcc<V> acc; acc.init();
    for (int it = 0; it < P.niter; ++it) {
        const uint32_t slot = P.acquire(it);
        const int z = c.z0 - 1 + it;
        V n9[3][3];
        load9s(P.sfield(slot, 0), vw, n9); if (BC) halo_scale(G, Hu, fu, z, n9); const V du = in_plane<float, true, false>(G, n9).dm;
        load9s(P.sfield(slot, 1), vw, n9); if (BC) halo_scale(G, Hv, fv, z, n9); const V dv = in_plane<float, true, false>(G, n9).md;
        load9s(P.sfield(slot, 2), vw, n9); if (BC) halo_scale(G, Hw, fw, z, n9); const V mw = in_plane<float, false, false>(G, n9).mm;
        const V ms = G.M[0] * (du + dv), dw = G.D[2][2] * mw;
        const V div = acc.step(ms + dw, G.M[1] * (du + dv), ms - dw);
        const int q = z - 1;
        if (q >= c.z0 && c.ok) stv(bout + at(c, q), -div * inv_dt);
    }
}

// q <- q - dt k f(p; w_x|y|z) (project_march); the pressure halo carries the solver's factors G.s      (maps: p | k, u, v, w)
__global__ void __launch_bounds__(NT) project_tma(const __grid_constant__ Maps M, const Geo<float> G, float dt, float* __restrict__ u,
                                                  float* __restrict__ v, float* __restrict__ w) {
    typedef V4 V;
    Pipe<1, 4> P;
    const Col<float, W> c = make_col<float, W>(G);
    P.start(M, blockIdx.x, blockIdx.y, blockIdx.z, G.nz, c.z1);
    const View vw = make_view(G, P.x0, P.y0, threadIdx.x, threadIdx.y);
    Halo6<float> H;
#pragma unroll
    for (int f = 0; f < 6; ++f) H.s[f] = G.s[f];
    const HaloFac<float> hf = halo_fac(G, c, H);
    GradRoll<float, V> g; g.init();
    for (int it = 0; it < P.niter; ++it) {
        const uint32_t slot = P.acquire(it);
        const int z = c.z0 - 1 + it;
        V n9[3][3];
        load9s(P.sfield(slot, 0), vw, n9);
        halo_scale(G, H, hf, z, n9);
        g.add(G, in_plane<float, true, false>(G, n9));
        const int q = z - 1;
        if (q >= c.z0 && c.ok) {
            V gx, gy, gz; g.grad(G, gx, gy, gz);
            const size_t c0 = at(c, q);
            const V f = dt * ldc(P.cfield(slot, 0), vw);
            stv(u + c0, ldc(P.cfield(slot, 1), vw) - f * gx); stv(v + c0, ldc(P.cfield(slot, 2), vw) - f * gy); stv(w + c0, ldc(P.cfield(slot, 3), vw) - f * gz);
        }
    }
}

// n_t = grad C / (eps_t + |grad C|) (normals_march)      (maps: C | -)
__global__ void __launch_bounds__(NT) normals_tma(const __grid_constant__ Maps M, const Geo<float> G, float* __restrict__ nx_,
                                                  float* __restrict__ ny_, float* __restrict__ nz_) {
    typedef V4 V;
    Pipe<1, 0> P;
    const Col<float, W> c = make_col<float, W>(G);
    P.start(M, blockIdx.x, blockIdx.y, blockIdx.z, G.nz, c.z1);
    const View vw = make_view(G, P.x0, P.y0, threadIdx.x, threadIdx.y);
    const float eps_t = 1e-7f / G.h[0];
    GradRoll<float, V> g; g.init();
    for (int it = 0; it < P.niter; ++it) {
        const uint32_t slot = P.acquire(it);
        V n9[3][3];
        load9s(P.sfield(slot, 0), vw, n9);
        g.add(G, in_plane<float, true, false>(G, n9));
        const int q = c.z0 - 2 + it;
        if (q >= c.z0 && c.ok) {
            V gx, gy, gz; g.grad(G, gx, gy, gz);
            const V inv = 1.f / (eps_t + psqrt(gx * gx + gy * gy + gz * gz));
            const size_t c0 = at(c, q);
            stv(nx_ + c0, gx * inv); stv(ny_ + c0, gy * inv); stv(nz_ + c0, gz * inv);
        }
    }
}

// force field F = -(s + s_t) and the curvature (surface_tension_march)      (maps: C, n_x, n_y, n_z | -)
__global__ void __launch_bounds__(NT) surface_tension_tma(const __grid_constant__ Maps M, const Geo<float> G, float rho_l, float rho_g,
                                                          float grav, float sigma_t, float* __restrict__ fu, float* __restrict__ fv,
                                                          float* __restrict__ fw, float* __restrict__ kappa) {
    typedef V4 V;
    Pipe<4, 0> P;
    const Col<float, W> c = make_col<float, W>(G);
    P.start(M, blockIdx.x, blockIdx.y, blockIdx.z, G.nz, c.z1);
    const View vw = make_view(G, P.x0, P.y0, threadIdx.x, threadIdx.y);
    GradRoll<float, V> g; g.init();
    ZAcc<V> acc; acc.init();
    V C0 = {}, C0n = {};
    for (int it = 0; it < P.niter; ++it) {
        const uint32_t slot = P.acquire(it);
        V n9[3][3];
        load9s(P.sfield(slot, 0), vw, n9);
        g.add(G, in_plane<float, true, false>(G, n9));
        C0 = C0n; C0n = n9[1][1];
        load9s(P.sfield(slot, 1), vw, n9); const V dx = in_plane<float, true, false>(G, n9).dm;
        load9s(P.sfield(slot, 2), vw, n9); const V dy = in_plane<float, true, false>(G, n9).md;
        load9s(P.sfield(slot, 3), vw, n9); const V mz = in_plane<float, false, false>(G, n9).mm;
        const V ms = G.M[0] * (dx + dy), dn = G.D[2][2] * mz;
        const V divn = acc.step(ms + dn, G.M[1] * (dx + dy), ms - dn);
        const int q = c.z0 - 2 + it;
        if (q >= c.z0 && c.ok) {
            V gx, gy, gz; g.grad(G, gx, gy, gz);
            const V kap = -divn;
            const size_t c0 = at(c, q);
            const V sk = -sigma_t * kap;
            stv(fu + c0, sk * gx); stv(fv + c0, sk * gy);
            stv(fw + c0, sk * gz + grav * mix01(rho_l, rho_g, C0));
            if (kappa) stv(kappa + c0, kap);
        }
    }
}

// Forcing terms of Eq. 18 with both pressures and the force field present (mom_forcing_march)      (maps: p_hs, p_nh, F0, F1, F2 | -)
// C, q~ and q_n are read at the centre only, by plain loads; the bottom ghost plane of p_hs (mirror + h_z g rho) needs the 3 x 3
// neighbourhood of C in plane 0, read once by the blocks of the lowest chunk.
__global__ void __launch_bounds__(NT) mom_forcing_tma(const __grid_constant__ Maps M, const Geo<float> G, const float* __restrict__ C, float rho_l,
                                                      float rho_g, float grav, float dt, float* __restrict__ q0, float* __restrict__ q1,
                                                      float* __restrict__ q2, const float* __restrict__ n0, const float* __restrict__ n1,
                                                      const float* __restrict__ n2, float* __restrict__ h0, float* __restrict__ h1,
                                                      float* __restrict__ h2) {
    typedef V4 V;
    typedef float T;
    Pipe<5, 0, 3> P;
    const Col<float, W> c = make_col<float, W>(G);
    P.start(M, blockIdx.x, blockIdx.y, blockIdx.z, G.nz, c.z1);
    const View vw = make_view(G, P.x0, P.y0, threadIdx.x, threadIdx.y);
    Halo6<T> Hn, Hh;
#pragma unroll
    for (int f = 0; f < 6; ++f) { Hn.s[f] = G.s[f]; Hh.s[f] = T(1); }
    Hh.s[5] = T(-1);
    const HaloFac<T> fn = halo_fac(G, c, Hn), fh = halo_fac(G, c, Hh);
    GradRoll<T, V> g; g.init();
    ZAcc<V> m0, m1, m2; m0.init(); m1.init(); m2.init();
    for (int it = 0; it < P.niter; ++it) {
        const uint32_t slot = P.acquire(it);
        const int z = c.z0 - 1 + it;
        V n9[3][3], t9[3][3];
        load9s(P.sfield(slot, 0), vw, t9);
        halo_scale(G, Hh, fh, z, t9);
        if (z < 0) {
            V c9[3][3];
            load9(G, c, C, z, c9);
#pragma unroll
            for (int b = 0; b < 3; ++b)
#pragma unroll
                for (int a = 0; a < 3; ++a) t9[b][a] = t9[b][a] + (G.h[2] * grav) * mix01(rho_l, rho_g, c9[b][a]);
        }
#pragma unroll
        for (int b = 0; b < 3; ++b)
#pragma unroll
            for (int a = 0; a < 3; ++a) n9[b][a] = V{} + t9[b][a];
        load9s(P.sfield(slot, 1), vw, t9);
        halo_scale(G, Hn, fn, z, t9);
#pragma unroll
        for (int b = 0; b < 3; ++b)
#pragma unroll
            for (int a = 0; a < 3; ++a) n9[b][a] = n9[b][a] + t9[b][a];
        g.add(G, in_plane<T, true, false>(G, n9));
        load9s(P.sfield(slot, 2), vw, t9); const V s0 = m0.stepM(G, in_plane<T, false, false>(G, t9).mm);
        load9s(P.sfield(slot, 3), vw, t9); const V s1 = m1.stepM(G, in_plane<T, false, false>(G, t9).mm);
        load9s(P.sfield(slot, 4), vw, t9); const V s2 = m2.stepM(G, in_plane<T, false, false>(G, t9).mm);
        const int q = z - 1;
        if (q >= c.z0 && c.ok) {
            V gx, gy, gz; g.grad(G, gx, gy, gz);
            const size_t c0 = at(c, q);
            const V Cc = ldv<T, W>(C + c0);
            const V f = dt / mix01(rho_l, rho_g, Cc);
            const V u = ldv<T, W>(q0 + c0) - f * (gx + s0), v = ldv<T, W>(q1 + c0) - f * (gy + s1), w = ldv<T, W>(q2 + c0) - f * (gz + s2);
            stv(q0 + c0, u); stv(q1 + c0, v); stv(q2 + c0, w);
            if (h0) {
                stv(h0 + c0, T(0.5) * (ldv<T, W>(n0 + c0) + u)); stv(h1 + c0, T(0.5) * (ldv<T, W>(n1 + c0) + v));
                stv(h2 + c0, T(0.5) * (ldv<T, W>(n2 + c0) + w));
            }
        }
    }
}

// the paper's stage-3 right-hand side, Eq. 53 (pressure_rhs_paper_march)      (maps: C, u, v, w | -)
__global__ void __launch_bounds__(NT) pressure_rhs_paper_tma(const __grid_constant__ Maps M, const Geo<float> G, float rho_l, float rho_g,
                                                             float inv_dt, float* __restrict__ bout) {
    typedef V4 V;
    typedef float T;
    Pipe<4, 0, 3> P;
    const Col<float, W> c = make_col<float, W>(G);
    P.start(M, blockIdx.x, blockIdx.y, blockIdx.z, G.nz, c.z1);
    const View vw = make_view(G, P.x0, P.y0, threadIdx.x, threadIdx.y);
    ZAcc<V> acc; acc.init();
    GradRoll<T, V> gr; gr.init();
    V q0[3] = {}, q0n[3] = {};
    for (int it = 0; it < P.niter; ++it) {
        const uint32_t slot = P.acquire(it);
        V r9[3][3], n9[3][3];
        load9s(P.sfield(slot, 0), vw, r9);
#pragma unroll
        for (int b = 0; b < 3; ++b)
#pragma unroll
            for (int a = 0; a < 3; ++a) r9[b][a] = mix01(rho_l, rho_g, r9[b][a]);
        gr.add(G, in_plane<T, true, false>(G, r9));
        V part[3];
#pragma unroll
        for (int d = 0; d < 3; ++d) {
            load9s(P.sfield(slot, 1 + d), vw, n9);
            q0[d] = q0n[d]; q0n[d] = n9[1][1];
#pragma unroll
            for (int b = 0; b < 3; ++b)
#pragma unroll
                for (int a = 0; a < 3; ++a) n9[b][a] = n9[b][a] * r9[b][a];
            if (d == 2) part[d] = in_plane<T, false, false>(G, n9).mm;
            else { const InPlane<V> r = in_plane<T, true, false>(G, n9); part[d] = d == 0 ? r.dm : r.md; }
        }
        const V ms = G.M[0] * (part[0] + part[1]), dw = G.D[2][2] * part[2];
        const V div = acc.step(ms + dw, G.M[1] * (part[0] + part[1]), ms - dw);
        const int q = c.z0 - 2 + it;
        if (q >= c.z0 && c.ok) {
            V gx, gy, gz; gr.grad(G, gx, gy, gz);
            stv(bout + at(c, q), (-div + (q0[0] * gx + q0[1] * gy + q0[2] * gz)) * inv_dt);
        }
    }
}

}  // namespace ft
