// flow_march.cuh -- z-marching versions of the explicit stencil kernels of flow.cu (included by it, inside its
// namespace, after Geo / k_abs_pg).  Same filters and readings; different evaluation order:
//
// Every filter of the path is a tensor product of 1-D factors (Eqs. 9-11): D = [-1,0,1]/(2d),
// M = [1,4,1]/6, K = [-1,2,-1]/d^2.  A thread owns W consecutive x points of one (j) row of a z chunk and marches
// along z (W = 4 in fp32, 2 in fp64; 1 when nx is not a multiple of that or a pointer is not 16-byte aligned).  Per
// plane and field it loads its 3 rows once -- one 16-byte vector and the two x neighbours per row -- applies the x and
// y factors, and keeps the in-plane results of the last three planes in registers; the z factor is applied when the
// plane above has arrived.  That is 9 / W load instructions per field and point instead of 27.  All arithmetic is
// written once on the W-wide value pack Pk.  Halos are zero-derivative copies (clamped indices, reading
// C9-iv), the pressure halo of the projection carries the solver's factors (reading C10).
#pragma once

constexpr int MBX = 32, MBY = 4, MZC = 16;   // block = MBX x MBY threads (W MBX x MBY columns), MZC output planes per block

// ---- W-wide value pack: element-wise arithmetic --------------------------------------------------------------------
template <typename T, int W>
struct Pk {
    T v[W];
    __device__ __forceinline__ T& operator[](int e) { return v[e]; }
    __device__ __forceinline__ const T& operator[](int e) const { return v[e]; }
};
#define MGB_PK_BIN(OP)                                                                                                  \
    template <typename T, int W> __device__ __forceinline__ Pk<T, W> operator OP(const Pk<T, W>& a, const Pk<T, W>& b) { \
        Pk<T, W> r;                                                                                                     \
        _Pragma("unroll") for (int e = 0; e < W; ++e) r.v[e] = a.v[e] OP b.v[e];                                        \
        return r;                                                                                                       \
    }                                                                                                                   \
    template <typename T, int W> __device__ __forceinline__ Pk<T, W> operator OP(const Pk<T, W>& a, T b) {               \
        Pk<T, W> r;                                                                                                     \
        _Pragma("unroll") for (int e = 0; e < W; ++e) r.v[e] = a.v[e] OP b;                                             \
        return r;                                                                                                       \
    }                                                                                                                   \
    template <typename T, int W> __device__ __forceinline__ Pk<T, W> operator OP(T a, const Pk<T, W>& b) {               \
        Pk<T, W> r;                                                                                                     \
        _Pragma("unroll") for (int e = 0; e < W; ++e) r.v[e] = a OP b.v[e];                                             \
        return r;                                                                                                       \
    }
MGB_PK_BIN(+)
MGB_PK_BIN(-)
MGB_PK_BIN(*)
MGB_PK_BIN(/)
#undef MGB_PK_BIN
// fp32 packs of even width: two lanes per instruction on the packed fp32 pipe of sm_100a (add / sub / mul .f32x2)
typedef unsigned long long pk64;
__device__ __forceinline__ pk64 pk_join(float lo, float hi) { pk64 r; asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi)); return r; }
__device__ __forceinline__ void pk_split(pk64 v, float& lo, float& hi) { asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v)); }
__device__ __forceinline__ pk64 pk_add(pk64 a, pk64 b) { pk64 r; asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }
__device__ __forceinline__ pk64 pk_sub(pk64 a, pk64 b) { pk64 r; asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }
__device__ __forceinline__ pk64 pk_mul(pk64 a, pk64 b) { pk64 r; asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }
#define MGB_PK_F32(OP, FN)                                                                                              \
    template <int W> __device__ __forceinline__ Pk<float, W> operator OP(const Pk<float, W>& a, const Pk<float, W>& b) { \
        Pk<float, W> r;                                                                                                 \
        if constexpr (W % 2 == 0) {                                                                                     \
            _Pragma("unroll") for (int e = 0; e < W; e += 2)                                                            \
                pk_split(FN(pk_join(a.v[e], a.v[e + 1]), pk_join(b.v[e], b.v[e + 1])), r.v[e], r.v[e + 1]);             \
        } else {                                                                                                        \
            _Pragma("unroll") for (int e = 0; e < W; ++e) r.v[e] = a.v[e] OP b.v[e];                                    \
        }                                                                                                               \
        return r;                                                                                                       \
    }                                                                                                                   \
    template <int W> __device__ __forceinline__ Pk<float, W> operator OP(const Pk<float, W>& a, float b) {               \
        Pk<float, W> r;                                                                                                 \
        if constexpr (W % 2 == 0) {                                                                                     \
            const pk64 bb = pk_join(b, b);                                                                              \
            _Pragma("unroll") for (int e = 0; e < W; e += 2) pk_split(FN(pk_join(a.v[e], a.v[e + 1]), bb), r.v[e], r.v[e + 1]); \
        } else {                                                                                                        \
            _Pragma("unroll") for (int e = 0; e < W; ++e) r.v[e] = a.v[e] OP b;                                         \
        }                                                                                                               \
        return r;                                                                                                       \
    }                                                                                                                   \
    template <int W> __device__ __forceinline__ Pk<float, W> operator OP(float a, const Pk<float, W>& b) {               \
        Pk<float, W> r;                                                                                                 \
        if constexpr (W % 2 == 0) {                                                                                     \
            const pk64 aa = pk_join(a, a);                                                                              \
            _Pragma("unroll") for (int e = 0; e < W; e += 2) pk_split(FN(aa, pk_join(b.v[e], b.v[e + 1])), r.v[e], r.v[e + 1]); \
        } else {                                                                                                        \
            _Pragma("unroll") for (int e = 0; e < W; ++e) r.v[e] = a OP b.v[e];                                         \
        }                                                                                                               \
        return r;                                                                                                       \
    }
MGB_PK_F32(+, pk_add)
MGB_PK_F32(-, pk_sub)
MGB_PK_F32(*, pk_mul)
#undef MGB_PK_F32
__device__ __forceinline__ pk64 pk_fma(pk64 a, pk64 b, pk64 c) { pk64 r; asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c)); return r; }
// s * a + b with one rounding (what contraction gives scalar code; the packed operators above are opaque to it)
template <typename T, int W> __device__ __forceinline__ Pk<T, W> pfma(T s, const Pk<T, W>& a, const Pk<T, W>& b) {
    Pk<T, W> r;
    if constexpr (sizeof(T) == 4 && W % 2 == 0) {
        const pk64 ss = pk_join(s, s);
#pragma unroll
        for (int e = 0; e < W; e += 2) pk_split(pk_fma(ss, pk_join(a.v[e], a.v[e + 1]), pk_join(b.v[e], b.v[e + 1])), r.v[e], r.v[e + 1]);
    } else {
#pragma unroll
        for (int e = 0; e < W; ++e) r.v[e] = fma(s, a.v[e], b.v[e]);
    }
    return r;
}
template <typename T, int W> __device__ __forceinline__ Pk<T, W> pfma(const Pk<T, W>& s, const Pk<T, W>& a, const Pk<T, W>& b) {
    Pk<T, W> r;
    if constexpr (sizeof(T) == 4 && W % 2 == 0) {
#pragma unroll
        for (int e = 0; e < W; e += 2)
            pk_split(pk_fma(pk_join(s.v[e], s.v[e + 1]), pk_join(a.v[e], a.v[e + 1]), pk_join(b.v[e], b.v[e + 1])), r.v[e], r.v[e + 1]);
    } else {
#pragma unroll
        for (int e = 0; e < W; ++e) r.v[e] = fma(s.v[e], a.v[e], b.v[e]);
    }
    return r;
}

template <typename T, int W> __device__ __forceinline__ Pk<T, W> operator-(const Pk<T, W>& a) {
    Pk<T, W> r;
#pragma unroll
    for (int e = 0; e < W; ++e) r.v[e] = -a.v[e];
    return r;
}
template <typename T, int W> __device__ __forceinline__ Pk<T, W> pdiv(const Pk<T, W>& a, const Pk<T, W>& b) {      // fdiv lane by lane
    Pk<T, W> r;
#pragma unroll
    for (int e = 0; e < W; ++e) r.v[e] = fdiv(a.v[e], b.v[e]);
    return r;
}
template <typename T, int W> __device__ __forceinline__ Pk<T, W> splat(T a) {
    Pk<T, W> r;
#pragma unroll
    for (int e = 0; e < W; ++e) r.v[e] = a;
    return r;
}
template <typename T, int W> __device__ __forceinline__ Pk<T, W> pabs(const Pk<T, W>& a) {
    Pk<T, W> r;
#pragma unroll
    for (int e = 0; e < W; ++e) r.v[e] = fabs(a.v[e]);
    return r;
}
template <typename T, int W> __device__ __forceinline__ Pk<T, W> psqrt(const Pk<T, W>& a) {
    Pk<T, W> r;
#pragma unroll
    for (int e = 0; e < W; ++e) r.v[e] = sqrt(a.v[e]);
    return r;
}
template <typename T, int W> __device__ __forceinline__ Pk<T, W> pmin(const Pk<T, W>& a, const Pk<T, W>& b) {
    Pk<T, W> r;
#pragma unroll
    for (int e = 0; e < W; ++e) r.v[e] = tmin(a.v[e], b.v[e]);
    return r;
}
template <typename T, int W> __device__ __forceinline__ Pk<T, W> pmax(const Pk<T, W>& a, const Pk<T, W>& b) {
    Pk<T, W> r;
#pragma unroll
    for (int e = 0; e < W; ++e) r.v[e] = tmax(a.v[e], b.v[e]);
    return r;
}
template <typename T, int W> __device__ __forceinline__ Pk<T, W> pmin(T a, const Pk<T, W>& b) { return pmin(splat<T, W>(a), b); }
template <typename T, int W> __device__ __forceinline__ Pk<T, W> pmax(T a, const Pk<T, W>& b) { return pmax(splat<T, W>(a), b); }

// Material property of the one-fluid model, Eqs. 2 / 19: a = a_l C + a_g (1 - C) with C limited to [0, 1] first
// (reading C11: the paper does not clip, but an undershoot C = -0.003 -- which its scheme only makes "less likely", P:359 --
// gives rho < 0 at rho_g / rho_l = 1e-3, an indefinite pressure operator and a blow-up of the collapsing column)
template <typename T, int W> __device__ __forceinline__ Pk<T, W> mix01(T al, T ag, const Pk<T, W>& C) {
    const Pk<T, W> c = pmax(T(0), pmin(T(1), C));
    return al * c + ag * (T(1) - c);
}
template <typename T> __device__ __forceinline__ T mix01(T al, T ag, T C) {
    const T c = tmax(T(0), tmin(T(1), C));
    return al * c + ag * (T(1) - c);
}

// aligned vector load / store of a pack (W sizeof(T) = 4, 8, 16 or 32 bytes)
template <typename T, int W>
__device__ __forceinline__ Pk<T, W> ldv(const T* __restrict__ p) {
    Pk<T, W> r;
    if constexpr (W == 1) r.v[0] = *p;
    else if constexpr (sizeof(T) == 4 && W == 4) { const float4 t = *reinterpret_cast<const float4*>(p); r.v[0] = t.x; r.v[1] = t.y; r.v[2] = t.z; r.v[3] = t.w; }
    else if constexpr (sizeof(T) == 8 && W == 2) { const double2 t = *reinterpret_cast<const double2*>(p); r.v[0] = t.x; r.v[1] = t.y; }
    else {
#pragma unroll
        for (int e = 0; e < W; ++e) r.v[e] = p[e];
    }
    return r;
}
template <typename T, int W>
__device__ __forceinline__ void stv(T* __restrict__ p, const Pk<T, W>& a) {
    if constexpr (W == 1) *p = a.v[0];
    else if constexpr (sizeof(T) == 4 && W == 4) *reinterpret_cast<float4*>(p) = make_float4(a.v[0], a.v[1], a.v[2], a.v[3]);
    else if constexpr (sizeof(T) == 8 && W == 2) *reinterpret_cast<double2*>(p) = make_double2(a.v[0], a.v[1]);
    else {
#pragma unroll
        for (int e = 0; e < W; ++e) p[e] = a.v[e];
    }
}

template <typename T, int W>
struct Col {           // z-invariant addressing of a thread's W points
    int i, j;          // first x index (a multiple of W), row
    int il, ir;        // clamped x neighbours of the pack's ends
    size_t row[3];     // nx * clamped j - 1, j, j + 1
    size_t nxy;
    int z0, z1;        // output planes [z0, z1)
    bool ok;
};

template <typename T, int W>
__device__ __forceinline__ Col<T, W> make_col(const Geo<T>& G) {
    Col<T, W> c;
    c.i = W * (blockIdx.x * MBX + threadIdx.x); c.j = blockIdx.y * MBY + threadIdx.y;
    c.ok = c.i < G.nx && c.j < G.ny;                      // nx is a multiple of W
    const int j = min(c.j, G.ny - 1);
    c.i = min(c.i, G.nx - W);
    c.il = max(c.i - 1, 0); c.ir = min(c.i + W, G.nx - 1);
    c.row[0] = (size_t)G.nx * max(j - 1, 0); c.row[1] = (size_t)G.nx * j; c.row[2] = (size_t)G.nx * min(j + 1, G.ny - 1);
    c.nxy = (size_t)G.nx * G.ny;
    c.z0 = blockIdx.z * MZC; c.z1 = min(c.z0 + MZC, G.nz);
    return c;
}

template <typename T, int W>
dim3 march_grid(const Geo<T>& G) { return dim3((G.nx + W * MBX - 1) / (W * MBX), (G.ny + MBY - 1) / MBY, (G.nz + MZC - 1) / MZC); }

// the 3 x 3 in-plane neighbourhood v[b][a] (b along y, a along x) of plane z (clamped) for the thread's W points
template <typename T, int W>
__device__ __forceinline__ void load9(const Geo<T>& G, const Col<T, W>& c, const T* __restrict__ f, int z, Pk<T, W> (&v)[3][3]) {
    const T* p = f + c.nxy * (size_t)min(max(z, 0), G.nz - 1);
#pragma unroll
    for (int b = 0; b < 3; ++b) {
        const T* r = p + c.row[b];
        const T l = r[c.il], rr = r[c.ir];
        v[b][1] = ldv<T, W>(r + c.i);
        v[b][0][0] = l; v[b][2][W - 1] = rr;
#pragma unroll
        for (int e = 1; e < W; ++e) { v[b][0][e] = v[b][1][e - 1]; v[b][2][e - 1] = v[b][1][e]; }
    }
}
// index of the thread's first point in plane q
template <typename T, int W>
__device__ __forceinline__ size_t at(const Col<T, W>& c, int q) { return c.nxy * q + c.row[1] + c.i; }

// Halo factors of one field, ghost = s * mirror (the clamped loads of load9 deliver the mirror value).  Used for
// the pressure in the projection (the solver's factors, reading C10) and for velocity components at free-slip walls
// (the wall-normal component is odd about the wall, s = -1; everything else is copied, s = +1).
template <typename T> struct Halo6 { T s[6]; };
template <typename T>
struct HaloFac { T fl, fr, fy[3]; };      // z-invariant factors of a thread's 3 x 3 neighbourhood
template <typename T, int W>
__device__ __forceinline__ HaloFac<T> halo_fac(const Geo<T>& G, const Col<T, W>& c, const Halo6<T>& H) {
    HaloFac<T> f;
    // only the outermost lane of a pack's left / right neighbour can be a ghost
    f.fl = c.i > 0 ? T(1) : H.s[0]; f.fr = c.i + W < G.nx ? T(1) : H.s[1];
    f.fy[0] = c.j > 0 ? T(1) : H.s[2]; f.fy[1] = T(1); f.fy[2] = c.j < G.ny - 1 ? T(1) : H.s[3];
    return f;
}
template <typename T, int W>
__device__ __forceinline__ void halo_scale(const Geo<T>& G, const Halo6<T>& H, const HaloFac<T>& f, int z, Pk<T, W> (&n9)[3][3]) {
    const T fz = z < 0 ? H.s[4] : (z >= G.nz ? H.s[5] : T(1));
#pragma unroll
    for (int b = 0; b < 3; ++b) {
        n9[b][0][0] *= f.fl; n9[b][2][W - 1] *= f.fr;
#pragma unroll
        for (int a = 0; a < 3; ++a) n9[b][a] = n9[b][a] * (fz * f.fy[b]);
    }
}

// in-plane tensor-product filters of a 3 x 3 neighbourhood
template <typename V>
struct InPlane {
    V mm, dm, md, km, mk;    // Mx My, Dx My, Mx Dy, Kx My, Mx Ky
};
// M = [1, 4, 1] / 6, D = [-1, 0, 1] / (2 d), K = [-1, 2, -1] / d^2: the row and column combinations are formed with the integer
// weights (one fused multiply-add each) and the constant factors applied once per result -- 17 instead of 23 instructions per point
// for (mm, dm, md); the kernels that use this are bound by instruction issue (profiles/r02_ncu_flow.md)
template <typename T, bool NEED_D, bool NEED_K, typename V>
__device__ __forceinline__ InPlane<V> in_plane(const Geo<T>& G, const V (&v)[3][3]) {
    const T m = G.M[0];                                   // 1/6
    V sm[3], sd[3], sk[3];                                // x combinations of the three rows, unscaled: 6 Mx, 2 d Dx, -d^2 Kx
#pragma unroll
    for (int b = 0; b < 3; ++b) {
        const V e = v[b][0] + v[b][2];
        sm[b] = pfma(T(4), v[b][1], e);
        if (NEED_D) sd[b] = v[b][2] - v[b][0];
        if (NEED_K) sk[b] = pfma(T(-2), v[b][1], e);
    }
    InPlane<V> r;
    const V smo = sm[0] + sm[2];
    r.mm = (m * m) * pfma(T(4), sm[1], smo);
    r.dm = r.md = r.km = r.mk = V{};
    if (NEED_D) { r.dm = (m * G.D[0][2]) * pfma(T(4), sd[1], sd[0] + sd[2]); r.md = (m * G.D[1][2]) * (sm[2] - sm[0]); }
    if (NEED_K) { r.km = (m * G.K[0][0]) * pfma(T(4), sk[1], sk[0] + sk[2]); r.mk = (m * G.K[1][0]) * pfma(T(-2), sm[1], smo); }
    return r;
}

// z factor applied on arrival: plane z of an in-plane result contributes `up` to the output of plane z - 1, `mid` to plane z
// and `dn` to plane z + 1; step() takes the three and returns the finished output of plane z - 1.  Two running sums per
// filtered quantity instead of three stored planes (and no register shuffling per plane).
template <typename V>
struct ZAcc {
    V A, B;       // partial outputs of planes z - 1 and z before plane z has arrived
    __device__ __forceinline__ void init() { A = V{}; B = V{}; }
    __device__ __forceinline__ V step(const V& up, const V& mid, const V& dn) { const V done = A + up; A = B + mid; B = dn; return done; }
    template <typename T> __device__ __forceinline__ V stepM(const Geo<T>& G, const V& v) { const V t = G.M[0] * v; const V done = A + t; A = pfma(T(4), t, B); B = t; return done; }   // Mz = [1, 4, 1] / 6
    template <typename T> __device__ __forceinline__ V stepK(const Geo<T>& G, const V& v) { const V t = G.K[2][0] * v; const V done = A + t; A = pfma(T(-2), t, B); B = t; return done; }   // Kz = [-1, 2, -1] / d^2
    template <typename T> __device__ __forceinline__ V stepD(const Geo<T>& G, const V& v) { const V t = G.D[2][2] * v; const V done = A + t; A = B; B = -t; return done; }   // Dz
};
template <typename V> __device__ __forceinline__ void push(V (&a)[3], const V& v) { a[0] = a[1]; a[1] = a[2]; a[2] = v; }

// b = -(1/dt) (f(u; w_x) + f(v; w_y) + f(w; w_z))  (reading C10; Eq. 53 structure)
// BC: the three fields carry the halo factors Hu, Hv, Hw (free-slip walls); otherwise their halos are copies
template <typename T, int W, bool BC = false>
__global__ void __launch_bounds__(MBX* MBY) pressure_rhs_march(const Geo<T> G, const T* __restrict__ u, const T* __restrict__ v,
                                                             const T* __restrict__ w, T inv_dt, T* __restrict__ bout,
                                                             const Halo6<T> Hu = {}, const Halo6<T> Hv = {}, const Halo6<T> Hw = {}) {
    typedef Pk<T, W> V;
    const Col<T, W> c = make_col<T, W>(G);
    HaloFac<T> fu = {}, fv = {}, fw = {};
    if (BC) { fu = halo_fac(G, c, Hu); fv = halo_fac(G, c, Hv); fw = halo_fac(G, c, Hw); }
    ZAcc<V> acc; acc.init();       // Mz (Dx My u + Mx Dy v) + Dz (Mx My w)
    for (int z = c.z0 - 1; z <= c.z1; ++z) {
        V n9[3][3];
        load9(G, c, u, z, n9); if (BC) halo_scale(G, Hu, fu, z, n9); const V du = in_plane<T, true, false>(G, n9).dm;
        load9(G, c, v, z, n9); if (BC) halo_scale(G, Hv, fv, z, n9); const V dv = in_plane<T, true, false>(G, n9).md;
        load9(G, c, w, z, n9); if (BC) halo_scale(G, Hw, fw, z, n9); const V mw = in_plane<T, false, false>(G, n9).mm;
        const V ms = G.M[0] * (du + dv), dw = G.D[2][2] * mw;
        const V div = acc.step(ms + dw, G.M[1] * (du + dv), ms - dw);
        const int q = z - 1;
        if (q >= c.z0 && c.ok) stv(bout + at(c, q), -div * inv_dt);
    }
}

// gradient by the FE first-derivative filters from rolling in-plane results
template <typename T, typename V>
struct GradRoll {
    ZAcc<V> ax, ay, az;
    V gx, gy, gz;       // gradient at plane z - 1 after add() of plane z
    __device__ __forceinline__ void init() { ax.init(); ay.init(); az.init(); }
    __device__ __forceinline__ void add(const Geo<T>& G, const InPlane<V>& r) { gx = ax.stepM(G, r.dm); gy = ay.stepM(G, r.md); gz = az.stepD(G, r.mm); }
    __device__ __forceinline__ void grad(const Geo<T>&, V& ox, V& oy, V& oz) const { ox = gx; oy = gy; oz = gz; }
};

// q <- q - dt k f(p; w_x|y|z) (Eq. 54); halo of p = s * mirror with the solver's factors
template <typename T, int W>
__global__ void __launch_bounds__(MBX* MBY) project_march(const Geo<T> G, const T* __restrict__ p, const T* __restrict__ kc, T dt,
                                                        T* __restrict__ u, T* __restrict__ v, T* __restrict__ w) {
    typedef Pk<T, W> V;
    const Col<T, W> c = make_col<T, W>(G);
    Halo6<T> H;
#pragma unroll
    for (int f = 0; f < 6; ++f) H.s[f] = G.s[f];
    const HaloFac<T> hf = halo_fac(G, c, H);
    GradRoll<T, V> g; g.init();
    for (int z = c.z0 - 1; z <= c.z1; ++z) {
        V n9[3][3];
        load9(G, c, p, z, n9);
        halo_scale(G, H, hf, z, n9);
        g.add(G, in_plane<T, true, false>(G, n9));
        const int q = z - 1;
        if (q >= c.z0 && c.ok) {
            V gx, gy, gz; g.grad(G, gx, gy, gz);
            const size_t c0 = at(c, q);
            const V f = dt * ldv<T, W>(kc + c0);
            stv(u + c0, ldv<T, W>(u + c0) - f * gx); stv(v + c0, ldv<T, W>(v + c0) - f * gy); stv(w + c0, ldv<T, W>(w + c0) - f * gz);
        }
    }
}

// Forcing terms of Eq. 18 applied to the predicted velocity:
//   q~_d <- q~_d - (dt / rho) ( f(p_hs + p~_nh; w_d) + f(F_d; w_m) ),   F = -(s + s_t)  (hydrostatic_rhs' force field),
// and optionally q_half' = (q_n + q~) / 2 (Eq. 46).  Halos: p_hs zero derivative on the sides, zero value on the top face,
// and below the bottom plane mirror + hz g rho(mirror) (dp_hs/dz = -rho g); p~_nh the solver's factors G.s; F copies.
// Either pressure and F may be absent (NULL).
template <typename T, int W>
__global__ void __launch_bounds__(MBX* MBY) mom_forcing_march(const Geo<T> G, const T* __restrict__ C, const T* __restrict__ phs,
                                                            const T* __restrict__ pnh, const T* __restrict__ F0,
                                                            const T* __restrict__ F1, const T* __restrict__ F2, T rho_l, T rho_g,
                                                            T grav, T dt, T* __restrict__ q0, T* __restrict__ q1, T* __restrict__ q2,
                                                            const T* __restrict__ n0, const T* __restrict__ n1,
                                                            const T* __restrict__ n2, T* __restrict__ h0, T* __restrict__ h1,
                                                            T* __restrict__ h2) {
    typedef Pk<T, W> V;
    const Col<T, W> c = make_col<T, W>(G);
    Halo6<T> Hn, Hh;
#pragma unroll
    for (int f = 0; f < 6; ++f) { Hn.s[f] = G.s[f]; Hh.s[f] = T(1); }
    Hh.s[5] = T(-1);
    const HaloFac<T> fn = halo_fac(G, c, Hn), fh = halo_fac(G, c, Hh);
    GradRoll<T, V> g; g.init();
    ZAcc<V> m0, m1, m2; m0.init(); m1.init(); m2.init();
    const bool have_p = phs != nullptr || pnh != nullptr, have_f = F0 != nullptr;
    for (int z = c.z0 - 1; z <= c.z1; ++z) {
        V n9[3][3], t9[3][3];
        if (have_p) {
#pragma unroll
            for (int b = 0; b < 3; ++b)
#pragma unroll
                for (int a = 0; a < 3; ++a) n9[b][a] = V{};
            if (phs) {
                load9(G, c, phs, z, t9);
                halo_scale(G, Hh, fh, z, t9);
                if (z < 0) {                                   // ghost plane below the bottom: + hz g rho(mirror)
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
                    for (int a = 0; a < 3; ++a) n9[b][a] = n9[b][a] + t9[b][a];
            }
            if (pnh) {
                load9(G, c, pnh, z, t9);
                halo_scale(G, Hn, fn, z, t9);
#pragma unroll
                for (int b = 0; b < 3; ++b)
#pragma unroll
                    for (int a = 0; a < 3; ++a) n9[b][a] = n9[b][a] + t9[b][a];
            }
            g.add(G, in_plane<T, true, false>(G, n9));
        }
        V s0 = {}, s1 = {}, s2 = {};
        if (have_f) {
            load9(G, c, F0, z, t9); s0 = m0.stepM(G, in_plane<T, false, false>(G, t9).mm);
            load9(G, c, F1, z, t9); s1 = m1.stepM(G, in_plane<T, false, false>(G, t9).mm);
            load9(G, c, F2, z, t9); s2 = m2.stepM(G, in_plane<T, false, false>(G, t9).mm);
        }
        const int q = z - 1;
        if (q >= c.z0 && c.ok) {
            V gx = {}, gy = {}, gz = {};
            if (have_p) g.grad(G, gx, gy, gz);
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

// steps 1-2 of reading C9: adv = u psi_x + v psi_y + w psi_z
template <typename T, int W, bool BC = false>
__global__ void __launch_bounds__(MBX* MBY) advection_march(const Geo<T> G, const T* __restrict__ psi, const T* __restrict__ u,
                                                          const T* __restrict__ v, const T* __restrict__ w, T* __restrict__ adv,
                                                          const Halo6<T> H = {}) {
    typedef Pk<T, W> V;
    const Col<T, W> c = make_col<T, W>(G);
    HaloFac<T> hf = {};
    if (BC) hf = halo_fac(G, c, H);
    GradRoll<T, V> g; g.init();
    for (int z = c.z0 - 1; z <= c.z1; ++z) {
        V n9[3][3];
        load9(G, c, psi, z, n9);
        if (BC) halo_scale(G, H, hf, z, n9);
        g.add(G, in_plane<T, true, false>(G, n9));
        const int q = z - 1;
        if (q >= c.z0 && c.ok) {
            V gx, gy, gz; g.grad(G, gx, gy, gz);
            const size_t c0 = at(c, q);
            stv(adv + c0, ldv<T, W>(u + c0) * gx + ldv<T, W>(v + c0) * gy + ldv<T, W>(w + c0) * gz);
        }
    }
}

// The advection terms of the three momentum components in one pass (steps 1-2 for psi = u, v, w): the advecting velocity IS
// (u, v, w), so each field is read once as a stencil and its centre value serves all three products -- 24 B/point instead of
// 3 x 20.  The centre pack of plane z - 1 is kept from the previous iteration of the march.
template <typename T, int W, bool BC = false>
__global__ void __launch_bounds__(MBX* MBY) advection3_march(const Geo<T> G, const T* __restrict__ u, const T* __restrict__ v,
                                                           const T* __restrict__ w, T* __restrict__ au, T* __restrict__ av,
                                                           T* __restrict__ aw, const Halo6<T> Hu = {}, const Halo6<T> Hv = {},
                                                           const Halo6<T> Hw = {}) {
    typedef Pk<T, W> V;
    const Col<T, W> c = make_col<T, W>(G);
    HaloFac<T> hu = {}, hv = {}, hw = {};
    if (BC) { hu = halo_fac(G, c, Hu); hv = halo_fac(G, c, Hv); hw = halo_fac(G, c, Hw); }
    GradRoll<T, V> gu, gv, gw; gu.init(); gv.init(); gw.init();
    V cu = {}, cv = {}, cw = {};                                  // centre values of plane z - 1
    for (int z = c.z0 - 1; z <= c.z1; ++z) {
        V n9[3][3];
        load9(G, c, u, z, n9);
        if (BC) halo_scale(G, Hu, hu, z, n9);
        gu.add(G, in_plane<T, true, false>(G, n9));
        const V nu = n9[1][1];
        load9(G, c, v, z, n9);
        if (BC) halo_scale(G, Hv, hv, z, n9);
        gv.add(G, in_plane<T, true, false>(G, n9));
        const V nv = n9[1][1];
        load9(G, c, w, z, n9);
        if (BC) halo_scale(G, Hw, hw, z, n9);
        gw.add(G, in_plane<T, true, false>(G, n9));
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

// Eqs. 26/27 on a pack (k_abs_pg of flow.cu lane by lane)
template <typename T, int W>
__device__ __forceinline__ Pk<T, W> k_abs_pk(const Geo<T>& G, const Pk<T, W>& a, const Pk<T, W>& px, const Pk<T, W>& py, const Pk<T, W>& pz) {
    Pk<T, W> r;
#pragma unroll
    for (int e = 0; e < W; ++e) r[e] = k_abs_pg(G, a[e], px[e], py[e], pz[e]);
    return r;
}

// momentum: k_c = rho min{k_max, k_abs(c)} + mu (Eqs. 30-32; k_square of the lost Eq. 28 omitted);
// k_abs from the gradient of the component and the mixed-mass residual a = 2 (Mx My Mz - E) adv (Eq. 29)
template <typename T, int W, bool BC = false>
__global__ void __launch_bounds__(MBX* MBY) mom_coeff_march(const Geo<T> G, const T* __restrict__ C, const T* __restrict__ comp,
                                                          const T* __restrict__ u, const T* __restrict__ v, const T* __restrict__ w,
                                                          const T* __restrict__ adv, T rho_l, T rho_g, T mu_l, T mu_g,
                                                          T* __restrict__ kc, const Halo6<T> H = {}) {
    typedef Pk<T, W> V;
    const Col<T, W> c = make_col<T, W>(G);
    HaloFac<T> hf = {};
    if (BC) hf = halo_fac(G, c, H);
    GradRoll<T, V> g; g.init();
    ZAcc<V> am; am.init();               // Mz of Mx My adv
    V a0 = {}, a0n = {};                 // adv at the centre of planes q, q + 1
    for (int z = c.z0 - 1; z <= c.z1; ++z) {
        V n9[3][3];
        load9(G, c, comp, z, n9);
        if (BC) halo_scale(G, H, hf, z, n9);
        g.add(G, in_plane<T, true, false>(G, n9));
        load9(G, c, adv, z, n9);
        const V madv = am.stepM(G, in_plane<T, false, false>(G, n9).mm);
        a0 = a0n; a0n = n9[1][1];
        const int q = z - 1;
        if (q >= c.z0 && c.ok) {
            V px, py, pz; g.grad(G, px, py, pz);
            const V a = T(2) * (madv - a0);
            const size_t c0 = at(c, q);
            const V Cc = ldv<T, W>(C + c0);
            const V rho = mix01(rho_l, rho_g, Cc);
            const V mu = mix01(mu_l, mu_g, Cc);
            const V kmax = G.h[0] * pabs(ldv<T, W>(u + c0)) + G.h[1] * pabs(ldv<T, W>(v + c0)) + G.h[2] * pabs(ldv<T, W>(w + c0));   // Eq. 30
            stv(kc + c0, rho * pmin(kmax, k_abs_pk(G, a, px, py, pz)) + mu);
        }
    }
}

// rolling in-plane parts of a filter  W = F_xy (x) F_z  applied to three fields (f, k, k f), combined as Eq. 12-13:
//   sum_j (-W_ij) 1/2 (k_i + k_j)(f_i - f_j) = 1/2 (W(k f) + k W(f) - f W(k))      [sum_j W_ij = 0]
template <typename V>
struct Diff3 {
    ZAcc<V> f, k, z;
    __device__ __forceinline__ void init() { f.init(); k.init(); z.init(); }
};

// s = rho adv + f^lap(c, k_c; w_lap) (Eq. 18 without pressure / source terms), q~ = q_n - dt s / rho (Eq. 45, sigma = 0),
// q_half' = (q_n + q~)/2 (Eq. 46).  w_lap = (Kx My + Mx Ky) Mz + Mx My Kz.
template <typename T, int W, bool BC = false>
__global__ void __launch_bounds__(MBX* MBY) mom_update_march(const Geo<T> G, const T* __restrict__ C, const T* __restrict__ comp,
                                                           const T* __restrict__ kc, const T* __restrict__ adv,
                                                           const T* __restrict__ qn, T rho_l, T rho_g, T dt, T* __restrict__ qt,
                                                           T* __restrict__ qhn, const Halo6<T> H = {}) {
    typedef Pk<T, W> V;
    const Col<T, W> c = make_col<T, W>(G);
    HaloFac<T> hf = {};
    if (BC) hf = halo_fac(G, c, H);
    Diff3<V> L; L.init();                        // w_lap of x, k, k x: Mz of the in-plane (Kx My + Mx Ky) + Kz of the in-plane Mx My
    V x0 = {}, x0n = {}, k0 = {}, k0n = {};
    for (int z = c.z0 - 1; z <= c.z1; ++z) {
        V nx9[3][3], nk9[3][3], nz9[3][3];
        load9(G, c, comp, z, nx9);
        if (BC) halo_scale(G, H, hf, z, nx9);    // the component's halo; k_c keeps its copy halo, so ghost(k c) = s k c (mirror)
        load9(G, c, kc, z, nk9);
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
            const V Cc = ldv<T, W>(C + c0);
            const V rho = mix01(rho_l, rho_g, Cc);
            const V s = rho * ldv<T, W>(adv + c0) + diff;
            const V qv = ldv<T, W>(qn + c0);
            const V t = qv - dt * s / rho;
            stv(qt + c0, t);
            if (qhn) stv(qhn + c0, T(0.5) * (qv + t));
        }
    }
}

// steps 3-10 of reading C9: directional diffusion coefficients k^x, k^y, k^z of the compressive scheme
// Eq. 34: minimum of the three products of consecutive differences of five values in a line
template <typename V>
__device__ __forceinline__ V det5(const V& a0, const V& a1, const V& a2, const V& a3, const V& a4) {
    const V d0 = a1 - a0, d1 = a2 - a1, d2 = a3 - a2, d3 = a4 - a3;
    return pmin(pmin(d0 * d1, d1 * d2), d2 * d3);
}
__device__ __forceinline__ int reflect(int a, int n) { return a < 0 ? -1 - a : (a >= n ? 2 * n - 1 - a : a); }   // copy halo, any depth

// DET5: the oscillation detectors S^x, S^y, S^z are the 5-point ones of Eq. 34 instead of Eq. 33
template <typename T, int W, bool DET5 = false>
__global__ void __launch_bounds__(MBX* MBY) vof_coeff_march(const Geo<T> G, const T* __restrict__ C, const T* __restrict__ u,
                                                          const T* __restrict__ v, const T* __restrict__ w,
                                                          const T* __restrict__ adv, T k_min, T k_max, T* __restrict__ kx,
                                                          T* __restrict__ ky, T* __restrict__ kz) {
    typedef Pk<T, W> V;
    const Col<T, W> c = make_col<T, W>(G);
    const T Kp = T(300), Km = T(300);        // K+, K- 
    const T beta = T(0.1), eps_x = T(1e-4);  // Eq. 36
    const T Kcal = T(3);                     // Eq. 39
    const T ih[3] = {T(1) / G.h[0], T(1) / G.h[1], T(1) / G.h[2]};
    GradRoll<T, V> g; g.init();
    ZAcc<V> am; am.init();                                        // Mz of Mx My adv
    V a0 = {}, a0n = {};                                          // adv at the centre of planes q, q + 1
    V Cc[3] = {};                                                 // C at the centre of planes q - 1, q, q + 1
    V Sx = {}, Sxn = {}, Sy = {}, Syn = {};                       // Eq. 33 in-plane products of planes q, q + 1
    // DET5: C at the centre of plane q - 2 (Cm2) and q + 2 (Cp2); x / y neighbours at distance 2 by reflected indices
    V Cm2 = {}, Cp2 = {};
    const int il2 = reflect(c.i - 2, G.nx), ir2 = reflect(c.i + W + 1, G.nx);
    const size_t rowm2 = (size_t)G.nx * reflect(min(c.j, G.ny - 1) - 2, G.ny), rowp2 = (size_t)G.nx * reflect(min(c.j, G.ny - 1) + 2, G.ny);
    if (DET5) Cc[2] = ldv<T, W>(C + c.nxy * (size_t)reflect(c.z0 - 2, G.nz) + c.row[1] + c.i);    // plane z0 - 2, pushed down to Cc[0] by the time plane z0 is finalised
    for (int z = c.z0 - 1; z <= c.z1; ++z) {
        V n9[3][3];
        load9(G, c, C, z, n9);
        g.add(G, in_plane<T, true, false>(G, n9));
        if (DET5) Cm2 = Cc[0];                                    // before the push Cc holds planes (z - 3, z - 2, z - 1): plane q - 2
        push(Cc, n9[1][1]);
        Sx = Sxn; Sy = Syn;
        if (DET5) {
            const T* pl = C + c.nxy * (size_t)min(max(z, 0), G.nz - 1);
            // x: the W + 4 values l2, l1, own 0 .. W - 1, r1, r2 of the centre row
            T line[W + 4];
            line[0] = pl[c.row[1] + il2]; line[1] = n9[1][0][0]; line[W + 2] = n9[1][2][W - 1]; line[W + 3] = pl[c.row[1] + ir2];
#pragma unroll
            for (int e = 0; e < W; ++e) line[e + 2] = n9[1][1][e];
#pragma unroll
            for (int e = 0; e < W; ++e) {
                const T d0 = line[e + 1] - line[e], d1 = line[e + 2] - line[e + 1], d2 = line[e + 3] - line[e + 2], d3 = line[e + 4] - line[e + 3];
                Sxn[e] = tmin(tmin(d0 * d1, d1 * d2), d2 * d3);
            }
            Syn = det5(ldv<T, W>(pl + rowm2 + c.i), n9[0][1], n9[1][1], n9[2][1], ldv<T, W>(pl + rowp2 + c.i));
            Cp2 = ldv<T, W>(C + c.nxy * (size_t)reflect(z + 1, G.nz) + c.row[1] + c.i);        // plane q + 2
        } else {
            Sxn = (n9[1][1] - n9[1][0]) * (n9[1][2] - n9[1][1]);
            Syn = (n9[1][1] - n9[0][1]) * (n9[2][1] - n9[1][1]);
        }
        load9(G, c, adv, z, n9);
        const V madv = am.stepM(G, in_plane<T, false, false>(G, n9).mm);
        a0 = a0n; a0n = n9[1][1];
        const int q = z - 1;
        if (q >= c.z0 && c.ok) {
            V Cx, Cy, Cz; g.grad(G, Cx, Cy, Cz);
            const V a = T(2) * (madv - a0);                                      // step 3, Eq. 29
            const V kabs = k_abs_pk(G, a, Cx, Cy, Cz);                           // step 4, Eq. 27
            const V C0 = Cc[1];
            V S[3] = {Sx, Sy, DET5 ? det5(Cm2, Cc[0], C0, Cc[2], Cp2) : (C0 - Cc[0]) * (Cc[2] - C0)};   // step 5, Eq. 33 / Eq. 34
#pragma unroll
            for (int e = 0; e < W; ++e)
                if (C0[e] > T(0.95) || C0[e] < T(0.05)) S[0][e] = S[1][e] = S[2][e] = T(-1);   // override
            const size_t c0 = at(c, q);
            const V uu = ldv<T, W>(u + c0), vv = ldv<T, W>(v + c0), ww = ldv<T, W>(w + c0);
            const V g2 = Cx * Cx + Cy * Cy + Cz * Cz;
            const V gq = pdiv(uu * Cx + vv * Cy + ww * Cz, eps_x + g2);           // step 7, Eq. 37
            const V us = gq * Cx, vs = gq * Cy, ws = gq * Cz;
            const V kneg = pdiv(-beta * (uu * uu + vv * vv + ww * ww),           // step 8, Eq. 36
                                eps_x + g2 * (pabs(us) + pabs(vs) + pabs(ws)) * T(1.0 / 3.0));
            T* const out[3] = {kx, ky, kz};
#pragma unroll
            for (int d = 0; d < 3; ++d) {
                const V wp = -pmax(T(-1), pmin(T(0), Kp * S[d]));                // step 6, Eq. 35
                const V wm = pmin(T(1), pmax(T(0), Km * S[d]));
                const V kk = wp * (Kcal * kabs) + wm * (kneg * ih[d]);           // steps 9, Eqs. 38-40
                stv(out[d] + c0, pmax(-k_min, pmin(k_max, kk)));                 // step 10, Eq. 41
            }
        }
    }
}

// steps 11-12: sC = adv + sum_d diff_d, diff_d = sum_{j != i} (-W^dd_ij) 1/2 (k^d_i + k^d_j)(C_i - C_j) (Eq. 12 collapsed,
// P:146-151) evaluated as 1/2 (W^dd(k^d C) + k^d W^dd(C) - C W^dd(k^d)), W^xx = Kx My Mz, W^yy = Mx Ky Mz, W^zz = Mx My Kz;
// Cnew = C - dt sC (Eq. 55)
template <typename T, int W>
__global__ void __launch_bounds__(MBX* MBY) vof_diffusion_march(const Geo<T> G, const T* __restrict__ C, const T* __restrict__ adv,
                                                              const T* __restrict__ kx, const T* __restrict__ ky,
                                                              const T* __restrict__ kz, T dt, T* __restrict__ sC,
                                                              T* __restrict__ Cnew) {
    typedef Pk<T, W> V;
    const Col<T, W> c = make_col<T, W>(G);
    Diff3<V> dx, dy, dz; dx.init(); dy.init(); dz.init();     // in-plane Kx My / Mx Ky / Mx My of (C, k^d, k^d C)
    V C0 = {}, C0n = {}, k0[3] = {}, k0n[3] = {};
    for (int z = c.z0 - 1; z <= c.z1; ++z) {
        V nc[3][3], nk[3][3], nz9[3][3];
        load9(G, c, C, z, nc);
        const InPlane<V> rc = in_plane<T, false, true>(G, nc);
        C0 = C0n; C0n = nc[1][1];
        const T* const kd[3] = {kx, ky, kz};
        V pk[3], pz[3];
#pragma unroll
        for (int d = 0; d < 3; ++d) {
            load9(G, c, kd[d], z, nk);
#pragma unroll
            for (int b = 0; b < 3; ++b)
#pragma unroll
                for (int a = 0; a < 3; ++a) nz9[b][a] = nk[b][a] * nc[b][a];
            k0[d] = k0n[d]; k0n[d] = nk[1][1];
            if (d == 2) {
                pk[d] = in_plane<T, false, false>(G, nk).mm; pz[d] = in_plane<T, false, false>(G, nz9).mm;
            } else {
                const InPlane<V> rk = in_plane<T, false, true>(G, nk), rz = in_plane<T, false, true>(G, nz9);
                pk[d] = d == 0 ? rk.km : rk.mk; pz[d] = d == 0 ? rz.km : rz.mk;
            }
        }
        const V xf = dx.f.stepM(G, rc.km), xk = dx.k.stepM(G, pk[0]), xz = dx.z.stepM(G, pz[0]);
        const V yf = dy.f.stepM(G, rc.mk), yk = dy.k.stepM(G, pk[1]), yz = dy.z.stepM(G, pz[1]);
        const V zf = dz.f.stepK(G, rc.mm), zk = dz.k.stepK(G, pk[2]), zz = dz.z.stepK(G, pz[2]);
        const int q = z - 1;
        if (q >= c.z0 && c.ok) {
            const V ddx = T(0.5) * (xz + k0[0] * xf - C0 * xk);
            const V ddy = T(0.5) * (yz + k0[1] * yf - C0 * yk);
            const V ddz = T(0.5) * (zz + k0[2] * zf - C0 * zk);
            const size_t c0 = at(c, q);
            const V s = ldv<T, W>(adv + c0) + ddx + ddy + ddz;
            if (sC) stv(sC + c0, s);
            if (Cnew) stv(Cnew + c0, C0 - dt * s);
        }
    }
}

// The paper's own stage-3 right-hand side, Eqs. 52-53: density on the right, constant-coefficient
// Laplacian:  b = -(1/dt) sum_d f(rho q_d; w_d) + (1/dt) sum_d q_d f(rho; w_d),  rho = rho_l C + rho_g (1 - C)  (Eq. 2).
template <typename T, int W>
__global__ void __launch_bounds__(MBX* MBY) pressure_rhs_paper_march(const Geo<T> G, const T* __restrict__ C, const T* __restrict__ u,
                                                                   const T* __restrict__ v, const T* __restrict__ w, T rho_l, T rho_g,
                                                                   T inv_dt, T* __restrict__ bout) {
    typedef Pk<T, W> V;
    const Col<T, W> c = make_col<T, W>(G);
    ZAcc<V> acc; acc.init();                                         // Mz (Dx My (rho u) + Mx Dy (rho v)) + Dz (Mx My (rho w))
    GradRoll<T, V> gr; gr.init();                                    // in-plane parts of grad rho
    V q0[3] = {}, q0n[3] = {};                                       // u, v, w at the centre of planes q, q + 1
    for (int z = c.z0 - 1; z <= c.z1; ++z) {
        V r9[3][3], n9[3][3];
        load9(G, c, C, z, r9);
#pragma unroll
        for (int b = 0; b < 3; ++b)
#pragma unroll
            for (int a = 0; a < 3; ++a) r9[b][a] = mix01(rho_l, rho_g, r9[b][a]);
        gr.add(G, in_plane<T, true, false>(G, r9));
        const T* const vel[3] = {u, v, w};
        V part[3];
#pragma unroll
        for (int d = 0; d < 3; ++d) {
            load9(G, c, vel[d], z, n9);
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
        const int q = z - 1;
        if (q >= c.z0 && c.ok) {
            V gx, gy, gz; gr.grad(G, gx, gy, gz);
            stv(bout + at(c, q), (-div + (q0[0] * gx + q0[1] * gy + q0[2] * gz)) * inv_dt);
        }
    }
}

// ---- stage 1, hydrostatic and surface-tension pressure (Eqs. 20-23, 44; readings in DESIGN.md) ----
// n_t = grad C / (eps_t + |grad C|), eps_t = 1e-7 / hx  (Eq. 23)
template <typename T, int W>
__global__ void __launch_bounds__(MBX* MBY) normals_march(const Geo<T> G, const T* __restrict__ C, T* __restrict__ nx_, T* __restrict__ ny_,
                                                        T* __restrict__ nz_) {
    typedef Pk<T, W> V;
    const Col<T, W> c = make_col<T, W>(G);
    const T eps_t = T(1e-7) / G.h[0];
    GradRoll<T, V> g; g.init();
    for (int z = c.z0 - 1; z <= c.z1; ++z) {
        V n9[3][3];
        load9(G, c, C, z, n9);
        g.add(G, in_plane<T, true, false>(G, n9));
        const int q = z - 1;
        if (q >= c.z0 && c.ok) {
            V gx, gy, gz; g.grad(G, gx, gy, gz);
            const V inv = T(1) / (eps_t + psqrt(gx * gx + gy * gy + gz * gz));
            const size_t c0 = at(c, q);
            stv(nx_ + c0, gx * inv); stv(ny_ + c0, gy * inv); stv(nz_ + c0, gz * inv);
        }
    }
}

// kappa = -(f(n_tu; w_x) + f(n_tv; w_y) + f(n_tw; w_z)) (Eqs. 5, 22; sign: reading N3);  s_t = sigma_t kappa grad C (Eq. 21);
// (fu, fv, fw) = -s_t + (0, 0, g rho), whose FE divergence is the right-hand side of Eq. 43
template <typename T, int W>
__global__ void __launch_bounds__(MBX* MBY) surface_tension_march(const Geo<T> G, const T* __restrict__ C, const T* __restrict__ nx_,
                                                                const T* __restrict__ ny_, const T* __restrict__ nz_, T rho_l, T rho_g,
                                                                T grav, T sigma_t, T* __restrict__ fu, T* __restrict__ fv,
                                                                T* __restrict__ fw, T* __restrict__ kappa) {
    typedef Pk<T, W> V;
    const Col<T, W> c = make_col<T, W>(G);
    GradRoll<T, V> g; g.init();
    ZAcc<V> acc; acc.init();                                      // Mz (Dx My n_x + Mx Dy n_y) + Dz (Mx My n_z)
    V C0 = {}, C0n = {};
    for (int z = c.z0 - 1; z <= c.z1; ++z) {
        V n9[3][3];
        load9(G, c, C, z, n9);
        g.add(G, in_plane<T, true, false>(G, n9));
        C0 = C0n; C0n = n9[1][1];
        load9(G, c, nx_, z, n9); const V dx = in_plane<T, true, false>(G, n9).dm;
        load9(G, c, ny_, z, n9); const V dy = in_plane<T, true, false>(G, n9).md;
        load9(G, c, nz_, z, n9); const V mz = in_plane<T, false, false>(G, n9).mm;
        const V ms = G.M[0] * (dx + dy), dn = G.D[2][2] * mz;
        const V divn = acc.step(ms + dn, G.M[1] * (dx + dy), ms - dn);
        const int q = z - 1;
        if (q >= c.z0 && c.ok) {
            V gx, gy, gz; g.grad(G, gx, gy, gz);
            const V kap = -divn;
            const size_t c0 = at(c, q);
            const V sk = -sigma_t * kap;                        // -s_t = sk grad C
            stv(fu + c0, sk * gx); stv(fv + c0, sk * gy);
            stv(fw + c0, sk * gz + grav * mix01(rho_l, rho_g, C0));
            if (kappa) stv(kappa + c0, kap);
        }
    }
}

// bottom boundary condition dp_hs/dz = -rho g: ghost below = mirror + hz g rho(mirror); its stencil contribution
// sum_j (-w_lap_ij) hz g rho_j over the ghost plane is added to b on the bottom plane
template <typename T>
__global__ void bottom_fold_kernel(const Geo<T> G, const T* __restrict__ C, T rho_l, T rho_g, T grav, T* __restrict__ b) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y * blockDim.y + threadIdx.y;
    if (i >= G.nx || j >= G.ny) return;
    T add = T(0);
#pragma unroll
    for (int bb = 0; bb < 3; ++bb)
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            const int ii = min(max(i + a - 1, 0), G.nx - 1), jj = min(max(j + bb - 1, 0), G.ny - 1);
            const T Cv = C[(size_t)jj * G.nx + ii];
            const T wl = (G.K[0][a] * G.M[bb] + G.M[a] * G.K[1][bb]) * G.M[0] + G.M[a] * G.M[bb] * G.K[2][0];
            add -= wl * G.h[2] * grav * mix01(rho_l, rho_g, Cv);
        }
    b[(size_t)j * G.nx + i] += add;
}
