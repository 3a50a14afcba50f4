// flow.cu -- explicit stencil residuals that feed the pressure solve (rows a8-a10 of the hot
// path): compressive-advection VoF residual, momentum advection-diffusion predictor, pressure
// right-hand side and velocity projection, plus the config-5 time step built from them.
//
// All filters are the NODAL (divided by m_l = dx dy dz, the paper's w_ml^-1) tensor
// products of the 1-D trilinear-FE factors (Eqs. 9-11):
//   derivative D = [-1, 0, 1]/(2 d),  mass M = [1, 4, 1]/6,  stiffness K = [-1, 2, -1]/d^2
//   w_x = Dx My Mz, ...;  w_xx = Kx My Mz, ...;  w_m/m_l = Mx My Mz;  w_lap = w_xx + w_yy + w_zz.
// Halos of C, velocities and derived fields are zero-derivative copies (reading C9-iv);
// the pressure halo in the projection uses the solver's factors (reading C10).
#include <cmath>

#include "solver.h"

namespace mgb {
namespace {

template <typename T>
struct Geo {
    int nx, ny, nz;
    T D[3][3];  // D[axis][-1..1]
    T K[3][3];
    T M[3];
    T h[3];
    T s[6];     // halo factors of the pressure (projection only)
    int uniform;
};

template <typename T>
Geo<T> make_geo(const mg_grid* g, const int* bc) {
    Geo<T> G;
    G.nx = g->nx; G.ny = g->ny; G.nz = g->nz;
    const double h[3] = {g->hx, g->hy, g->hz};
    for (int a = 0; a < 3; ++a) {
        G.D[a][0] = (T)(-0.5 / h[a]); G.D[a][1] = T(0); G.D[a][2] = (T)(0.5 / h[a]);
        G.K[a][0] = G.K[a][2] = (T)(-1.0 / (h[a] * h[a])); G.K[a][1] = (T)(2.0 / (h[a] * h[a]));
        G.h[a] = (T)h[a];
    }
    G.M[0] = G.M[2] = (T)(1.0 / 6.0); G.M[1] = (T)(4.0 / 6.0);
    for (int f = 0; f < 6; ++f) G.s[f] = bc ? (T)(bc[f] == MG_BC_NEUMANN ? 1.0 : (bc[f] == MG_BC_DIRICHLET ? -1.0 : 0.0)) : T(1);
    G.uniform = (g->hx == g->hy && g->hy == g->hz);
    return G;
}

constexpr int BX = 64, BY = 4;

template <typename T>
dim3 grid_for(const Geo<T>& G) { return dim3((G.nx + BX - 1) / BX, (G.ny + BY - 1) / BY, G.nz); }

struct Nb {  // clamped neighbour indices (copy halo)
    int ix[3], jy[3], kz[3];
};

template <typename T>
__device__ __forceinline__ Nb neighbours(const Geo<T>& G, int i, int j, int k) {
    Nb n;
    n.ix[0] = i > 0 ? i - 1 : 0; n.ix[1] = i; n.ix[2] = i < G.nx - 1 ? i + 1 : G.nx - 1;
    n.jy[0] = j > 0 ? j - 1 : 0; n.jy[1] = j; n.jy[2] = j < G.ny - 1 ? j + 1 : G.ny - 1;
    n.kz[0] = k > 0 ? k - 1 : 0; n.kz[1] = k; n.kz[2] = k < G.nz - 1 ? k + 1 : G.nz - 1;
    return n;
}

template <typename T>
__device__ __forceinline__ size_t at(const Geo<T>& G, const Nb& n, int a, int b, int c) {
    return (size_t)n.ix[a] + (size_t)G.nx * ((size_t)n.jy[b] + (size_t)G.ny * n.kz[c]);
}

// gradient of f by the FE first-derivative filters (Eq. 11 / m_l), copy halo
template <typename T>
__device__ __forceinline__ void fe_gradient(const Geo<T>& G, const Nb& n, const T* __restrict__ f, T& gx, T& gy, T& gz) {
    T sx = T(0), sy = T(0), sz = T(0);
#pragma unroll
    for (int c = 0; c < 3; ++c)
#pragma unroll
        for (int b = 0; b < 3; ++b)
#pragma unroll
            for (int a = 0; a < 3; ++a) {
                const T v = f[at(G, n, a, b, c)];
                if (a != 1) sx += (G.D[0][a] * G.M[b] * G.M[c]) * v;
                if (b != 1) sy += (G.M[a] * G.D[1][b] * G.M[c]) * v;
                if (c != 1) sz += (G.M[a] * G.M[b] * G.D[2][c]) * v;
            }
    gx = sx; gy = sy; gz = sz;
}

// Eq. 29: a = alpha_a f(adv; w_m/m_l - E), alpha_a = 2
template <typename T>
__device__ __forceinline__ T mixed_mass(const Geo<T>& G, const Nb& n, const T* __restrict__ adv) {
    T s = T(0);
#pragma unroll
    for (int c = 0; c < 3; ++c)
#pragma unroll
        for (int b = 0; b < 3; ++b)
#pragma unroll
            for (int a = 0; a < 3; ++a) {
                T wgt = G.M[a] * G.M[b] * G.M[c];
                if (a == 1 && b == 1 && c == 1) wgt -= T(1);
                s += wgt * adv[at(G, n, a, b, c)];
            }
    return T(2) * s;
}

// Eqs. 26/27: alpha_kabs = 1/16 (p = 1), eps_k = 1e-7; Eq. 27 on
// uniform spacing, Eq. 26 otherwise (reading C9-ii).
template <typename T>
__device__ __forceinline__ T k_abs_pg(const Geo<T>& G, T a, T px, T py, T pz) {
    const T alpha_kabs = T(1.0 / 16.0), eps_k = T(1e-7);
    const T ax = fabs(px), ay = fabs(py), az = fabs(pz);
    const T s = ax + ay + az;
    if (G.uniform) return alpha_kabs * G.h[0] * fabs(a) / (eps_k + s / T(3));
    return alpha_kabs * fabs(a) * (G.h[0] * ax + G.h[1] * ay + G.h[2] * az) / (eps_k + s * s / T(3));
}

template <typename T> __device__ __forceinline__ T tmin(T a, T b) { return a < b ? a : b; }
template <typename T> __device__ __forceinline__ T tmax(T a, T b) { return a > b ? a : b; }

#define POINT_PROLOGUE                                                                          \
    const int i = blockIdx.x * BX + threadIdx.x, j = blockIdx.y * BY + threadIdx.y, k = blockIdx.z; \
    if (i >= G.nx || j >= G.ny) return;                                                          \
    const Nb n = neighbours(G, i, j, k);                                                         \
    const size_t c0 = (size_t)i + (size_t)G.nx * ((size_t)j + (size_t)G.ny * k)

// steps 1-2 of reading C9: adv = u psi_x + v psi_y + w psi_z
template <typename T>
__global__ void __launch_bounds__(BX* BY) advection_kernel(const Geo<T> G, const T* __restrict__ psi, const T* __restrict__ u,
                                                          const T* __restrict__ v, const T* __restrict__ w, T* __restrict__ adv) {
    POINT_PROLOGUE;
    T px, py, pz;
    fe_gradient(G, n, psi, px, py, pz);
    adv[c0] = u[c0] * px + v[c0] * py + w[c0] * pz;
}

// steps 3-10 of reading C9: directional diffusion coefficients k^x, k^y, k^z of the compressive scheme
template <typename T>
__global__ void __launch_bounds__(BX* BY) vof_coeff_kernel(const Geo<T> G, const T* __restrict__ C, const T* __restrict__ u,
                                                          const T* __restrict__ v, const T* __restrict__ w,
                                                          const T* __restrict__ adv, T k_min, T k_max, T* __restrict__ kx,
                                                          T* __restrict__ ky, T* __restrict__ kz) {
    POINT_PROLOGUE;
    const T Kp = T(300), Km = T(300);        // K+, K- 
    const T beta = T(0.1), eps_x = T(1e-4);  // Eq. 36
    const T Kcal = T(3);                     // Eq. 39
    T Cx, Cy, Cz;
    fe_gradient(G, n, C, Cx, Cy, Cz);
    const T a = mixed_mass(G, n, adv);                                   // step 3, Eq. 29
    const T kabs = k_abs_pg(G, a, Cx, Cy, Cz);                           // step 4, Eq. 27
    const T C0 = C[c0];
    T S[3];                                                              // step 5, Eq. 33
    S[0] = (C0 - C[at(G, n, 0, 1, 1)]) * (C[at(G, n, 2, 1, 1)] - C0);
    S[1] = (C0 - C[at(G, n, 1, 0, 1)]) * (C[at(G, n, 1, 2, 1)] - C0);
    S[2] = (C0 - C[at(G, n, 1, 1, 0)]) * (C[at(G, n, 1, 1, 2)] - C0);
    if (C0 > T(0.95) || C0 < T(0.05)) S[0] = S[1] = S[2] = T(-1);        // override
    const T uu = u[c0], vv = v[c0], ww = w[c0];
    const T g2 = Cx * Cx + Cy * Cy + Cz * Cz;
    const T gq = (uu * Cx + vv * Cy + ww * Cz) / (eps_x + g2);           // step 7, Eq. 37
    const T us = gq * Cx, vs = gq * Cy, ws = gq * Cz;
    const T kneg = -beta * (uu * uu + vv * vv + ww * ww) /               // step 8, Eq. 36
                   (eps_x + g2 * (fabs(us) + fabs(vs) + fabs(ws)) / T(3));
    T* const out[3] = {kx, ky, kz};
#pragma unroll
    for (int d = 0; d < 3; ++d) {
        const T wp = -tmax(T(-1), tmin(T(0), Kp * S[d]));                // step 6, Eq. 35
        const T wm = tmin(T(1), tmax(T(0), Km * S[d]));
        const T kk = wp * (Kcal * kabs) + wm * (kneg / G.h[d]);          // steps 9, Eqs. 38-40
        out[d][c0] = tmax(-k_min, tmin(k_max, kk));                      // step 10, Eq. 41
    }
}

// steps 11-12: sC = adv + sum_d diff_d, diff_d = sum_{j != i} (-W^dd_ij) 1/2 (k^d_i + k^d_j)(C_i - C_j)
// (Eq. 12 collapsed); Cnew = C - dt sC (Eq. 55)
template <typename T>
__global__ void __launch_bounds__(BX* BY) vof_diffusion_kernel(const Geo<T> G, const T* __restrict__ C, const T* __restrict__ adv,
                                                              const T* __restrict__ kx, const T* __restrict__ ky,
                                                              const T* __restrict__ kz, T dt, T* __restrict__ sC,
                                                              T* __restrict__ Cnew) {
    POINT_PROLOGUE;
    const T C0 = C[c0], kx0 = kx[c0], ky0 = ky[c0], kz0 = kz[c0];
    T dx = T(0), dy = T(0), dz = T(0);
#pragma unroll
    for (int c = 0; c < 3; ++c)
#pragma unroll
        for (int b = 0; b < 3; ++b)
#pragma unroll
            for (int a = 0; a < 3; ++a) {
                if (a == 1 && b == 1 && c == 1) continue;
                const size_t q = at(G, n, a, b, c);
                const T dC = T(0.5) * (C0 - C[q]);
                dx -= (G.K[0][a] * G.M[b] * G.M[c]) * (kx0 + kx[q]) * dC;
                dy -= (G.M[a] * G.K[1][b] * G.M[c]) * (ky0 + ky[q]) * dC;
                dz -= (G.M[a] * G.M[b] * G.K[2][c]) * (kz0 + kz[q]) * dC;
            }
    const T s = adv[c0] + dx + dy + dz;
    if (sC) sC[c0] = s;
    if (Cnew) Cnew[c0] = C0 - dt * s;
}

// momentum: k_c = rho min{k_max, k_abs(c)} + mu (Eqs. 30-32; k_square of the lost Eq. 28 omitted)
template <typename T>
__global__ void __launch_bounds__(BX* BY) mom_coeff_kernel(const Geo<T> G, const T* __restrict__ C, const T* __restrict__ comp,
                                                          const T* __restrict__ u, const T* __restrict__ v, const T* __restrict__ w,
                                                          const T* __restrict__ adv, T rho_l, T rho_g, T mu_l, T mu_g,
                                                          T* __restrict__ kc) {
    POINT_PROLOGUE;
    T px, py, pz;
    fe_gradient(G, n, comp, px, py, pz);
    const T a = mixed_mass(G, n, adv);
    const T Cc = C[c0];
    const T rho = rho_l * Cc + rho_g * (T(1) - Cc);
    const T mu = mu_l * Cc + mu_g * (T(1) - Cc);
    const T kmax = G.h[0] * fabs(u[c0]) + G.h[1] * fabs(v[c0]) + G.h[2] * fabs(w[c0]);   // Eq. 30
    const T kabs = k_abs_pg(G, a, px, py, pz);
    kc[c0] = rho * tmin(kmax, kabs) + mu;
}

// s = rho adv + f^lap(c, k_c; w_lap) (Eq. 18 without pressure / source terms), q~ = q_n - dt s / rho (Eq. 45,
// sigma = 0), q_half' = (q_n + q~)/2 (Eq. 46)
template <typename T>
__global__ void __launch_bounds__(BX* BY) mom_update_kernel(const Geo<T> G, const T* __restrict__ C, const T* __restrict__ comp,
                                                           const T* __restrict__ kc, const T* __restrict__ adv,
                                                           const T* __restrict__ qn, T rho_l, T rho_g, T dt, T* __restrict__ qt,
                                                           T* __restrict__ qhn) {
    POINT_PROLOGUE;
    const T x0 = comp[c0], k0 = kc[c0];
    T diff = T(0);
#pragma unroll
    for (int c = 0; c < 3; ++c)
#pragma unroll
        for (int b = 0; b < 3; ++b)
#pragma unroll
            for (int a = 0; a < 3; ++a) {
                if (a == 1 && b == 1 && c == 1) continue;
                const size_t q = at(G, n, a, b, c);
                const T wl = G.K[0][a] * G.M[b] * G.M[c] + G.M[a] * G.K[1][b] * G.M[c] + G.M[a] * G.M[b] * G.K[2][c];
                diff -= wl * T(0.5) * (k0 + kc[q]) * (x0 - comp[q]);
            }
    const T Cc = C[c0];
    const T rho = rho_l * Cc + rho_g * (T(1) - Cc);
    const T s = rho * adv[c0] + diff;
    const T t = qn[c0] - dt * s / rho;
    qt[c0] = t;
    if (qhn) qhn[c0] = T(0.5) * (qn[c0] + t);
}

// b = -(1/dt)(f(u; w_x) + f(v; w_y) + f(w; w_z))  (reading C10; Eq. 53 structure)
template <typename T>
__global__ void __launch_bounds__(BX* BY) pressure_rhs_kernel(const Geo<T> G, const T* __restrict__ u, const T* __restrict__ v,
                                                             const T* __restrict__ w, T inv_dt, T* __restrict__ bout) {
    POINT_PROLOGUE;
    T sx = T(0), sy = T(0), sz = T(0);
#pragma unroll
    for (int c = 0; c < 3; ++c)
#pragma unroll
        for (int b = 0; b < 3; ++b)
#pragma unroll
            for (int a = 0; a < 3; ++a) {
                const size_t q = at(G, n, a, b, c);
                if (a != 1) sx += (G.D[0][a] * G.M[b] * G.M[c]) * u[q];
                if (b != 1) sy += (G.M[a] * G.D[1][b] * G.M[c]) * v[q];
                if (c != 1) sz += (G.M[a] * G.M[b] * G.D[2][c]) * w[q];
            }
    bout[c0] = -(sx + sy + sz) * inv_dt;
}

// q <- q - dt k f(p; w_x|y|z) (Eq. 54); halo of p = s * mirror with the solver's factors
template <typename T>
__global__ void __launch_bounds__(BX* BY) project_kernel(const Geo<T> G, const T* __restrict__ p, const T* __restrict__ kc, T dt,
                                                        T* __restrict__ u, T* __restrict__ v, T* __restrict__ w) {
    POINT_PROLOGUE;
    T fx[3] = {i > 0 ? T(1) : G.s[0], T(1), i < G.nx - 1 ? T(1) : G.s[1]};
    T fy[3] = {j > 0 ? T(1) : G.s[2], T(1), j < G.ny - 1 ? T(1) : G.s[3]};
    T fz[3] = {k > 0 ? T(1) : G.s[4], T(1), k < G.nz - 1 ? T(1) : G.s[5]};
    T gx = T(0), gy = T(0), gz = T(0);
#pragma unroll
    for (int c = 0; c < 3; ++c)
#pragma unroll
        for (int b = 0; b < 3; ++b)
#pragma unroll
            for (int a = 0; a < 3; ++a) {
                const T val = fx[a] * fy[b] * fz[c] * p[at(G, n, a, b, c)];
                if (a != 1) gx += (G.D[0][a] * G.M[b] * G.M[c]) * val;
                if (b != 1) gy += (G.M[a] * G.D[1][b] * G.M[c]) * val;
                if (c != 1) gz += (G.M[a] * G.M[b] * G.D[2][c]) * val;
            }
    const T f = dt * kc[c0];
    u[c0] -= f * gx; v[c0] -= f * gy; w[c0] -= f * gz;
}

struct Scratch {  // stream-ordered scratch fields
    cudaStream_t st;
    void* p[4] = {nullptr, nullptr, nullptr, nullptr};
    int n = 0;
    explicit Scratch(cudaStream_t s) : st(s) {}
    int alloc(int count, size_t bytes) {
        for (n = 0; n < count; ++n)
            if (cudaMallocAsync(&p[n], bytes, st) != cudaSuccess) {
                set_error("flow scratch: cudaMallocAsync failed: %s", cudaGetErrorString(cudaGetLastError()));
                return MG_EALLOC;
            }
        return 0;
    }
    ~Scratch() { for (int q = 0; q < n; ++q) cudaFreeAsync(p[q], st); }
};

template <typename T>
int vof_residual_t(const mg_grid* g, const T* C, const T* u, const T* v, const T* w, double dt, T* sC, T* Cnew, cudaStream_t st) {
    const Geo<T> G = make_geo<T>(g, nullptr);
    const size_t bytes = npts(g->nx, g->ny, g->nz) * sizeof(T);
    Scratch ws(st);
    int rc = ws.alloc(4, bytes);
    if (rc) return rc;
    T *adv = (T*)ws.p[0], *kx = (T*)ws.p[1], *ky = (T*)ws.p[2], *kz = (T*)ws.p[3];
    const double hmax = fmax(g->hx, fmax(g->hy, g->hz)), hmin = fmin(g->hx, fmin(g->hy, g->hz));
    const double k_min = 1e-4 / dt * hmax * hmax, k_max = 0.05 / dt * hmin * hmin;   // Eq. 42
    const dim3 grd = grid_for(G), blk(BX, BY);
    advection_kernel<T><<<grd, blk, 0, st>>>(G, C, u, v, w, adv);
    vof_coeff_kernel<T><<<grd, blk, 0, st>>>(G, C, u, v, w, adv, (T)k_min, (T)k_max, kx, ky, kz);
    vof_diffusion_kernel<T><<<grd, blk, 0, st>>>(G, C, adv, kx, ky, kz, (T)dt, sC, Cnew);
    MGB_LAUNCH_CHECK();
    return 0;
}

template <typename T>
int mom_predictor_t(const mg_grid* g, const T* C, const T* const qh[3], const T* const qn[3], double rho_l, double rho_g,
                    double mu_l, double mu_g, double dt, T* const qt[3], T* const qhn[3], cudaStream_t st) {
    const Geo<T> G = make_geo<T>(g, nullptr);
    const size_t bytes = npts(g->nx, g->ny, g->nz) * sizeof(T);
    Scratch ws(st);
    int rc = ws.alloc(2, bytes);
    if (rc) return rc;
    T *adv = (T*)ws.p[0], *kc = (T*)ws.p[1];
    const dim3 grd = grid_for(G), blk(BX, BY);
    for (int c = 0; c < 3; ++c) {
        advection_kernel<T><<<grd, blk, 0, st>>>(G, qh[c], qh[0], qh[1], qh[2], adv);
        mom_coeff_kernel<T><<<grd, blk, 0, st>>>(G, C, qh[c], qh[0], qh[1], qh[2], adv, (T)rho_l, (T)rho_g, (T)mu_l, (T)mu_g, kc);
        mom_update_kernel<T><<<grd, blk, 0, st>>>(G, C, qh[c], kc, adv, qn[c], (T)rho_l, (T)rho_g, (T)dt, qt[c],
                                                  qhn ? qhn[c] : (T*)nullptr);
    }
    MGB_LAUNCH_CHECK();
    return 0;
}

template <typename T>
int pressure_rhs_t(const mg_grid* g, const T* u, const T* v, const T* w, double dt, T* b, cudaStream_t st) {
    const Geo<T> G = make_geo<T>(g, nullptr);
    pressure_rhs_kernel<T><<<grid_for(G), dim3(BX, BY), 0, st>>>(G, u, v, w, (T)(1.0 / dt), b);
    MGB_LAUNCH_CHECK();
    return 0;
}

template <typename T>
int project_t(const mg_grid* g, const int* bc, const T* p, const T* k, double dt, T* u, T* v, T* w, cudaStream_t st) {
    const Geo<T> G = make_geo<T>(g, bc);
    project_kernel<T><<<grid_for(G), dim3(BX, BY), 0, st>>>(G, p, k, (T)dt, u, v, w);
    MGB_LAUNCH_CHECK();
    return 0;
}

bool grid_ok(const mg_grid* g, int dtype) {
    if (!g || g->nx < 1 || g->ny < 1 || g->nz < 1 || !(g->hx > 0) || !(g->hy > 0) || !(g->hz > 0) ||
        (dtype != MG_F32 && dtype != MG_F64)) {
        set_error("invalid grid or dtype");
        return false;
    }
    return true;
}

}  // namespace
}  // namespace mgb

using namespace mgb;

extern "C" {

int vof_residual(const mg_grid* grid, int dtype, const void* d_C, const void* d_u, const void* d_v, const void* d_w, double dt,
                 void* d_sC_out, void* d_Cnew_out, void* cuda_stream) {
    if (!grid_ok(grid, dtype)) return MG_EINVAL;
    if (!d_C || !d_u || !d_v || !d_w || !(dt > 0.0) || (!d_sC_out && !d_Cnew_out) || d_Cnew_out == d_C || d_sC_out == d_C) {
        set_error("vof_residual: NULL / aliased argument or dt <= 0");
        return MG_EINVAL;
    }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if (dtype == MG_F32)
        return vof_residual_t<float>(grid, (const float*)d_C, (const float*)d_u, (const float*)d_v, (const float*)d_w, dt,
                                     (float*)d_sC_out, (float*)d_Cnew_out, st);
    return vof_residual_t<double>(grid, (const double*)d_C, (const double*)d_u, (const double*)d_v, (const double*)d_w, dt,
                                  (double*)d_sC_out, (double*)d_Cnew_out, st);
}

int mom_predictor(const mg_grid* grid, int dtype, const void* d_C, const void* const d_qh[3], const void* const d_qn[3],
                  double rho_l, double rho_g, double mu_l, double mu_g, double dt, void* const d_qt[3], void* const d_qhn[3],
                  void* cuda_stream) {
    if (!grid_ok(grid, dtype)) return MG_EINVAL;
    if (!d_C || !d_qh || !d_qn || !d_qt || !(dt > 0.0)) { set_error("mom_predictor: NULL argument or dt <= 0"); return MG_EINVAL; }
    for (int c = 0; c < 3; ++c) {
        if (!d_qh[c] || !d_qn[c] || !d_qt[c] || (d_qhn && !d_qhn[c])) { set_error("mom_predictor: NULL component"); return MG_EINVAL; }
        for (int e = 0; e < 3; ++e)
            if (d_qt[c] == d_qh[e] || d_qt[c] == d_qn[e] || (d_qhn && (d_qhn[c] == d_qh[e] || d_qhn[c] == d_qn[e]))) {
                set_error("mom_predictor: outputs alias inputs");
                return MG_EINVAL;
            }
    }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if (dtype == MG_F32)
        return mom_predictor_t<float>(grid, (const float*)d_C, (const float* const*)d_qh, (const float* const*)d_qn, rho_l, rho_g,
                                      mu_l, mu_g, dt, (float* const*)d_qt, (float* const*)d_qhn, st);
    return mom_predictor_t<double>(grid, (const double*)d_C, (const double* const*)d_qh, (const double* const*)d_qn, rho_l, rho_g,
                                   mu_l, mu_g, dt, (double* const*)d_qt, (double* const*)d_qhn, st);
}

int pressure_rhs(const mg_grid* grid, int dtype, const void* d_u, const void* d_v, const void* d_w, double dt, void* d_b,
                 void* cuda_stream) {
    if (!grid_ok(grid, dtype)) return MG_EINVAL;
    if (!d_u || !d_v || !d_w || !d_b || !(dt > 0.0)) { set_error("pressure_rhs: NULL argument or dt <= 0"); return MG_EINVAL; }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if (dtype == MG_F32) return pressure_rhs_t<float>(grid, (const float*)d_u, (const float*)d_v, (const float*)d_w, dt, (float*)d_b, st);
    return pressure_rhs_t<double>(grid, (const double*)d_u, (const double*)d_v, (const double*)d_w, dt, (double*)d_b, st);
}

int project_velocity(const mg_grid* grid, const int bc[6], int dtype, const void* d_p, const void* d_k, double dt, void* d_u,
                     void* d_v, void* d_w, void* cuda_stream) {
    if (!grid_ok(grid, dtype)) return MG_EINVAL;
    if (!bc || !d_p || !d_k || !d_u || !d_v || !d_w) { set_error("project_velocity: NULL argument"); return MG_EINVAL; }
    for (int f = 0; f < 6; ++f)
        if (bc[f] < 0 || bc[f] > 2) { set_error("project_velocity: bc[%d] invalid", f); return MG_EINVAL; }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if (dtype == MG_F32)
        return project_t<float>(grid, bc, (const float*)d_p, (const float*)d_k, dt, (float*)d_u, (float*)d_v, (float*)d_w, st);
    return project_t<double>(grid, bc, (const double*)d_p, (const double*)d_k, dt, (double*)d_u, (double*)d_v, (double*)d_w, st);
}

// Config-5 time step, stages 2-4 of P:403-505 (readings C9, C10):
//   stage 2: q_half = q_n; twice: (q~, q_half) = predictor(C_n; q_half, q_n)        (Eqs. 45-46, two iterations P:443)
//   stage 3: k = 1/rho(C_n); b = -(1/dt) D.q~; solve A(k) p = b from p = 0; q = q~ - dt k G p   (Eqs. 48, 52-54)
//   stage 4: C <- C - dt s~_C(C_n, q)                                              (Eqs. 16, 55)
int flow_time_step(mg_solver* s, void* d_C, void* d_u, void* d_v, void* d_w, void* d_p, double rho_l, double rho_g, double mu_l,
                   double mu_g, double dt, double tol, int max_cycles, int* cycles_out, double* relres_out) {
    if (!s || !d_C || !d_u || !d_v || !d_w || !d_p) { set_error("flow_time_step: NULL argument"); return MG_EINVAL; }
    int prev = -1;
    cudaGetDevice(&prev);
    cudaSetDevice(s->device);
    const size_t es = s->dtype == MG_F64 ? 8 : 4, bytes = s->lv[0].n * es;
    cudaStream_t st = s->st;
    int rc = 0;
    {
        Scratch ws(st), ws2(st);
        if ((rc = ws.alloc(4, bytes)) || (rc = ws2.alloc(3, bytes))) { if (prev >= 0) cudaSetDevice(prev); return rc; }
        void* qt[3] = {ws.p[0], ws.p[1], ws.p[2]};
        void* qh[3] = {ws2.p[0], ws2.p[1], ws2.p[2]};
        void* bbuf = ws.p[3];
        const void* qn[3] = {d_u, d_v, d_w};
        rc = mom_predictor(&s->grid, s->dtype, d_C, qn, qn, rho_l, rho_g, mu_l, mu_g, dt, qt, qh, st);
        if (!rc) { const void* qhc[3] = {qh[0], qh[1], qh[2]}; rc = mom_predictor(&s->grid, s->dtype, d_C, qhc, qn, rho_l, rho_g, mu_l, mu_g, dt, qt, nullptr, st); }
        if (!rc) rc = mg_set_coefficient_from_vof(s, d_C, rho_l, rho_g);
        if (!rc) rc = pressure_rhs(&s->grid, s->dtype, qt[0], qt[1], qt[2], dt, bbuf, st);
        int status = 0;
        if (!rc) {
            rc = cudaMemsetAsync(d_p, 0, bytes, st) == cudaSuccess ? 0 : MG_ECUDA;
            if (!rc) status = mg_solve(s, d_p, bbuf, tol, max_cycles, cycles_out, relres_out);
            if (status < 0) rc = status;
        }
        if (!rc) rc = project_velocity(&s->grid, s->bc, s->dtype, d_p, s->lv[0].k, dt, qt[0], qt[1], qt[2], st);
        // stage 4 with the projected velocity; C updated through a scratch copy (output must not alias C)
        if (!rc) rc = vof_residual(&s->grid, s->dtype, d_C, qt[0], qt[1], qt[2], dt, nullptr, bbuf, st);
        if (!rc) {
            cudaMemcpyAsync(d_C, bbuf, bytes, cudaMemcpyDeviceToDevice, st);
            cudaMemcpyAsync(d_u, qt[0], bytes, cudaMemcpyDeviceToDevice, st);
            cudaMemcpyAsync(d_v, qt[1], bytes, cudaMemcpyDeviceToDevice, st);
            cudaMemcpyAsync(d_w, qt[2], bytes, cudaMemcpyDeviceToDevice, st);
            if (cudaGetLastError() != cudaSuccess) { set_error("flow_time_step: copy failed"); rc = MG_ECUDA; }
        }
        if (!rc) rc = status;
    }
    if (prev >= 0) cudaSetDevice(prev);
    return rc;
}

}  // extern "C"
