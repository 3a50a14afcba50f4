// flow.cu -- explicit stencil residuals that feed the pressure solve (rows a8-a10 of the hot
// path): compressive-advection VoF residual, momentum advection-diffusion predictor, pressure
// right-hand side and velocity projection, plus the config-5 time step built from them.
// The kernels are in flow_march.cuh (z-marching, W consecutive x points per thread).
//
// All filters are the NODAL (divided by m_l = dx dy dz, the paper's w_ml^-1) tensor
// products of the 1-D trilinear-FE factors (Eqs. 9-11):
//   derivative D = [-1, 0, 1]/(2 d),  mass M = [1, 4, 1]/6,  stiffness K = [-1, 2, -1]/d^2
//   w_x = Dx My Mz, ...;  w_xx = Kx My Mz, ...;  w_m/m_l = Mx My Mz;  w_lap = w_xx + w_yy + w_zz.
// Halos of C, velocities and derived fields are zero-derivative copies (reading C9-iv);
// the pressure halo in the projection uses the solver's factors (reading C10).
#include <algorithm>
#include <cmath>
#include <cstdint>
#include <initializer_list>
#include <mutex>

#include "fused.h"
#include "solver.h"
#include "lean_kernel.cuh"

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

// Eqs. 26/27: alpha_kabs = 1/16 (p = 1), eps_k = 1e-7; Eq. 27 on
// uniform spacing, Eq. 26 otherwise (reading C9-ii).
// a / b: fp32 by the approximate reciprocal (2 ulp; the true division costs ~12 instructions and a branch, and the coefficient
// kernels, which are bound by instruction issue, do three per point), fp64 exactly
__device__ __forceinline__ float fdiv(float a, float b) { return __fdividef(a, b); }
__device__ __forceinline__ double fdiv(double a, double b) { return a / b; }

template <typename T>
__device__ __forceinline__ T k_abs_pg(const Geo<T>& G, T a, T px, T py, T pz) {
    const T alpha_kabs = T(1.0 / 16.0), eps_k = T(1e-7);
    const T ax = fabs(px), ay = fabs(py), az = fabs(pz);
    const T s = ax + ay + az;
    const T third = T(1.0 / 3.0);       // a multiplication, not a second division per point
    if (G.uniform) return fdiv(alpha_kabs * G.h[0] * fabs(a), eps_k + s * third);
    return fdiv(alpha_kabs * fabs(a) * (G.h[0] * ax + G.h[1] * ay + G.h[2] * az), eps_k + s * s * third);
}

template <typename T> __device__ __forceinline__ T tmin(T a, T b) { return a < b ? a : b; }
template <typename T> __device__ __forceinline__ T tmax(T a, T b) { return a > b ? a : b; }

#include "flow_march.cuh"
#include "flow_tma.cuh"

// W-wide kernels need nx % W == 0 and 16-byte aligned fields (vector loads); otherwise the W = 1 instantiation runs
template <typename T> constexpr int vec_w() { return sizeof(T) == 4 ? 4 : 2; }
template <typename T>
bool can_vec(const mg_grid* g, std::initializer_list<const void*> ptrs) {
    if (g->nx % vec_w<T>() != 0) return false;
    for (const void* q : ptrs)
        if (q && (reinterpret_cast<uintptr_t>(q) & 15u)) return false;
    return true;
}
// WV: the pack width of the vector instantiation (a divisor of vec_w<T>())
#define MGB_MARCH_W(KERNEL, WV, VEC, G, st, ...)                                                        \
    do {                                                                                                \
        if (VEC) KERNEL<T, WV><<<march_grid<T, WV>(G), dim3(MBX, MBY), 0, st>>>(G, __VA_ARGS__);        \
        else KERNEL<T, 1><<<march_grid<T, 1>(G), dim3(MBX, MBY), 0, st>>>(G, __VA_ARGS__);              \
    } while (0)
#define MGB_MARCH(KERNEL, VEC, G, st, ...) MGB_MARCH_W(KERNEL, vec_w<T>(), VEC, G, st, __VA_ARGS__)
// the instantiation with halo factors (free-slip walls): the trailing arguments are the Halo6 sets
#define MGB_MARCH_BC(KERNEL, VEC, G, st, ...)                                                                         \
    do {                                                                                                              \
        if (VEC) KERNEL<T, vec_w<T>(), true><<<march_grid<T, vec_w<T>()>(G), dim3(MBX, MBY), 0, st>>>(G, __VA_ARGS__); \
        else KERNEL<T, 1, true><<<march_grid<T, 1>(G), dim3(MBX, MBY), 0, st>>>(G, __VA_ARGS__);                       \
    } while (0)

#define MGB_MARCH_BC_W(KERNEL, WV, VEC, G, st, ...)                                                     \
    do {                                                                                                \
        if (VEC) KERNEL<T, WV, true><<<march_grid<T, WV>(G), dim3(MBX, MBY), 0, st>>>(G, __VA_ARGS__);  \
        else KERNEL<T, 1, true><<<march_grid<T, 1>(G), dim3(MBX, MBY), 0, st>>>(G, __VA_ARGS__);        \
    } while (0)

// halo factors of a field from mg_bc codes (0 copy: +1, 1 odd about the face: -1, 2 zero halo: 0)
template <typename T>
Halo6<T> make_halo(const int* codes) {
    Halo6<T> H;
    for (int f = 0; f < 6; ++f) H.s[f] = (T)(codes[f] == MG_BC_NEUMANN ? 1.0 : (codes[f] == MG_BC_DIRICHLET ? -1.0 : 0.0));
    return H;
}

template <typename T>
__global__ void __launch_bounds__(256) axpy_kernel(size_t n, T* __restrict__ y, const T* __restrict__ x) {
    for (size_t c = blockIdx.x * (size_t)blockDim.x + threadIdx.x; c < n; c += (size_t)gridDim.x * blockDim.x) y[c] += x[c];
}
template <typename T>
int launch_axpy(size_t n, T* y, const T* x, cudaStream_t st) {
    axpy_kernel<T><<<(int)std::min<size_t>((n + 255) / 256, (size_t)sm_count() * 16), 256, 0, st>>>(n, y, x);
    MGB_LAUNCH_CHECK();
    return 0;
}

struct Scratch {  // stream-ordered scratch fields
    cudaStream_t st;
    void* p[4] = {nullptr, nullptr, nullptr, nullptr};
    int n = 0;
    explicit Scratch(cudaStream_t s) : st(s) {}
    int alloc(int count, size_t bytes) {
        // keep freed scratch in the device's default pool: with the default release threshold (0) every synchronisation
        // hands the memory back to the driver and the next call pays milliseconds to map it again
        static bool pool_set[64] = {false};
        int dev = 0;
        if (cudaGetDevice(&dev) == cudaSuccess && dev >= 0 && dev < 64 && !pool_set[dev]) {
            cudaMemPool_t pool;
            if (cudaDeviceGetDefaultMemPool(&pool, dev) == cudaSuccess) {
                unsigned long long keep = ~0ull;
                cudaMemPoolSetAttribute(pool, cudaMemPoolAttrReleaseThreshold, &keep);
            }
            pool_set[dev] = true;
        }
        for (n = 0; n < count; ++n)
            if (cudaMallocAsync(&p[n], bytes, st) != cudaSuccess) {
                set_error("flow scratch: cudaMallocAsync failed: %s", cudaGetErrorString(cudaGetLastError()));
                return MG_EALLOC;
            }
        return 0;
    }
    ~Scratch() { for (int q = 0; q < n; ++q) cudaFreeAsync(p[q], st); }
};

// ---- TMA-staged variants (flow_tma.cuh): fp32, vector path ------------------------------------------------------------
inline bool tma_path() { static const bool off = getenv("MG_NO_FLOW_TMA") != nullptr; return !off; }
// descriptors of `ns` stencil fields followed by `nc` centre fields
inline int fill_maps(ft::Maps* M, const mg_grid* g, std::initializer_list<const float*> stencil, std::initializer_list<const float*> centre) {
    int f = 0, rc;
    for (const float* p : stencil) if ((rc = make_tmap_f32(&M->m[f++], p, g->nx, g->ny, g->nz, ft::PX, ft::PY))) return rc;
    for (const float* p : centre) if ((rc = make_tmap_f32(&M->m[f++], p, g->nx, g->ny, g->nz, ft::TX, ft::TY))) return rc;
    for (; f < ft::MAXF; ++f) M->m[f] = M->m[0];
    return 0;
}
template <int NSF, int NCF, int ND = ft::NS, typename K>
int setup_tma_kernel(K kernel) { return kernel_setup((const void*)kernel, ft::NT, ft::Ring<NSF, NCF, ND>::SMEM, nullptr, true); }

template <typename T>
int vof_residual_t(const mg_grid* g, const T* C, const T* u, const T* v, const T* w, double dt, int detector, T* sC, T* Cnew, cudaStream_t st) {
    const Geo<T> G = make_geo<T>(g, nullptr);
    const size_t bytes = npts(g->nx, g->ny, g->nz) * sizeof(T);
    Scratch ws(st);
    int rc = ws.alloc(4, bytes);
    if (rc) return rc;
    T *adv = (T*)ws.p[0], *kx = (T*)ws.p[1], *ky = (T*)ws.p[2], *kz = (T*)ws.p[3];
    const double hmax = fmax(g->hx, fmax(g->hy, g->hz)), hmin = fmin(g->hx, fmin(g->hy, g->hz));
    const double k_min = 1e-4 / dt * hmax * hmax, k_max = 0.05 / dt * hmin * hmin;   // Eq. 42
    const bool vec = can_vec<T>(g, {C, u, v, w, sC, Cnew});
    bool staged = false;
    if constexpr (sizeof(T) == 4) {
        if (vec && tma_path()) {
            ft::Maps M;
            if ((rc = fill_maps(&M, g, {(const float*)C}, {(const float*)u, (const float*)v, (const float*)w}))) return rc;
            if ((rc = setup_tma_kernel<1, 3>(ft::advection_tma))) return rc;
            ft::advection_tma<<<march_grid<float, 4>(G), dim3(MBX, MBY), ft::Ring<1, 3>::SMEM, st>>>(M, G, (float*)adv);
            staged = true;
        }
    }
    if (!staged) MGB_MARCH(advection_march, vec, G, st, C, u, v, w, adv);
    if constexpr (sizeof(T) == 4) {
        if (staged && detector != 5) {       // Eq. 33 detectors: coefficient and diffusion kernels staged by TMA as well
            ft::Maps M;
            if ((rc = fill_maps(&M, g, {(const float*)C, (const float*)adv}, {(const float*)u, (const float*)v, (const float*)w}))) return rc;
            if ((rc = setup_tma_kernel<2, 3>(ft::vof_coeff_tma))) return rc;
            ft::vof_coeff_tma<<<march_grid<float, 4>(G), dim3(MBX, MBY), ft::Ring<2, 3>::SMEM, st>>>(M, G, (float)k_min, (float)k_max, (float*)kx,
                                                                                                  (float*)ky, (float*)kz);
            if ((rc = fill_maps(&M, g, {(const float*)C, (const float*)kx, (const float*)ky, (const float*)kz}, {(const float*)adv}))) return rc;
            if ((rc = setup_tma_kernel<4, 1>(ft::vof_diffusion_tma))) return rc;
            ft::vof_diffusion_tma<<<march_grid<float, 4>(G), dim3(MBX, MBY), ft::Ring<4, 1>::SMEM, st>>>(M, G, (float)dt, (float*)sC, (float*)Cnew);
            MGB_LAUNCH_CHECK();
            return 0;
        }
    }
    // division-heavy: 4-wide packs cost more in registers than they save in loads (231 vs 248 us at 256^3)
    if (detector == 5) {       // Eq. 34 (vof_coeff_march<T, W, true>)
        if (vec) vof_coeff_march<T, 2, true><<<march_grid<T, 2>(G), dim3(MBX, MBY), 0, st>>>(G, C, u, v, w, adv, (T)k_min, (T)k_max, kx, ky, kz);
        else vof_coeff_march<T, 1, true><<<march_grid<T, 1>(G), dim3(MBX, MBY), 0, st>>>(G, C, u, v, w, adv, (T)k_min, (T)k_max, kx, ky, kz);
    } else
    MGB_MARCH_W(vof_coeff_march, 2, vec, G, st, C, u, v, w, adv, (T)k_min, (T)k_max, kx, ky, kz);
    MGB_MARCH(vof_diffusion_march, vec, G, st, C, adv, kx, ky, kz, (T)dt, sC, Cnew);
    MGB_LAUNCH_CHECK();
    return 0;
}

// vof_residual_t with the four scratch fields given by the caller (vof_residual_noalloc); nothing is allocated or freed
template <typename T>
int vof_residual_scratch_t(const mg_grid* g, const T* C, const T* u, const T* v, const T* w, double dt, int detector, T* sC, T* Cnew,
                           T* adv, T* kx, T* ky, T* kz, cudaStream_t st) {
    const Geo<T> G = make_geo<T>(g, nullptr);
    const double hmax = fmax(g->hx, fmax(g->hy, g->hz)), hmin = fmin(g->hx, fmin(g->hy, g->hz));
    const double k_min = 1e-4 / dt * hmax * hmax, k_max = 0.05 / dt * hmin * hmin;   // Eq. 42
    const bool vec = can_vec<T>(g, {C, u, v, w, sC, Cnew});
    MGB_MARCH(advection_march, vec, G, st, C, u, v, w, adv);
    if (detector == 5) {       // Eq. 34
        if (vec) vof_coeff_march<T, 2, true><<<march_grid<T, 2>(G), dim3(MBX, MBY), 0, st>>>(G, C, u, v, w, adv, (T)k_min, (T)k_max, kx, ky, kz);
        else vof_coeff_march<T, 1, true><<<march_grid<T, 1>(G), dim3(MBX, MBY), 0, st>>>(G, C, u, v, w, adv, (T)k_min, (T)k_max, kx, ky, kz);
    } else
    MGB_MARCH_W(vof_coeff_march, 2, vec, G, st, C, u, v, w, adv, (T)k_min, (T)k_max, kx, ky, kz);
    MGB_MARCH(vof_diffusion_march, vec, G, st, C, adv, kx, ky, kz, (T)dt, sC, Cnew);
    MGB_LAUNCH_CHECK();
    return 0;
}

// mom_predictor_t with the TMA-staged kernels (fp32 vector path): same launches, same arithmetic
template <bool BC>
int mom_predictor_tma_bc(const mg_grid* g, const Geo<float>& G, const float* C, const float* const qh[3], const float* const qn[3], const int* vbc,
                         double rho_l, double rho_g, double mu_l, double mu_g, double dt, float* const qt[3], float* const qhn[3],
                         float* const adv[3], float* kc, cudaStream_t st) {
    int rc;
    ft::Maps M;
    const dim3 grid = march_grid<float, 4>(G), block(MBX, MBY);
    Halo6<float> H[3] = {};
    for (int c = 0; c < 3; ++c) H[c] = BC ? make_halo<float>(vbc + 6 * c) : Halo6<float>{};
    if ((rc = fill_maps(&M, g, {qh[0], qh[1], qh[2]}, {}))) return rc;
    if ((rc = setup_tma_kernel<3, 0>(ft::advection3_tma<BC>))) return rc;
    ft::advection3_tma<BC><<<grid, block, ft::Ring<3, 0>::SMEM, st>>>(M, G, adv[0], adv[1], adv[2], H[0], H[1], H[2]);
    if ((rc = setup_tma_kernel<2, 4, 3>(ft::mom_coeff_tma<BC>)) || (rc = setup_tma_kernel<2, 3, 3>(ft::mom_update_tma<BC>))) return rc;
    for (int c = 0; c < 3; ++c) {
        if ((rc = fill_maps(&M, g, {qh[c], adv[c]}, {C, qh[0], qh[1], qh[2]}))) return rc;
        ft::mom_coeff_tma<BC><<<grid, block, ft::Ring<2, 4, 3>::SMEM, st>>>(M, G, (float)rho_l, (float)rho_g, (float)mu_l, (float)mu_g, kc, H[c]);
        if ((rc = fill_maps(&M, g, {qh[c], kc}, {C, adv[c], qn[c]}))) return rc;
        ft::mom_update_tma<BC><<<grid, block, ft::Ring<2, 3, 3>::SMEM, st>>>(M, G, (float)rho_l, (float)rho_g, (float)dt, qt[c], qhn ? qhn[c] : nullptr, H[c]);
    }
    MGB_LAUNCH_CHECK();
    return 0;
}
inline int mom_predictor_tma(const mg_grid* g, const Geo<float>& G, const float* C, const float* const qh[3], const float* const qn[3], const int* vbc,
                             double rho_l, double rho_g, double mu_l, double mu_g, double dt, float* const qt[3], float* const qhn[3],
                             float* const adv[3], float* kc, cudaStream_t st) {
    return vbc ? mom_predictor_tma_bc<true>(g, G, C, qh, qn, vbc, rho_l, rho_g, mu_l, mu_g, dt, qt, qhn, adv, kc, st)
               : mom_predictor_tma_bc<false>(g, G, C, qh, qn, vbc, rho_l, rho_g, mu_l, mu_g, dt, qt, qhn, adv, kc, st);
}

template <typename T>
int mom_predictor_t(const mg_grid* g, const T* C, const T* const qh[3], const T* const qn[3], const int* vbc, double rho_l, double rho_g,
                    double mu_l, double mu_g, double dt, T* const qt[3], T* const qhn[3], cudaStream_t st) {
    const Geo<T> G = make_geo<T>(g, nullptr);
    const size_t bytes = npts(g->nx, g->ny, g->nz) * sizeof(T);
    Scratch ws(st);
    int rc = ws.alloc(4, bytes);
    if (rc) return rc;
    T *adv[3] = {(T*)ws.p[0], (T*)ws.p[1], (T*)ws.p[2]}, *kc = (T*)ws.p[3];
    const bool vec = can_vec<T>(g, {C, qh[0], qh[1], qh[2], qn[0], qn[1], qn[2], qt[0], qt[1], qt[2], qhn ? qhn[0] : nullptr,
                                    qhn ? qhn[1] : nullptr, qhn ? qhn[2] : nullptr});
    if constexpr (sizeof(T) == 4) {
        if (vec && tma_path()) return mom_predictor_tma(g, G, (const float*)C, (const float* const*)qh, (const float* const*)qn, vbc, rho_l, rho_g,
                                                        mu_l, mu_g, dt, (float* const*)qt, (float* const*)qhn, (float* const*)adv, (float*)kc, st);
    }
    // the advection terms of all three components in one pass (each velocity field is read once), then coefficient and update per
    // component.  2-wide packs: three rolling gradients do not fit the registers of a 4-wide one.
    if (vbc) MGB_MARCH_BC_W(advection3_march, 2, vec, G, st, qh[0], qh[1], qh[2], adv[0], adv[1], adv[2], make_halo<T>(vbc),
                            make_halo<T>(vbc + 6), make_halo<T>(vbc + 12));
    else MGB_MARCH_W(advection3_march, 2, vec, G, st, qh[0], qh[1], qh[2], adv[0], adv[1], adv[2]);
    for (int c = 0; c < 3; ++c) {
        if (vbc) {      // free-slip walls: the component's own halo factors in its gradient and its diffusion
            const Halo6<T> H = make_halo<T>(vbc + 6 * c);
            MGB_MARCH_BC(mom_coeff_march, vec, G, st, C, qh[c], qh[0], qh[1], qh[2], adv[c], (T)rho_l, (T)rho_g, (T)mu_l, (T)mu_g, kc, H);
            MGB_MARCH_BC(mom_update_march, vec, G, st, C, qh[c], kc, adv[c], qn[c], (T)rho_l, (T)rho_g, (T)dt, qt[c], qhn ? qhn[c] : (T*)nullptr, H);
            continue;
        }
        MGB_MARCH(mom_coeff_march, vec, G, st, C, qh[c], qh[0], qh[1], qh[2], adv[c], (T)rho_l, (T)rho_g, (T)mu_l, (T)mu_g, kc);
        MGB_MARCH(mom_update_march, vec, G, st, C, qh[c], kc, adv[c], qn[c], (T)rho_l, (T)rho_g, (T)dt, qt[c], qhn ? qhn[c] : (T*)nullptr);
    }
    MGB_LAUNCH_CHECK();
    return 0;
}

inline int pressure_rhs_tma_launch(const mg_grid* g, const Geo<float>& G, const float* u, const float* v, const float* w, const int* vbc,
                                   float inv_dt, float* b, cudaStream_t st) {
    int rc;
    ft::Maps M;
    if ((rc = fill_maps(&M, g, {u, v, w}, {}))) return rc;
    const dim3 grid = march_grid<float, 4>(G), block(MBX, MBY);
    if (vbc) {
        if ((rc = setup_tma_kernel<3, 0, 3>(ft::pressure_rhs_tma<true>))) return rc;
        ft::pressure_rhs_tma<true><<<grid, block, ft::Ring<3, 0, 3>::SMEM, st>>>(M, G, inv_dt, b, make_halo<float>(vbc), make_halo<float>(vbc + 6),
                                                                                make_halo<float>(vbc + 12));
    } else {
        if ((rc = setup_tma_kernel<3, 0, 3>(ft::pressure_rhs_tma<false>))) return rc;
        ft::pressure_rhs_tma<false><<<grid, block, ft::Ring<3, 0, 3>::SMEM, st>>>(M, G, inv_dt, b, Halo6<float>{}, Halo6<float>{}, Halo6<float>{});
    }
    MGB_LAUNCH_CHECK();
    return 0;
}

template <typename T>
int pressure_rhs_t(const mg_grid* g, const T* u, const T* v, const T* w, const int* vbc, double dt, T* b, cudaStream_t st) {
    const Geo<T> G = make_geo<T>(g, nullptr);
    if constexpr (sizeof(T) == 4) {
        if (can_vec<T>(g, {u, v, w, b}) && tma_path()) return pressure_rhs_tma_launch(g, G, u, v, w, vbc, (float)(1.0 / dt), b, st);
    }
    if (vbc) MGB_MARCH_BC(pressure_rhs_march, can_vec<T>(g, {u, v, w, b}), G, st, u, v, w, (T)(1.0 / dt), b, make_halo<T>(vbc),
                          make_halo<T>(vbc + 6), make_halo<T>(vbc + 12));
    else MGB_MARCH(pressure_rhs_march, can_vec<T>(g, {u, v, w, b}), G, st, u, v, w, (T)(1.0 / dt), b);
    MGB_LAUNCH_CHECK();
    return 0;
}

// q~ <- q~ - (dt / rho)(grad(p_hs + p_nh) + M F), q_half' = (q_n + q~)/2 (mom_forcing_march)
template <typename T>
int mom_forcing_t(const mg_grid* g, const T* C, const T* phs, const T* pnh, const int* pbc, double grav, const T* const F[3],
                  double rho_l, double rho_g, double dt, T* const qt[3], const T* const qn[3], T* const qhn[3], cudaStream_t st) {
    const Geo<T> G = make_geo<T>(g, pbc);
    const bool vec = can_vec<T>(g, {C, phs, pnh, F ? F[0] : nullptr, F ? F[1] : nullptr, F ? F[2] : nullptr, qt[0], qt[1], qt[2],
                                    qhn ? qn[0] : nullptr, qhn ? qn[1] : nullptr, qhn ? qn[2] : nullptr, qhn ? qhn[0] : nullptr,
                                    qhn ? qhn[1] : nullptr, qhn ? qhn[2] : nullptr});
    if constexpr (sizeof(T) == 4) {
        if (vec && tma_path() && phs && pnh && F) {          // the configuration of the four-stage step: every term present
            const Geo<float> Gf = G;
            ft::Maps M;
            int rc;
            if ((rc = fill_maps(&M, g, {(const float*)phs, (const float*)pnh, (const float*)F[0], (const float*)F[1], (const float*)F[2]}, {})) ||
                (rc = setup_tma_kernel<5, 0, 3>(ft::mom_forcing_tma))) return rc;
            ft::mom_forcing_tma<<<march_grid<float, 4>(Gf), dim3(MBX, MBY), ft::Ring<5, 0, 3>::SMEM, st>>>(
                M, Gf, (const float*)C, (float)rho_l, (float)rho_g, (float)grav, (float)dt, (float*)qt[0], (float*)qt[1], (float*)qt[2],
                qhn ? (const float*)qn[0] : nullptr, qhn ? (const float*)qn[1] : nullptr, qhn ? (const float*)qn[2] : nullptr,
                qhn ? (float*)qhn[0] : nullptr, qhn ? (float*)qhn[1] : nullptr, qhn ? (float*)qhn[2] : nullptr);
            MGB_LAUNCH_CHECK();
            return 0;
        }
    }
    // five stencil fields: 2-wide packs keep the rolling sums in registers
    MGB_MARCH_W(mom_forcing_march, 2, vec, G, st, C, phs, pnh, F ? F[0] : (const T*)nullptr, F ? F[1] : (const T*)nullptr,
                F ? F[2] : (const T*)nullptr, (T)rho_l, (T)rho_g, (T)grav, (T)dt, qt[0], qt[1], qt[2],
                qhn ? qn[0] : (const T*)nullptr, qhn ? qn[1] : (const T*)nullptr, qhn ? qn[2] : (const T*)nullptr,
                qhn ? qhn[0] : (T*)nullptr, qhn ? qhn[1] : (T*)nullptr, qhn ? qhn[2] : (T*)nullptr);
    MGB_LAUNCH_CHECK();
    return 0;
}

template <typename T>
int pressure_rhs_paper_t(const mg_grid* g, const T* C, const T* u, const T* v, const T* w, double rho_l, double rho_g, double dt, T* b,
                         cudaStream_t st) {
    const Geo<T> G = make_geo<T>(g, nullptr);
    if constexpr (sizeof(T) == 4) {
        if (can_vec<T>(g, {C, u, v, w, b}) && tma_path()) {
            ft::Maps M;
            int rc;
            if ((rc = fill_maps(&M, g, {C, u, v, w}, {})) || (rc = setup_tma_kernel<4, 0, 3>(ft::pressure_rhs_paper_tma))) return rc;
            ft::pressure_rhs_paper_tma<<<march_grid<float, 4>(G), dim3(MBX, MBY), ft::Ring<4, 0, 3>::SMEM, st>>>(M, G, (float)rho_l, (float)rho_g,
                                                                                                         (float)(1.0 / dt), b);
            MGB_LAUNCH_CHECK();
            return 0;
        }
    }
    MGB_MARCH(pressure_rhs_paper_march, can_vec<T>(g, {C, u, v, w, b}), G, st, C, u, v, w, (T)rho_l, (T)rho_g, (T)(1.0 / dt), b);
    MGB_LAUNCH_CHECK();
    return 0;
}

template <typename T>
int hydrostatic_rhs_t(const mg_grid* g, const T* C, double rho_l, double rho_g, double grav, double sigma_t, T* b, T* kappa,
                      T* const force[3], cudaStream_t st) {
    const Geo<T> G = make_geo<T>(g, nullptr);
    const size_t bytes = npts(g->nx, g->ny, g->nz) * sizeof(T);
    Scratch ws(st), ws2(st);
    int rc;
    if ((rc = ws.alloc(3, bytes)) || (!force && (rc = ws2.alloc(3, bytes)))) return rc;
    T *n0 = (T*)ws.p[0], *n1 = (T*)ws.p[1], *n2 = (T*)ws.p[2];
    T *f0 = force ? force[0] : (T*)ws2.p[0], *f1 = force ? force[1] : (T*)ws2.p[1], *f2 = force ? force[2] : (T*)ws2.p[2];
    const bool vec = can_vec<T>(g, {C, b, kappa, force ? force[0] : nullptr, force ? force[1] : nullptr, force ? force[2] : nullptr});
    bool staged = false;
    if constexpr (sizeof(T) == 4) {
        if (vec && tma_path()) {
            ft::Maps M;
            const dim3 grid = march_grid<float, 4>(G), block(MBX, MBY);
            if ((rc = fill_maps(&M, g, {(const float*)C}, {})) || (rc = setup_tma_kernel<1, 0>(ft::normals_tma))) return rc;
            ft::normals_tma<<<grid, block, ft::Ring<1, 0>::SMEM, st>>>(M, G, (float*)n0, (float*)n1, (float*)n2);
            if ((rc = fill_maps(&M, g, {(const float*)C, (const float*)n0, (const float*)n1, (const float*)n2}, {})) ||
                (rc = setup_tma_kernel<4, 0>(ft::surface_tension_tma))) return rc;
            ft::surface_tension_tma<<<grid, block, ft::Ring<4, 0>::SMEM, st>>>(M, G, (float)rho_l, (float)rho_g, (float)grav, (float)sigma_t, (float*)f0,
                                                                                (float*)f1, (float*)f2, (float*)kappa);
            if ((rc = pressure_rhs_tma_launch(g, G, f0, f1, f2, nullptr, -1.f, b, st))) return rc;
            staged = true;
        }
    }
    if (!staged) {
        MGB_MARCH(normals_march, vec, G, st, C, n0, n1, n2);
        MGB_MARCH(surface_tension_march, vec, G, st, C, n0, n1, n2, (T)rho_l, (T)rho_g, (T)grav, (T)sigma_t, f0, f1, f2, kappa);
    }
    if (!staged) MGB_MARCH(pressure_rhs_march, vec, G, st, f0, f1, f2, T(-1), b);       // b = +(f(fu; w_x) + f(fv; w_y) + f(fw; w_z))
    bottom_fold_kernel<T><<<dim3((g->nx + 31) / 32, (g->ny + 7) / 8), dim3(32, 8), 0, st>>>(G, C, (T)rho_l, (T)rho_g, (T)grav, b);
    MGB_LAUNCH_CHECK();
    return 0;
}

template <typename T>
int project_t(const mg_grid* g, const int* bc, const T* p, const T* k, double dt, T* u, T* v, T* w, cudaStream_t st) {
    const Geo<T> G = make_geo<T>(g, bc);
    if constexpr (sizeof(T) == 4) {
        if (can_vec<T>(g, {p, k, u, v, w}) && tma_path()) {
            int rc;
            ft::Maps M;
            if ((rc = fill_maps(&M, g, {p}, {k, u, v, w}))) return rc;
            if ((rc = setup_tma_kernel<1, 4>(ft::project_tma))) return rc;
            ft::project_tma<<<march_grid<float, 4>(G), dim3(MBX, MBY), ft::Ring<1, 4>::SMEM, st>>>(M, G, (float)dt, u, v, w);
            MGB_LAUNCH_CHECK();
            return 0;
        }
    }
    MGB_MARCH(project_march, can_vec<T>(g, {p, k, u, v, w}), G, st, p, k, (T)dt, u, v, w);
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

// ---- vof_residual_noalloc: scratch that exists without any allocation call ----------------------------------------------------
// The four intermediate fields of the VoF residual (adv, k^x, k^y, k^z) in a file-scope device array: VOF_NOALLOC_SCRATCH_BYTES
// (include/mg.h, 8 MiB) on every GPU that loads the library, until the process exits.  In HOST code `g_vof_scratch` is only a
// stand-in for the symbol, not a device address: the address is asked for once per device, with that device current
// (cudaGetSymbolAddress), and that pointer is what the kernels get.
static __device__ __align__(256) unsigned char g_vof_scratch[VOF_NOALLOC_SCRATCH_BYTES];

static int vof_scratch_address(unsigned char** out) {
    static std::mutex mu;
    static unsigned char* addr[64] = {nullptr};
    int dev = -1;
    MGB_CUDA(cudaGetDevice(&dev));
    std::lock_guard<std::mutex> lock(mu);
    if (dev >= 0 && dev < 64 && addr[dev]) { *out = addr[dev]; return 0; }
    unsigned char* p = nullptr;
    MGB_CUDA(cudaGetSymbolAddress((void**)&p, g_vof_scratch));
    if (!p) { set_error("vof_residual_noalloc: no device address for the scratch array"); return MG_ECUDA; }
    if (dev >= 0 && dev < 64) addr[dev] = p;
    *out = p;
    return 0;
}

extern "C" {

int vof_residual(const mg_grid* grid, int dtype, const void* d_C, const void* d_u, const void* d_v, const void* d_w, double dt,
                 void* d_sC_out, void* d_Cnew_out, void* cuda_stream) {
    return vof_residual_ex(grid, dtype, d_C, d_u, d_v, d_w, dt, 3, d_sC_out, d_Cnew_out, cuda_stream);
}

int vof_residual_ex(const mg_grid* grid, int dtype, const void* d_C, const void* d_u, const void* d_v, const void* d_w, double dt,
                    int detector, void* d_sC_out, void* d_Cnew_out, void* cuda_stream) {
    if (!grid_ok(grid, dtype)) return MG_EINVAL;
    if (detector != 3 && detector != 5) { set_error("vof_residual: detector %d is not 3 (Eq. 33) or 5 (Eq. 34)", detector); return MG_EINVAL; }
    if (!d_C || !d_u || !d_v || !d_w || !(dt > 0.0) || (!d_sC_out && !d_Cnew_out) || d_Cnew_out == d_C || d_sC_out == d_C) {
        set_error("vof_residual: NULL / aliased argument or dt <= 0");
        return MG_EINVAL;
    }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if (dtype == MG_F32)
        return vof_residual_t<float>(grid, (const float*)d_C, (const float*)d_u, (const float*)d_v, (const float*)d_w, dt, detector,
                                     (float*)d_sC_out, (float*)d_Cnew_out, st);
    return vof_residual_t<double>(grid, (const double*)d_C, (const double*)d_u, (const double*)d_v, (const double*)d_w, dt, detector,
                                  (double*)d_sC_out, (double*)d_Cnew_out, st);
}

int vof_residual_noalloc(const mg_grid* grid, int dtype, const void* d_C, const void* d_u, const void* d_v, const void* d_w, double dt,
                         int detector, void* d_sC_out, void* d_Cnew_out, void* cuda_stream) {
    if (!grid_ok(grid, dtype)) return MG_EINVAL;
    if (detector != 3 && detector != 5) { set_error("vof_residual_noalloc: detector %d is not 3 (Eq. 33) or 5 (Eq. 34)", detector); return MG_EINVAL; }
    if (!d_C || !d_u || !d_v || !d_w || !(dt > 0.0) || (!d_sC_out && !d_Cnew_out) || d_Cnew_out == d_C || d_sC_out == d_C) {
        set_error("vof_residual_noalloc: NULL / aliased argument or dt <= 0");
        return MG_EINVAL;
    }
    const size_t esz = dtype == MG_F32 ? 4 : 8;
    const size_t field = (npts(grid->nx, grid->ny, grid->nz) * esz + 255) / 256 * 256;      // every field starts 256-byte aligned
    if (4 * field > (size_t)VOF_NOALLOC_SCRATCH_BYTES) {
        set_error("vof_residual_noalloc: %dx%dx%d %s needs %zu bytes of scratch, the static array holds %zu (VOF_NOALLOC_SCRATCH_BYTES); "
                  "use vof_residual_ex", grid->nx, grid->ny, grid->nz, dtype == MG_F32 ? "fp32" : "fp64", 4 * field,
                  (size_t)VOF_NOALLOC_SCRATCH_BYTES);
        return MG_EINVAL;
    }
    unsigned char* base = nullptr;
    int rc = vof_scratch_address(&base);
    if (rc) return rc;
    // nothing in the scratch has to start at zero: the first kernel writes every point of adv, the second every point of k^x, k^y,
    // k^z, before the kernel that reads them -- whatever an earlier call left there is overwritten
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if (dtype == MG_F32)
        return vof_residual_scratch_t<float>(grid, (const float*)d_C, (const float*)d_u, (const float*)d_v, (const float*)d_w, dt, detector,
                                             (float*)d_sC_out, (float*)d_Cnew_out, (float*)base, (float*)(base + field),
                                             (float*)(base + 2 * field), (float*)(base + 3 * field), st);
    return vof_residual_scratch_t<double>(grid, (const double*)d_C, (const double*)d_u, (const double*)d_v, (const double*)d_w, dt, detector,
                                          (double*)d_sC_out, (double*)d_Cnew_out, (double*)base, (double*)(base + field),
                                          (double*)(base + 2 * field), (double*)(base + 3 * field), st);
}

static bool vbc_ok(const int* vbc) {
    for (int e = 0; vbc && e < 18; ++e)
        if (vbc[e] < 0 || vbc[e] > 2) { set_error("velocity halo code vbc[%d] = %d is not an mg_bc", e, vbc[e]); return false; }
    return true;
}

int mom_predictor(const mg_grid* grid, int dtype, const void* d_C, const void* const d_qh[3], const void* const d_qn[3],
                  double rho_l, double rho_g, double mu_l, double mu_g, double dt, void* const d_qt[3], void* const d_qhn[3],
                  void* cuda_stream) {
    return mom_predictor_bc(grid, dtype, d_C, d_qh, d_qn, nullptr, rho_l, rho_g, mu_l, mu_g, dt, d_qt, d_qhn, cuda_stream);
}

int mom_predictor_bc(const mg_grid* grid, int dtype, const void* d_C, const void* const d_qh[3], const void* const d_qn[3],
                     const int vbc[18], double rho_l, double rho_g, double mu_l, double mu_g, double dt, void* const d_qt[3],
                     void* const d_qhn[3], void* cuda_stream) {
    if (!grid_ok(grid, dtype) || !vbc_ok(vbc)) return MG_EINVAL;
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
        return mom_predictor_t<float>(grid, (const float*)d_C, (const float* const*)d_qh, (const float* const*)d_qn, vbc, rho_l, rho_g,
                                      mu_l, mu_g, dt, (float* const*)d_qt, (float* const*)d_qhn, st);
    return mom_predictor_t<double>(grid, (const double*)d_C, (const double* const*)d_qh, (const double* const*)d_qn, vbc, rho_l, rho_g,
                                   mu_l, mu_g, dt, (double* const*)d_qt, (double* const*)d_qhn, st);
}

int mom_forcing(const mg_grid* grid, int dtype, const void* d_C, const void* d_phs, const void* d_pnh, const int pbc[6], double grav,
                const void* const d_force[3], double rho_l, double rho_g, double dt, void* const d_qt[3], const void* const d_qn[3],
                void* const d_qhn[3], void* cuda_stream) {
    if (!grid_ok(grid, dtype)) return MG_EINVAL;
    if (!d_C || !d_qt || !d_qt[0] || !d_qt[1] || !d_qt[2] || !(dt > 0.0) || !(rho_l > 0.0) || !(rho_g > 0.0) || (d_pnh && !pbc) ||
        (d_force && (!d_force[0] || !d_force[1] || !d_force[2])) ||
        (d_qhn && (!d_qn || !d_qn[0] || !d_qn[1] || !d_qn[2] || !d_qhn[0] || !d_qhn[1] || !d_qhn[2]))) {
        set_error("mom_forcing: NULL argument, dt <= 0 or density <= 0");
        return MG_EINVAL;
    }
    for (int f = 0; pbc && f < 6; ++f)
        if (pbc[f] < 0 || pbc[f] > 2) { set_error("mom_forcing: pbc[%d] invalid", f); return MG_EINVAL; }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if (dtype == MG_F32)
        return mom_forcing_t<float>(grid, (const float*)d_C, (const float*)d_phs, (const float*)d_pnh, pbc, grav, (const float* const*)d_force,
                                    rho_l, rho_g, dt, (float* const*)d_qt, (const float* const*)d_qn, (float* const*)d_qhn, st);
    return mom_forcing_t<double>(grid, (const double*)d_C, (const double*)d_phs, (const double*)d_pnh, pbc, grav, (const double* const*)d_force,
                                 rho_l, rho_g, dt, (double* const*)d_qt, (const double* const*)d_qn, (double* const*)d_qhn, st);
}

int pressure_rhs(const mg_grid* grid, int dtype, const void* d_u, const void* d_v, const void* d_w, double dt, void* d_b,
                 void* cuda_stream) {
    return pressure_rhs_bc(grid, dtype, d_u, d_v, d_w, nullptr, dt, d_b, cuda_stream);
}

int pressure_rhs_bc(const mg_grid* grid, int dtype, const void* d_u, const void* d_v, const void* d_w, const int vbc[18], double dt,
                    void* d_b, void* cuda_stream) {
    if (!grid_ok(grid, dtype) || !vbc_ok(vbc)) return MG_EINVAL;
    if (!d_u || !d_v || !d_w || !d_b || !(dt > 0.0)) { set_error("pressure_rhs: NULL argument or dt <= 0"); return MG_EINVAL; }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if (dtype == MG_F32) return pressure_rhs_t<float>(grid, (const float*)d_u, (const float*)d_v, (const float*)d_w, vbc, dt, (float*)d_b, st);
    return pressure_rhs_t<double>(grid, (const double*)d_u, (const double*)d_v, (const double*)d_w, vbc, dt, (double*)d_b, st);
}

int pressure_rhs_paper(const mg_grid* grid, int dtype, const void* d_C, const void* d_u, const void* d_v, const void* d_w, double rho_l,
                       double rho_g, double dt, void* d_b, void* cuda_stream) {
    if (!grid_ok(grid, dtype)) return MG_EINVAL;
    if (!d_C || !d_u || !d_v || !d_w || !d_b || !(dt > 0.0) || !(rho_l > 0.0) || !(rho_g > 0.0)) {
        set_error("pressure_rhs_paper: NULL argument, dt <= 0 or density <= 0");
        return MG_EINVAL;
    }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if (dtype == MG_F32)
        return pressure_rhs_paper_t<float>(grid, (const float*)d_C, (const float*)d_u, (const float*)d_v, (const float*)d_w, rho_l, rho_g,
                                           dt, (float*)d_b, st);
    return pressure_rhs_paper_t<double>(grid, (const double*)d_C, (const double*)d_u, (const double*)d_v, (const double*)d_w, rho_l,
                                        rho_g, dt, (double*)d_b, st);
}

int hydrostatic_rhs(const mg_grid* grid, int dtype, const void* d_C, double rho_l, double rho_g, double grav, double sigma_t, void* d_b,
                    void* d_kappa_out, void* cuda_stream) {
    return hydrostatic_rhs_force(grid, dtype, d_C, rho_l, rho_g, grav, sigma_t, d_b, d_kappa_out, nullptr, cuda_stream);
}

int hydrostatic_rhs_force(const mg_grid* grid, int dtype, const void* d_C, double rho_l, double rho_g, double grav, double sigma_t,
                          void* d_b, void* d_kappa_out, void* const d_force_out[3], void* cuda_stream) {
    if (!grid_ok(grid, dtype)) return MG_EINVAL;
    if (!d_C || !d_b || !(rho_l > 0.0) || !(rho_g > 0.0) || (d_force_out && (!d_force_out[0] || !d_force_out[1] || !d_force_out[2]))) {
        set_error("hydrostatic_rhs: NULL argument or density <= 0");
        return MG_EINVAL;
    }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if (dtype == MG_F32)
        return hydrostatic_rhs_t<float>(grid, (const float*)d_C, rho_l, rho_g, grav, sigma_t, (float*)d_b, (float*)d_kappa_out,
                                        (float* const*)d_force_out, st);
    return hydrostatic_rhs_t<double>(grid, (const double*)d_C, rho_l, rho_g, grav, sigma_t, (double*)d_b, (double*)d_kappa_out,
                                     (double* const*)d_force_out, st);
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
static int time_step_impl(mg_solver* s, bool pcg, void* d_C, void* d_u, void* d_v, void* d_w, void* d_p, double rho_l, double rho_g,
                          double mu_l, double mu_g, double dt, double tol, int max_cycles, int* cycles_out, double* relres_out) {
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
            if (!rc) status = pcg ? mg_pcg_solve(s, d_p, bbuf, tol, max_cycles, cycles_out, relres_out)
                                  : mg_solve(s, d_p, bbuf, tol, max_cycles, cycles_out, relres_out);
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

int flow_time_step(mg_solver* s, void* d_C, void* d_u, void* d_v, void* d_w, void* d_p, double rho_l, double rho_g, double mu_l,
                   double mu_g, double dt, double tol, int max_cycles, int* cycles_out, double* relres_out) {
    return time_step_impl(s, false, d_C, d_u, d_v, d_w, d_p, rho_l, rho_g, mu_l, mu_g, dt, tol, max_cycles, cycles_out, relres_out);
}

// The same step with the pressure solved by V-cycle-preconditioned CG (oracle time_step(solver="pcg"))
int flow_time_step_pcg(mg_solver* s, void* d_C, void* d_u, void* d_v, void* d_w, void* d_p, double rho_l, double rho_g, double mu_l,
                       double mu_g, double dt, double tol, int max_iter, int* iters_out, double* relres_out) {
    return time_step_impl(s, true, d_C, d_u, d_v, d_w, d_p, rho_l, rho_g, mu_l, mu_g, dt, tol, max_iter, iters_out, relres_out);
}

// The paper's four-stage step (oracle time_step_full):
//   stage 1: b_hs and the force field F = -(s + s_t) from C^n (Eqs. 20-23, 43-44); A p_hs = b_hs with the constant-coefficient
//            solver s_hs from p_hs = 0, hs_cycles cycles (the paper's fixed 20) or to hs_tol
//   stage 2: q_half = q_n; twice: q~ = predictor(C_n; q_half, q_n) with free-slip wall halos, then the forcing terms of
//            Eq. 18 (grad p_hs, grad of the previous p_nh, mass-filtered sources); q_half = (q_n + q~)/2   (Eqs. 45-46)
//   stage 3: k = 1/rho(C_n); b = -(1/dt) D.q~ (wall halos); A(k) dp = b with s_nh; q = q~ - dt k G dp; p_nh += dp   (reading C10)
//   stage 4: C <- C - dt s~_C(C_n, q)
// walls[6]: 1 = free-slip wall, 0 = open face (x-, x+, y-, y+, z-, z+).  Both solvers: same grid and dtype, bc {N,N,N,N,N,D}.
int flow_time_step_full(mg_solver* s_hs, mg_solver* s, void* d_C, void* d_u, void* d_v, void* d_w, void* d_phs, void* d_pnh,
                        double rho_l, double rho_g, double mu_l, double mu_g, double grav, double sigma_t, double dt, double tol,
                        int max_cycles, double hs_tol, int hs_cycles, const int walls[6], int* cycles_out, double* relres_out) {
    return flow_time_step_full_ex(s_hs, s, d_C, d_u, d_v, d_w, d_phs, d_pnh, rho_l, rho_g, mu_l, mu_g, grav, sigma_t, dt, tol, max_cycles,
                                  hs_tol, hs_cycles, walls, 0, cycles_out, relres_out);
}

int flow_time_step_full_ex(mg_solver* s_hs, mg_solver* s, void* d_C, void* d_u, void* d_v, void* d_w, void* d_phs, void* d_pnh,
                           double rho_l, double rho_g, double mu_l, double mu_g, double grav, double sigma_t, double dt, double tol,
                           int max_cycles, double hs_tol, int hs_cycles, const int walls[6], int pressure_solver, int* cycles_out,
                           double* relres_out) {
    if (pressure_solver != 0 && pressure_solver != 1) { set_error("flow_time_step_full_ex: pressure_solver %d is not 0 (cycles) or 1 (PCG)", pressure_solver); return MG_EINVAL; }
    if (!s || !s_hs || !d_C || !d_u || !d_v || !d_w || !d_phs || !d_pnh || !walls) { set_error("flow_time_step_full: NULL argument"); return MG_EINVAL; }
    if (s_hs->dtype != s->dtype || s_hs->grid.nx != s->grid.nx || s_hs->grid.ny != s->grid.ny || s_hs->grid.nz != s->grid.nz ||
        s_hs->grid.hx != s->grid.hx || s_hs->device != s->device || s_hs->st != s->st || s_hs->var_k) {
        set_error("flow_time_step_full: the two solvers need the same grid, dtype, device and stream, and s_hs a constant coefficient");
        return MG_EINVAL;
    }
    int vbc[18];
    for (int c = 0; c < 3; ++c)
        for (int f = 0; f < 6; ++f) vbc[6 * c + f] = (walls[f] && f / 2 == c) ? MG_BC_DIRICHLET : MG_BC_NEUMANN;
    int prev = -1;
    cudaGetDevice(&prev);
    cudaSetDevice(s->device);
    const size_t n = s->lv[0].n, es = s->dtype == MG_F64 ? 8 : 4, bytes = n * es;
    cudaStream_t st = s->st;
    int rc = 0;
    {
        Scratch ws(st), ws2(st), ws3(st);
        if ((rc = ws.alloc(4, bytes)) || (rc = ws2.alloc(4, bytes)) || (rc = ws3.alloc(3, bytes))) { if (prev >= 0) cudaSetDevice(prev); return rc; }
        void* qt[3] = {ws.p[0], ws.p[1], ws.p[2]};
        void* qh[3] = {ws2.p[0], ws2.p[1], ws2.p[2]};
        void* force[3] = {ws3.p[0], ws3.p[1], ws3.p[2]};
        void* bbuf = ws.p[3];
        void* dp = ws2.p[3];
        const void* qn[3] = {d_u, d_v, d_w};
        const void* fc[3] = {force[0], force[1], force[2]};
        int status = 0;
        // stage 1
        rc = hydrostatic_rhs_force(&s->grid, s->dtype, d_C, rho_l, rho_g, grav, sigma_t, bbuf, nullptr, force, st);
        if (!rc) rc = cudaMemsetAsync(d_phs, 0, bytes, st) == cudaSuccess ? 0 : MG_ECUDA;
        if (!rc) { status = mg_solve(s_hs, d_phs, bbuf, hs_tol, hs_cycles, nullptr, nullptr); if (status < 0) rc = status; }
        // stage 2
        if (!rc) rc = mom_predictor_bc(&s->grid, s->dtype, d_C, qn, qn, vbc, rho_l, rho_g, mu_l, mu_g, dt, qt, nullptr, st);
        if (!rc) rc = mom_forcing(&s->grid, s->dtype, d_C, d_phs, d_pnh, s->bc, grav, fc, rho_l, rho_g, dt, qt, qn, qh, st);
        if (!rc) { const void* qhc[3] = {qh[0], qh[1], qh[2]}; rc = mom_predictor_bc(&s->grid, s->dtype, d_C, qhc, qn, vbc, rho_l, rho_g, mu_l, mu_g, dt, qt, nullptr, st); }
        if (!rc) rc = mom_forcing(&s->grid, s->dtype, d_C, d_phs, d_pnh, s->bc, grav, fc, rho_l, rho_g, dt, qt, nullptr, nullptr, st);
        // stage 3
        if (!rc) rc = mg_set_coefficient_from_vof(s, d_C, rho_l, rho_g);
        if (!rc) rc = pressure_rhs_bc(&s->grid, s->dtype, qt[0], qt[1], qt[2], vbc, dt, bbuf, st);
        if (!rc) rc = cudaMemsetAsync(dp, 0, bytes, st) == cudaSuccess ? 0 : MG_ECUDA;
        if (!rc) {
            status = pressure_solver == 1 ? mg_pcg_solve(s, dp, bbuf, tol, max_cycles, cycles_out, relres_out)
                                          : mg_solve(s, dp, bbuf, tol, max_cycles, cycles_out, relres_out);
            if (status < 0) rc = status;
        }
        if (!rc) rc = project_velocity(&s->grid, s->bc, s->dtype, dp, s->lv[0].k, dt, qt[0], qt[1], qt[2], st);
        if (!rc) rc = s->dtype == MG_F32 ? launch_axpy<float>(n, (float*)d_pnh, (const float*)dp, st)
                                         : launch_axpy<double>(n, (double*)d_pnh, (const double*)dp, st);
        // stage 4
        if (!rc) rc = vof_residual(&s->grid, s->dtype, d_C, qt[0], qt[1], qt[2], dt, nullptr, bbuf, st);
        if (!rc) {
            cudaMemcpyAsync(d_C, bbuf, bytes, cudaMemcpyDeviceToDevice, st);
            cudaMemcpyAsync(d_u, qt[0], bytes, cudaMemcpyDeviceToDevice, st);
            cudaMemcpyAsync(d_v, qt[1], bytes, cudaMemcpyDeviceToDevice, st);
            cudaMemcpyAsync(d_w, qt[2], bytes, cudaMemcpyDeviceToDevice, st);
            if (cudaGetLastError() != cudaSuccess) { set_error("flow_time_step_full: copy failed"); rc = MG_ECUDA; }
        }
        if (!rc) rc = status;
    }
    if (prev >= 0) cudaSetDevice(prev);
    return rc;
}

// Time step with the PAPER'S stage 3 (oracle time_step_paper): constant-coefficient Laplacian, density on the
// right (Eqs. 52-53), `cycles` multigrid cycles per solve from a zero guess (the paper's fixed 20), correction Eq. 54,
// the stage repeated `passes` times (twice); d_p receives the accumulated p_nh.  The solver's coefficient is reset to
// constant.  relres_out: relative residual of the last solve.
int flow_time_step_paper(mg_solver* s, void* d_C, void* d_u, void* d_v, void* d_w, void* d_p, double rho_l, double rho_g, double mu_l,
                         double mu_g, double dt, int cycles, int passes, double* relres_out) {
    if (!s || !d_C || !d_u || !d_v || !d_w || !d_p || cycles < 1 || passes < 1) { set_error("flow_time_step_paper: invalid argument"); return MG_EINVAL; }
    int prev = -1;
    cudaGetDevice(&prev);
    cudaSetDevice(s->device);
    const size_t n = s->lv[0].n, es = s->dtype == MG_F64 ? 8 : 4, bytes = n * es;
    cudaStream_t st = s->st;
    int rc = 0;
    {
        Scratch ws(st), ws2(st);
        if ((rc = ws.alloc(4, bytes)) || (rc = ws2.alloc(4, bytes))) { if (prev >= 0) cudaSetDevice(prev); return rc; }
        void* qt[3] = {ws.p[0], ws.p[1], ws.p[2]};
        void* qh[3] = {ws2.p[0], ws2.p[1], ws2.p[2]};
        void* bbuf = ws.p[3];
        void* kbuf = ws2.p[3];
        void* dp = qh[0];                       // the half-level velocities are dead after stage 2
        const void* qn[3] = {d_u, d_v, d_w};
        rc = mom_predictor(&s->grid, s->dtype, d_C, qn, qn, rho_l, rho_g, mu_l, mu_g, dt, qt, qh, st);
        if (!rc) { const void* qhc[3] = {qh[0], qh[1], qh[2]}; rc = mom_predictor(&s->grid, s->dtype, d_C, qhc, qn, rho_l, rho_g, mu_l, mu_g, dt, qt, nullptr, st); }
        if (!rc && s->var_k) rc = mg_set_coefficient(s, nullptr);
        if (!rc) rc = s->dtype == MG_F32 ? launch_k_from_vof<float>(n, (const float*)d_C, rho_l, rho_g, (float*)kbuf, st)
                                         : launch_k_from_vof<double>(n, (const double*)d_C, rho_l, rho_g, (double*)kbuf, st);
        if (!rc) rc = cudaMemsetAsync(d_p, 0, bytes, st) == cudaSuccess ? 0 : MG_ECUDA;
        for (int pass = 0; pass < passes && !rc; ++pass) {
            rc = pressure_rhs_paper(&s->grid, s->dtype, d_C, qt[0], qt[1], qt[2], rho_l, rho_g, dt, bbuf, st);
            if (!rc) rc = cudaMemsetAsync(dp, 0, bytes, st) == cudaSuccess ? 0 : MG_ECUDA;
            if (!rc) { const int status = mg_solve(s, dp, bbuf, 0.0, cycles, nullptr, relres_out); if (status < 0) rc = status; }
            if (!rc) rc = project_velocity(&s->grid, s->bc, s->dtype, dp, kbuf, dt, qt[0], qt[1], qt[2], st);
            if (!rc) rc = s->dtype == MG_F32 ? launch_axpy<float>(n, (float*)d_p, (const float*)dp, st)
                                             : launch_axpy<double>(n, (double*)d_p, (const double*)dp, st);
        }
        if (!rc) rc = vof_residual(&s->grid, s->dtype, d_C, qt[0], qt[1], qt[2], dt, nullptr, bbuf, st);
        if (!rc) {
            cudaMemcpyAsync(d_C, bbuf, bytes, cudaMemcpyDeviceToDevice, st);
            cudaMemcpyAsync(d_u, qt[0], bytes, cudaMemcpyDeviceToDevice, st);
            cudaMemcpyAsync(d_v, qt[1], bytes, cudaMemcpyDeviceToDevice, st);
            cudaMemcpyAsync(d_w, qt[2], bytes, cudaMemcpyDeviceToDevice, st);
            if (cudaGetLastError() != cudaSuccess) { set_error("flow_time_step_paper: copy failed"); rc = MG_ECUDA; }
        }
    }
    if (prev >= 0) cudaSetDevice(prev);
    return rc;
}

}  // extern "C"
