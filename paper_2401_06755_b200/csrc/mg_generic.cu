// mg_generic.cu -- generic one-point-per-thread kernels of the multigrid path: any spacing
// (all 27 weights), any boundary mix, fp32 and fp64, one sweep per pass.  They are the path for
// anisotropic grids, for fp64, for mg_apply_operator / mg_residual, and the un-fused comparison
// path (mg_set_fused(s, 0)); the tuned uniform-grid fp32 kernels live in mg_fused.cu.
//
// Operator (reading C1/C2; Eqs. 8, 12-13):
//   constant k:  (A x)_i = sum_j w_ij x_j
//   variable k:  (A x)_i = sum_{j != i} (-w_ij) 1/2 (k_i + k_j) (x_i - x_j)   [Eq. 13 collapsed, sum_j w_ij = 0]
//   D_i = sum_{j != i} (-w_ij) 1/2 (k_i + k_j)   (constant k: w_000)
// Halo: ghost(x) = s_face * x(mirror), factors multiply at edges/corners; ghost(k) = k(mirror).
#include "common.cuh"

namespace mgb {

namespace {

template <typename T>
__device__ __forceinline__ void mirror3(int c, int n, T s_lo, T s_hi, int idx[3], T fac[3]) {
    idx[1] = c; fac[1] = T(1);
    if (c > 0) { idx[0] = c - 1; fac[0] = T(1); } else { idx[0] = 0; fac[0] = s_lo; }
    if (c < n - 1) { idx[2] = c + 1; fac[2] = T(1); } else { idx[2] = n - 1; fac[2] = s_hi; }
}

// Ax and D at point (i, j, kz).  TX is the type of x (double in the mixed-precision residual).
template <typename T, bool VAR>
__device__ __forceinline__ void stencil_point(const Level<T>& L, const T* __restrict__ kc, const T* __restrict__ x,
                                              int i, int j, int kz, T& Ax, T& D) {
    int ix[3], jy[3], kk[3];
    T fx[3], fy[3], fz[3];
    mirror3<T>(i, L.nx, L.s[0], L.s[1], ix, fx);
    mirror3<T>(j, L.ny, L.s[2], L.s[3], jy, fy);
    mirror3<T>(kz, L.nz, L.s[4], L.s[5], kk, fz);
    const size_t c0 = (size_t)i + (size_t)L.nx * ((size_t)j + (size_t)L.ny * kz);
    const T xi = x[c0];
    T ax = T(0), d = T(0);
    if (VAR) {
        const T ki = kc[c0];
#pragma unroll
        for (int c = 0; c < 3; ++c)
#pragma unroll
            for (int b = 0; b < 3; ++b) {
                const size_t row = (size_t)L.nx * ((size_t)jy[b] + (size_t)L.ny * kk[c]);
                const T fyz = fy[b] * fz[c];
#pragma unroll
                for (int a = 0; a < 3; ++a) {
                    if (a == 1 && b == 1 && c == 1) continue;
                    const T xj = fx[a] * fyz * x[row + ix[a]];
                    const T kj = kc[row + ix[a]];
                    const T cw = T(-0.5) * L.w[a + 3 * b + 9 * c] * (ki + kj);
                    ax += cw * (xi - xj);
                    d += cw;
                }
            }
    } else {
#pragma unroll
        for (int c = 0; c < 3; ++c)
#pragma unroll
            for (int b = 0; b < 3; ++b) {
                const size_t row = (size_t)L.nx * ((size_t)jy[b] + (size_t)L.ny * kk[c]);
                const T fyz = fy[b] * fz[c];
#pragma unroll
                for (int a = 0; a < 3; ++a) ax += L.w[a + 3 * b + 9 * c] * (fx[a] * fyz * x[row + ix[a]]);
            }
        d = L.w[13];
    }
    Ax = ax; D = d;
}

constexpr int BX = 64, BY = 4;

template <typename T>
inline dim3 grid_for(const Level<T>& L) { return dim3((L.nx + BX - 1) / BX, (L.ny + BY - 1) / BY, L.nz); }

// mode 0: y = A x;  1: y = x + omega (b - A x)/D;  2: y = b - A x
template <typename T, bool VAR, int MODE>
__global__ void __launch_bounds__(BX* BY) point_kernel(const Level<T> L, const T* __restrict__ kc, const T* __restrict__ x,
                                                      const T* __restrict__ b, T* __restrict__ y) {
    const int i = blockIdx.x * BX + threadIdx.x, j = blockIdx.y * BY + threadIdx.y, kz = blockIdx.z;
    if (i >= L.nx || j >= L.ny) return;
    T Ax, D;
    stencil_point<T, VAR>(L, kc, x, i, j, kz, Ax, D);
    const size_t c0 = (size_t)i + (size_t)L.nx * ((size_t)j + (size_t)L.ny * kz);
    if (MODE == 0) y[c0] = Ax;
    else if (MODE == 1) y[c0] = x[c0] + L.omega * (b[c0] - Ax) / D;
    else y[c0] = b[c0] - Ax;
}

__device__ __forceinline__ double block_sum(double v) {
    __shared__ double red[32];
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    const int tid = threadIdx.x + blockDim.x * (threadIdx.y + blockDim.y * threadIdx.z);
    const int nw = (blockDim.x * blockDim.y * blockDim.z + 31) / 32;
    if ((tid & 31) == 0) red[tid >> 5] = v;
    __syncthreads();
    if (tid < 32) {
        v = tid < nw ? red[tid] : 0.0;
        for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    }
    return v;  // valid in thread 0
}

template <typename T, bool VAR>
__global__ void __launch_bounds__(BX* BY) residual_norm_kernel(const Level<T> L, const T* __restrict__ kc,
                                                              const T* __restrict__ x, const T* __restrict__ b,
                                                              T* __restrict__ r, double* __restrict__ acc) {
    const int i = blockIdx.x * BX + threadIdx.x, j = blockIdx.y * BY + threadIdx.y, kz = blockIdx.z;
    double sq = 0.0;
    if (i < L.nx && j < L.ny) {
        T Ax, D;
        stencil_point<T, VAR>(L, kc, x, i, j, kz, Ax, D);
        const size_t c0 = (size_t)i + (size_t)L.nx * ((size_t)j + (size_t)L.ny * kz);
        const T rr = b[c0] - Ax;
        if (r) r[c0] = rr;
        sq = (double)rr * (double)rr;
    }
    sq = block_sum(sq);
    if (threadIdx.x == 0 && threadIdx.y == 0) atomicAdd(acc, sq);
}

// Mixed precision: fp64 operator on the fp64 iterate, fp32 right-hand side, fp32 residual out.
template <bool VAR>
__global__ void __launch_bounds__(BX* BY) residual_mixed_kernel(const Level<double> L, const double* __restrict__ kc,
                                                               const double* __restrict__ x, const float* __restrict__ b,
                                                               float* __restrict__ r, double* __restrict__ acc) {
    const int i = blockIdx.x * BX + threadIdx.x, j = blockIdx.y * BY + threadIdx.y, kz = blockIdx.z;
    double sq = 0.0;
    if (i < L.nx && j < L.ny) {
        double Ax, D;
        stencil_point<double, VAR>(L, kc, x, i, j, kz, Ax, D);
        const size_t c0 = (size_t)i + (size_t)L.nx * ((size_t)j + (size_t)L.ny * kz);
        const double rr = (double)b[c0] - Ax;
        r[c0] = (float)rr;
        sq = rr * rr;
    }
    sq = block_sum(sq);
    if (threadIdx.x == 0 && threadIdx.y == 0) atomicAdd(acc, sq);
}

// restriction = mean of the 8 children; prolongation = piecewise constant (reading C5, Fig. 5)
template <typename T>
__global__ void restrict_kernel(int nxc, int nyc, int nzc, const T* __restrict__ f, T* __restrict__ c) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y * blockDim.y + threadIdx.y, k = blockIdx.z;
    if (i >= nxc || j >= nyc) return;
    const size_t nxf = 2 * (size_t)nxc, nyf = 2 * (size_t)nyc;
    T s = T(0);
#pragma unroll
    for (int dk = 0; dk < 2; ++dk)
#pragma unroll
        for (int dj = 0; dj < 2; ++dj) {
            const size_t row = nxf * ((2 * j + dj) + nyf * (size_t)(2 * k + dk)) + 2 * i;
            s += f[row] + f[row + 1];
        }
    c[(size_t)i + (size_t)nxc * (j + (size_t)nyc * k)] = T(0.125) * s;
}

template <typename T>
__global__ void prolong_add_kernel(int nxf, int nyf, int nzf, const T* __restrict__ xc, T* __restrict__ xf) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y * blockDim.y + threadIdx.y, k = blockIdx.z;
    if (i >= nxf || j >= nyf) return;
    const size_t nxc = nxf / 2, nyc = nyf / 2;
    xf[(size_t)i + (size_t)nxf * (j + (size_t)nyf * k)] += xc[(i >> 1) + nxc * ((j >> 1) + nyc * (size_t)(k >> 1))];
}

template <typename TA, typename TK>
__global__ void k_from_vof_kernel(size_t n, const TA* __restrict__ alpha, double rho_l, double rho_g, TK* __restrict__ k) {
    for (size_t c = blockIdx.x * (size_t)blockDim.x + threadIdx.x; c < n; c += (size_t)gridDim.x * blockDim.x) {
        TK a = (TK)alpha[c];
        a = a < TK(0) ? TK(0) : (a > TK(1) ? TK(1) : a);          // reading C11: rho from the volume fraction limited to [0, 1]
        k[c] = TK(1) / ((TK)rho_l * a + (TK)rho_g * (TK(1) - a));
    }
}

template <typename T>
__global__ void sumsq_kernel(size_t n, const T* __restrict__ v, double* __restrict__ acc) {
    double s = 0.0;
    for (size_t c = blockIdx.x * (size_t)blockDim.x + threadIdx.x; c < n; c += (size_t)gridDim.x * blockDim.x) {
        const double t = (double)v[c];
        s += t * t;
    }
    s = block_sum(s);
    if (threadIdx.x == 0) atomicAdd(acc, s);
}

template <typename TA, typename TB>
__global__ void cast_kernel(size_t n, const TA* __restrict__ a, TB* __restrict__ b) {
    for (size_t c = blockIdx.x * (size_t)blockDim.x + threadIdx.x; c < n; c += (size_t)gridDim.x * blockDim.x)
        b[c] = (TB)a[c];
}

__global__ void axpy_mixed_kernel(size_t n, double* __restrict__ x, const float* __restrict__ e) {
    for (size_t c = blockIdx.x * (size_t)blockDim.x + threadIdx.x; c < n; c += (size_t)gridDim.x * blockDim.x)
        x[c] += (double)e[c];
}

inline int ew_blocks(size_t n) {
    size_t b = (n + 255) / 256;
    const size_t cap = (size_t)sm_count() * 16;
    return (int)(b < cap ? (b ? b : 1) : cap);
}

}  // namespace

template <typename T>
int launch_apply(const Level<T>& L, const T* k, const T* x, T* y, cudaStream_t st) {
    if (k) point_kernel<T, true, 0><<<grid_for(L), dim3(BX, BY), 0, st>>>(L, k, x, nullptr, y);
    else point_kernel<T, false, 0><<<grid_for(L), dim3(BX, BY), 0, st>>>(L, k, x, nullptr, y);
    MGB_LAUNCH_CHECK();
    return 0;
}

template <typename T>
int launch_jacobi(const Level<T>& L, const T* k, const T* x, const T* b, T* xnew, cudaStream_t st) {
    if (k) point_kernel<T, true, 1><<<grid_for(L), dim3(BX, BY), 0, st>>>(L, k, x, b, xnew);
    else point_kernel<T, false, 1><<<grid_for(L), dim3(BX, BY), 0, st>>>(L, k, x, b, xnew);
    MGB_LAUNCH_CHECK();
    return 0;
}

template <typename T>
int launch_residual(const Level<T>& L, const T* k, const T* x, const T* b, T* r, cudaStream_t st) {
    if (k) point_kernel<T, true, 2><<<grid_for(L), dim3(BX, BY), 0, st>>>(L, k, x, b, r);
    else point_kernel<T, false, 2><<<grid_for(L), dim3(BX, BY), 0, st>>>(L, k, x, b, r);
    MGB_LAUNCH_CHECK();
    return 0;
}

template <typename T>
int launch_residual_norm(const Level<T>& L, const T* k, const T* x, const T* b, T* r, double* d_acc, cudaStream_t st) {
    if (k) residual_norm_kernel<T, true><<<grid_for(L), dim3(BX, BY), 0, st>>>(L, k, x, b, r, d_acc);
    else residual_norm_kernel<T, false><<<grid_for(L), dim3(BX, BY), 0, st>>>(L, k, x, b, r, d_acc);
    MGB_LAUNCH_CHECK();
    return 0;
}

int launch_residual_mixed(const Level<double>& L, const double* k64, const double* x64, const float* b32, float* r32,
                          double* d_acc, cudaStream_t st) {
    if (k64) residual_mixed_kernel<true><<<grid_for(L), dim3(BX, BY), 0, st>>>(L, k64, x64, b32, r32, d_acc);
    else residual_mixed_kernel<false><<<grid_for(L), dim3(BX, BY), 0, st>>>(L, k64, x64, b32, r32, d_acc);
    MGB_LAUNCH_CHECK();
    return 0;
}

template <typename T>
int launch_restrict(int nxc, int nyc, int nzc, const T* fine, T* coarse, cudaStream_t st) {
    dim3 blk(32, 4), grd((nxc + 31) / 32, (nyc + 3) / 4, nzc);
    restrict_kernel<T><<<grd, blk, 0, st>>>(nxc, nyc, nzc, fine, coarse);
    MGB_LAUNCH_CHECK();
    return 0;
}

template <typename T>
int launch_prolong_add(int nxf, int nyf, int nzf, const T* xc, T* xf, cudaStream_t st) {
    dim3 blk(64, 4), grd((nxf + 63) / 64, (nyf + 3) / 4, nzf);
    prolong_add_kernel<T><<<grd, blk, 0, st>>>(nxf, nyf, nzf, xc, xf);
    MGB_LAUNCH_CHECK();
    return 0;
}

template <typename T>
int launch_k_from_vof(size_t n, const T* alpha, double rho_l, double rho_g, T* k, cudaStream_t st) {
    k_from_vof_kernel<T, T><<<ew_blocks(n), 256, 0, st>>>(n, alpha, rho_l, rho_g, k);
    MGB_LAUNCH_CHECK();
    return 0;
}

int launch_k64_from_vof(size_t n, const float* alpha, double rho_l, double rho_g, double* k64, cudaStream_t st) {
    k_from_vof_kernel<float, double><<<ew_blocks(n), 256, 0, st>>>(n, alpha, rho_l, rho_g, k64);
    MGB_LAUNCH_CHECK();
    return 0;
}

template <typename T>
int launch_sumsq(size_t n, const T* v, double* d_acc, cudaStream_t st) {
    sumsq_kernel<T><<<ew_blocks(n), 256, 0, st>>>(n, v, d_acc);
    MGB_LAUNCH_CHECK();
    return 0;
}

namespace {
__global__ void record_acc_kernel(double* acc0, double* hist, int* ctr) {
    hist[*ctr] = *acc0;
    *acc0 = 0.0;
    *ctr += 1;
}
}  // namespace
int launch_record_acc(double* acc0, double* hist, int* ctr, cudaStream_t st) {
    record_acc_kernel<<<1, 1, 0, st>>>(acc0, hist, ctr);
    MGB_LAUNCH_CHECK();
    return 0;
}
int launch_axpy_mixed(size_t n, double* x64, const float* e32, cudaStream_t st) {
    axpy_mixed_kernel<<<ew_blocks(n), 256, 0, st>>>(n, x64, e32);
    MGB_LAUNCH_CHECK();
    return 0;
}
int launch_cast_f2d(size_t n, const float* a, double* b, cudaStream_t st) {
    cast_kernel<float, double><<<ew_blocks(n), 256, 0, st>>>(n, a, b);
    MGB_LAUNCH_CHECK();
    return 0;
}
int launch_cast_d2f(size_t n, const double* a, float* b, cudaStream_t st) {
    cast_kernel<double, float><<<ew_blocks(n), 256, 0, st>>>(n, a, b);
    MGB_LAUNCH_CHECK();
    return 0;
}

#define INSTANTIATE(T)                                                                                        \
    template int launch_apply<T>(const Level<T>&, const T*, const T*, T*, cudaStream_t);                      \
    template int launch_jacobi<T>(const Level<T>&, const T*, const T*, const T*, T*, cudaStream_t);           \
    template int launch_residual<T>(const Level<T>&, const T*, const T*, const T*, T*, cudaStream_t);         \
    template int launch_residual_norm<T>(const Level<T>&, const T*, const T*, const T*, T*, double*, cudaStream_t); \
    template int launch_restrict<T>(int, int, int, const T*, T*, cudaStream_t);                               \
    template int launch_prolong_add<T>(int, int, int, const T*, T*, cudaStream_t);                            \
    template int launch_k_from_vof<T>(size_t, const T*, double, double, T*, cudaStream_t);                    \
    template int launch_sumsq<T>(size_t, const T*, double*, cudaStream_t);
INSTANTIATE(float)
INSTANTIATE(double)

}  // namespace mgb
