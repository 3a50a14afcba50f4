// common.cuh -- shared declarations of the libmg_b200 CUDA sources (product code; never
// included by, and never including, anything under oracle/).
#pragma once
#include <cuda_runtime.h>
#include <cstdint>
#include <cstdio>

namespace mgb {

// Thread-local error text behind mg_last_error().
void set_error(const char* fmt, ...);

#define MGB_CUDA(call)                                                                         \
    do {                                                                                       \
        cudaError_t e_ = (call);                                                               \
        if (e_ != cudaSuccess) {                                                               \
            ::mgb::set_error("%s:%d: %s -> %s", __FILE__, __LINE__, #call, cudaGetErrorString(e_)); \
            return -3; /* MG_ECUDA */                                                          \
        }                                                                                      \
    } while (0)

#define MGB_LAUNCH_CHECK() MGB_CUDA(cudaGetLastError())

// Geometry + stencil of one multigrid level, passed to kernels by value.
//   w[27]: nodal 27-point filter of -Laplace, index (ii+1) + 3*(jj+1) + 9*(kk+1), ii along x
//          (trilinear FE: (K M M + M K M + M M K)/m_l; Eqs. 8, 11 P:109-138, reading C1).
//   s[6]:  halo factors ghost = s * mirror for x-, x+, y-, y+, z-, z+ (reading C3).
template <typename T>
struct Level {
    int nx, ny, nz;
    T w[27];
    T s[6];
    T omega;
};

struct Dim3i { int nx, ny, nz; };

inline __host__ __device__ size_t npts(int nx, int ny, int nz) { return (size_t)nx * ny * nz; }

// Per-device facts and one-time kernel set-up (mg_api.cu).  Both are keyed by the CURRENT device and thread-safe:
// cudaFuncSetAttribute and the occupancy query apply per device, so a process-wide "done" flag would leave a second GPU
// of the same process without its opt-in to > 48 KB of dynamic shared memory.
int sm_count();                                                   // multiprocessors of the current device
// opt-in to `smem` bytes of dynamic shared memory (+ the maximum shared-memory carve-out if asked: the TMA-ring kernels want
// it, the cp.async marching kernels lose a third of their speed without L1) and the resident blocks per SM
int kernel_setup(const void* fn, int threads, size_t smem, int* ctas_per_sm, bool max_carveout = false);

// ---- launchers of the generic (any spacing, any BC, one sweep per pass) kernels: mg_generic.cu
template <typename T> int launch_apply(const Level<T>& L, const T* k, const T* x, T* y, cudaStream_t st);
template <typename T> int launch_jacobi(const Level<T>& L, const T* k, const T* x, const T* b, T* xnew, cudaStream_t st);
template <typename T> int launch_residual(const Level<T>& L, const T* k, const T* x, const T* b, T* r, cudaStream_t st);
template <typename T> int launch_restrict(int nxc, int nyc, int nzc, const T* fine, T* coarse, cudaStream_t st);
template <typename T> int launch_prolong_add(int nxf, int nyf, int nzf, const T* xc, T* xf, cudaStream_t st);
template <typename T> int launch_k_from_vof(size_t n, const T* alpha, double rho_l, double rho_g, T* k, cudaStream_t st);
// sum of squares into *d_acc (fp64, must be zeroed by the caller on the same stream)
template <typename T> int launch_sumsq(size_t n, const T* v, double* d_acc, cudaStream_t st);
// ||b - A x||^2 accumulated into *d_acc without storing r (r may be NULL) or storing it
template <typename T> int launch_residual_norm(const Level<T>& L, const T* k, const T* x, const T* b, T* r, double* d_acc, cudaStream_t st);
// mixed precision outer loop: r32 = float(b32 - A64 x64), ||r||^2 into *d_acc
int launch_residual_mixed(const Level<double>& L, const double* k64, const double* x64, const float* b32, float* r32,
                          double* d_acc, cudaStream_t st);
// z-marching residual for uniform grids (march_kernel.cuh): r = b - A x (r may be NULL), ||r||^2 added to *acc (may be NULL)
bool march_supported(int nx, int ny, int nz, double hx, double hy, double hz);
template <typename TXT, typename TB>
int launch_march_residual(int nx, int ny, int nz, double h, const double s[6], const TXT* x, const TXT* k, const TB* b, TB* r,
                          double* acc, cudaStream_t st, int dotx = 0,    // dotx: accumulate sum out * x instead of sum out^2
                          float* yout = nullptr);   // yout: also store out / D (fp32), the Jacobi seed of a correction cycle
}  // namespace mgb
struct mg_solver;
namespace mgb {
int ensure_mixed_buffers(mg_solver* s);   // x64, k64, r32, e32 of the mixed-precision loops (mg_api.cu)
int vcycle_zero_guess(mg_solver* s, void* x, const void* b);   // V-cycle from x = 0; x need not be initialised (mg_api.cu)
int launch_axpy_mixed(size_t n, double* x64, const float* e32, cudaStream_t st);  // x64 += e32
int launch_record_acc(double* acc0, double* hist, int* ctr, cudaStream_t st);     // hist[(*ctr)++] = *acc0; *acc0 = 0
int launch_cast_f2d(size_t n, const float* a, double* b, cudaStream_t st);
int launch_cast_d2f(size_t n, const double* a, float* b, cudaStream_t st);
int launch_k64_from_vof(size_t n, const float* alpha, double rho_l, double rho_g, double* k64, cudaStream_t st);

}  // namespace mgb
