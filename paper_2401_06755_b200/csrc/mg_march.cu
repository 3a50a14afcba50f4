// mg_march.cu -- host side of the z-marching residual kernel (march_kernel.cuh).
#include "march_kernel.cuh"
#include "solver.h"

namespace mgb {

bool march_supported(int nx, int ny, int nz, double hx, double hy, double hz) {
    return hx == hy && hy == hz && nx % 4 == 0 && nx >= 4 && ny >= 1 && nz >= 1;
}

template <typename TXT, typename TB>
int launch_march_residual(int nx, int ny, int nz, double h, const double s[6], const TXT* x, const TXT* k, const TB* b, TB* r,
                          double* acc, cudaStream_t st, int dotx, float* yout) {
    mk::MParams P;
    P.nx = nx; P.ny = ny; P.nz = nz;
    for (int f = 0; f < 6; ++f) P.s[f] = s[f];
    P.cc = 1.0 / (24.0 * h * h);
    P.dotx = dotx;
    const int tx = (nx + mk::TX - 1) / mk::TX, ty = (ny + mk::TY - 1) / mk::TY;
    // z chunks: one wave of resident blocks; every chunk pays 2 extra planes
    const size_t smem = (size_t)2 * mk::NSTG * mk::Lay<TXT>::ROW * mk::PYS * sizeof(TXT) + (size_t)mk::NBS * mk::NT * 4 * sizeof(TB);
    int per_sm = 1, rc0;
    if ((rc0 = kernel_setup((const void*)mk::march_residual_kernel<TXT, TB, true, true>, mk::NT, smem, &per_sm))) return rc0;
    if ((rc0 = kernel_setup((const void*)mk::march_residual_kernel<TXT, TB, false, true>, mk::NT, smem, nullptr))) return rc0;
    if ((rc0 = kernel_setup((const void*)mk::march_residual_kernel<TXT, TB, true, false>, mk::NT, smem, nullptr))) return rc0;
    if ((rc0 = kernel_setup((const void*)mk::march_residual_kernel<TXT, TB, false, false>, mk::NT, smem, nullptr))) return rc0;
    const int want = (sm_count() * per_sm) / (tx * ty);
    const int nch = want < 1 ? 1 : (want > nz ? nz : want);
    P.zchunk = (nz + nch - 1) / nch;
    const dim3 grid(tx, ty, (nz + P.zchunk - 1) / P.zchunk);
    if (b && dotx) { set_error("march residual: dotx needs b == NULL"); return MG_EINVAL; }
    if (k && b) mk::march_residual_kernel<TXT, TB, true, true><<<grid, mk::NT, smem, st>>>(P, x, k, b, r, acc, yout);
    else if (k) mk::march_residual_kernel<TXT, TB, true, false><<<grid, mk::NT, smem, st>>>(P, x, k, b, r, acc, yout);
    else if (b) mk::march_residual_kernel<TXT, TB, false, true><<<grid, mk::NT, smem, st>>>(P, x, k, b, r, acc, yout);
    else mk::march_residual_kernel<TXT, TB, false, false><<<grid, mk::NT, smem, st>>>(P, x, k, b, r, acc, yout);
    MGB_LAUNCH_CHECK();
    return 0;
}

template int launch_march_residual<double, float>(int, int, int, double, const double*, const double*, const double*, const float*, float*, double*, cudaStream_t, int, float*);
template int launch_march_residual<double, double>(int, int, int, double, const double*, const double*, const double*, const double*, double*, double*, cudaStream_t, int, float*);
template int launch_march_residual<float, float>(int, int, int, double, const double*, const float*, const float*, const float*, float*, double*, cudaStream_t, int, float*);

}  // namespace mgb
