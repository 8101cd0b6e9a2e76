// tu_grad.cu -- instantiations and launchers of k_grad_recompute (grad.cuh); see launch.h
#include "launch.h"
#include "kernels.cuh"
#include "grad.cuh"

cudaError_t mipwa_occupancy_grad_recompute(const int* n_spin, int fl, size_t smem, int* blocks_per_sm)
{
    cudaError_t e = cudaSuccess;
    MIPWA_DISPATCH_SIGFL(n_spin[0], n_spin[1], n_spin[2], fl,
                         e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(blocks_per_sm, k_grad_recompute<R1, R2, FL, false>,
                                                                           MIPWA_GRAD_BLOCK, smem));
    return e;
}

cudaError_t mipwa_launch_grad_recompute(const int* n_spin, int fl, int grid, size_t smem, cudaStream_t st,
                                        const DevModel& m, const double* e12, const double* e13,
                                        const unsigned short* eseg, const double* eb, double kappa, long long n_ev,
                                        const double* g12,
                                        const double* g13, const double* gw, const unsigned short* gseg,
                                        long long n_norm, double* partials, double2* f_ev, double2* f_nm)
{
    if (eb)
        return mipwa_launch_grad_recompute_mix(n_spin, fl, grid, smem, st, m, e12, e13, eseg, eb, kappa, n_ev, g12, g13, gw,
                                               gseg, n_norm, partials);
    MIPWA_DISPATCH_SIGFL(n_spin[0], n_spin[1], n_spin[2], fl,
                         (k_grad_recompute<R1, R2, FL, false><<<grid, MIPWA_GRAD_BLOCK, smem, st>>>(
                             m, e12, e13, eseg, nullptr, 0.0, n_ev, g12, g13, gw, gseg, n_norm, partials, f_ev, f_nm)));
    return cudaGetLastError();
}
