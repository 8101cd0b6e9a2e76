// tu_recompute.cu -- instantiations and launchers of k_nll_recompute (kernels.cuh); see launch.h
#include "launch.h"
#include "kernels.cuh"

cudaError_t mipwa_occupancy_nll_recompute(const int* n_spin, int fl, int* blocks_per_sm)
{
    cudaError_t e = cudaSuccess;
    MIPWA_DISPATCH_SIGFL(n_spin[0], n_spin[1], n_spin[2], fl,
                         e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(blocks_per_sm, k_nll_recompute<R1, R2, FL, false>,
                                                                           MIPWA_REC_BLOCK, 0));
    return e;
}

cudaError_t mipwa_launch_nll_recompute(const int* n_spin, int fl, int grid, cudaStream_t st, const DevModel& m,
                                       const double* e12, const double* e13, const unsigned short* eseg,
                                       const double* eb, double kappa, long long n_ev,
                                       const double* g12, const double* g13, const double* gw,
                                       const unsigned short* gseg, long long n_norm, double2* partials,
                                       unsigned int* ticket, double* result)
{
    if (eb)
        return mipwa_launch_nll_recompute_mix(n_spin, fl, grid, st, m, e12, e13, eseg, eb, kappa, n_ev, g12, g13, gw, gseg,
                                              n_norm, partials, ticket, result);
    MIPWA_DISPATCH_SIGFL(n_spin[0], n_spin[1], n_spin[2], fl,
                         (k_nll_recompute<R1, R2, FL, false><<<grid, MIPWA_REC_BLOCK, 0, st>>>(
                             m, e12, e13, eseg, nullptr, 0.0, n_ev, g12, g13, gw, gseg, n_norm, partials, ticket, result)));
    return cudaGetLastError();
}
