// tu_recompute_mix.cu -- instantiations and launcher of the mixture form of k_nll_recompute (kernels.cuh); see launch.h
#include "launch.h"
#include "kernels.cuh"

cudaError_t mipwa_launch_nll_recompute_mix(const int* n_spin, int fl, int grid, cudaStream_t st, const DevModel& m,
                                           const PointRec* ev, double kappa, long long n_ev, const PointRec* nm,
                                           long long n_norm, double2* partials, unsigned int* ticket, double* result,
                                           long long tag, const double* integral_src)
{
    MIPWA_DISPATCH_SIGFL(n_spin[0], n_spin[1], n_spin[2], fl,
                         (k_nll_recompute<R1, R2, FL, true><<<grid, MIPWA_REC_BLOCK, 0, st>>>(
                             m, ev, kappa, n_ev, nm, n_norm, partials, ticket, result, tag, integral_src)));
    return cudaGetLastError();
}
