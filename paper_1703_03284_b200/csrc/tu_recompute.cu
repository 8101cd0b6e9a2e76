// tu_recompute.cu -- instantiations and launchers of k_nll_recompute (kernels.cuh); see launch.h
#include "launch.h"
#include "kernels.cuh"

cudaError_t mipwa_launch_nll_recompute(const int* n_spin, int fl, bool mix, int grid, cudaStream_t st, const DevModel& m,
                                       const PointRec* ev, double kappa, long long n_ev, const PointRec* nm,
                                       long long n_norm, double2* partials, unsigned int* ticket, double* result,
                                       long long tag)
{
    if (mix)
        return mipwa_launch_nll_recompute_mix(n_spin, fl, grid, st, m, ev, kappa, n_ev, nm, n_norm, partials, ticket,
                                              result, tag);
    MIPWA_DISPATCH_SIGFL(n_spin[0], n_spin[1], n_spin[2], fl,
                         (k_nll_recompute<R1, R2, FL, false><<<grid, MIPWA_REC_BLOCK, 0, st>>>(
                             m, ev, 0.0, n_ev, nm, n_norm, partials, ticket, result, tag)));
    return cudaGetLastError();
}
