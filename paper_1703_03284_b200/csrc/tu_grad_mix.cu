// tu_grad_mix.cu -- instantiations and launcher of the mixture form of k_grad_recompute (grad.cuh); see launch.h
#include "launch.h"
#include "kernels.cuh"
#include "grad.cuh"

cudaError_t mipwa_launch_grad_recompute_mix(const int* n_spin, int fl, int grid, size_t smem, cudaStream_t st,
                                            const DevModel& m, const double* e12, const double* e13,
                                            const unsigned short* eseg, const double* eb, double kappa, long long n_ev,
                                            const double* g12, const double* g13, const double* gw,
                                            const unsigned short* gseg, long long n_norm, double* partials)
{
    MIPWA_DISPATCH_SIGFL(n_spin[0], n_spin[1], n_spin[2], fl,
                         (k_grad_recompute<R1, R2, FL, true><<<grid, MIPWA_GRAD_BLOCK, smem, st>>>(
                             m, e12, e13, eseg, eb, kappa, n_ev, g12, g13, gw, gseg, n_norm, partials, nullptr, nullptr)));
    return cudaGetLastError();
}
