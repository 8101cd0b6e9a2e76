// tu_grad_mix.cu -- instantiations and launcher of the mixture form of k_grad_recompute (grad.cuh); see launch.h
#include "launch.h"
#include "kernels.cuh"
#include "grad.cuh"

cudaError_t mipwa_grad_set_smem_mix(const int* n_spin, int fl, size_t smem)
{
    cudaError_t e = cudaSuccess;
    MIPWA_DISPATCH_SIGFL(n_spin[0], n_spin[1], n_spin[2], fl,
                         (e = cudaFuncSetAttribute(k_grad_recompute<R1, R2, FL, true, 0>,
                                                   cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem)));
    return e;
}

cudaError_t mipwa_launch_grad_recompute_mix(const int* n_spin, int fl, int grid, int ev_blocks, size_t smem,
                                            cudaStream_t st, const DevModel& m, const PointRec* ev, double kappa,
                                            long long n_ev, const PointRec* nm, long long n_norm, double* partials)
{
    MIPWA_DISPATCH_SIGFL(n_spin[0], n_spin[1], n_spin[2], fl,
                         (k_grad_recompute<R1, R2, FL, true, 0><<<grid, MIPWA_GRAD_BLOCK, smem, st>>>(
                             m, ev, kappa, n_ev, nm, n_norm, ev_blocks, partials, nullptr, nullptr)));
    return cudaGetLastError();
}
