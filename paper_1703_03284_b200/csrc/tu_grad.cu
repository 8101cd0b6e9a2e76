// tu_grad.cu -- instantiations and launchers of k_grad_recompute (grad.cuh), plain form; see launch.h
#include "launch.h"
#include "kernels.cuh"
#include "grad.cuh"

cudaError_t mipwa_grad_set_smem(const int* n_spin, int fl, bool mix, int shp, size_t smem)
{
    if (mix) return mipwa_grad_set_smem_mix(n_spin, fl, smem);
    if (shp) return mipwa_grad_set_smem_shp(n_spin, fl, shp, smem);
    cudaError_t e = cudaSuccess;
    MIPWA_DISPATCH_SIGFL(n_spin[0], n_spin[1], n_spin[2], fl,
                         (e = cudaFuncSetAttribute(k_grad_recompute<R1, R2, FL, false, 0>,
                                                   cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem)));
    return e;
}

cudaError_t mipwa_launch_grad_recompute(const int* n_spin, int fl, bool mix, int shp, int grid, int ev_blocks, size_t smem,
                                        cudaStream_t st, const DevModel& m, const PointRec* ev, double kappa,
                                        long long n_ev, const PointRec* nm, long long n_norm, double* partials,
                                        double2* f_ev, double2* f_nm)
{
    if (mix)
        return mipwa_launch_grad_recompute_mix(n_spin, fl, grid, ev_blocks, smem, st, m, ev, kappa, n_ev, nm, n_norm,
                                               partials);
    if (shp)
        return mipwa_launch_grad_recompute_shp(n_spin, fl, shp, grid, ev_blocks, smem, st, m, ev, n_ev, nm, n_norm,
                                               partials);
    MIPWA_DISPATCH_SIGFL(n_spin[0], n_spin[1], n_spin[2], fl,
                         (k_grad_recompute<R1, R2, FL, false, 0><<<grid, MIPWA_GRAD_BLOCK, smem, st>>>(
                             m, ev, 0.0, n_ev, nm, n_norm, ev_blocks, partials, f_ev, f_nm)));
    return cudaGetLastError();
}
