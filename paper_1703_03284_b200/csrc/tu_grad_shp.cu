// tu_grad_shp.cu -- instantiations and launchers of k_grad_recompute (grad.cuh) with the shape sums of ONE floating
// resonance (the first device slot of its spin) folded in: mipwa_nll_grad_full / mipwa_nll_grad_parts; see launch.h
#include "launch.h"
#include "kernels.cuh"
#include "grad.cuh"

namespace {
// SHP = 1 needs a spin-1 slot, SHP = 2 a spin-2 slot; the generic <-1, -1> form has no compile-time slots: those
// combinations resolve to SHP = 0 here and are refused (the caller then takes the k_grad_shape route).
template <int R1, int R2, int FL, int SHP>
struct ShpKernel {
    static cudaError_t set_smem(size_t smem)
    {
        return cudaFuncSetAttribute(k_grad_recompute<R1, R2, FL, false, SHP>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                    (int)smem);
    }
    static cudaError_t launch(int grid, int ev_blocks, size_t smem, cudaStream_t st, const DevModel& m, const PointRec* ev,
                              long long n_ev, const PointRec* nm, long long n_norm, double* partials)
    {
        k_grad_recompute<R1, R2, FL, false, SHP><<<grid, MIPWA_GRAD_BLOCK, smem, st>>>(m, ev, 0.0, n_ev, nm, n_norm, ev_blocks,
                                                                                       partials, nullptr, nullptr);
        return cudaGetLastError();
    }
};
template <int R1, int R2, int FL>
struct ShpKernel<R1, R2, FL, 0> {
    static cudaError_t set_smem(size_t) { return cudaErrorInvalidValue; }
    static cudaError_t launch(int, int, size_t, cudaStream_t, const DevModel&, const PointRec*, long long, const PointRec*,
                              long long, double*)
    {
        return cudaErrorInvalidValue;
    }
};
template <int R1, int R2> constexpr int shp1() { return R1 >= 1 ? 1 : 0; }
template <int R1, int R2> constexpr int shp2() { return (R1 >= 0 && R2 >= 1) ? 2 : 0; }
}  // namespace

cudaError_t mipwa_grad_set_smem_shp(const int* n_spin, int fl, int shp, size_t smem)
{
    cudaError_t e = cudaErrorInvalidValue;
    MIPWA_DISPATCH_SIGFL(n_spin[0], n_spin[1], n_spin[2], fl,
                         (e = shp == 1 ? ShpKernel<R1, R2, FL, shp1<R1, R2>()>::set_smem(smem)
                                       : ShpKernel<R1, R2, FL, shp2<R1, R2>()>::set_smem(smem)));
    return e;
}

cudaError_t mipwa_launch_grad_recompute_shp(const int* n_spin, int fl, int shp, int grid, int ev_blocks, size_t smem,
                                            cudaStream_t st, const DevModel& m, const PointRec* ev, long long n_ev,
                                            const PointRec* nm, long long n_norm, double* partials)
{
    cudaError_t e = cudaErrorInvalidValue;
    MIPWA_DISPATCH_SIGFL(n_spin[0], n_spin[1], n_spin[2], fl,
                         (e = shp == 1 ? ShpKernel<R1, R2, FL, shp1<R1, R2>()>::launch(grid, ev_blocks, smem, st, m, ev, n_ev, nm,
                                                                                      n_norm, partials)
                                       : ShpKernel<R1, R2, FL, shp2<R1, R2>()>::launch(grid, ev_blocks, smem, st, m, ev, n_ev, nm,
                                                                                      n_norm, partials)));
    return e;
}
