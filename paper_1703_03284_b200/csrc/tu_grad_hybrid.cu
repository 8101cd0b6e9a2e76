// tu_grad_hybrid.cu -- instantiations and launchers of k_grad_hybrid (grad_hybrid.cuh); see launch.h
#include "launch.h"
#include "kernels.cuh"
#include "grad_hybrid.cuh"

cudaError_t mipwa_occupancy_grad_hybrid(int f1, int f2, int rc, int fl, size_t smem, int* blocks_per_sm)
{
    bool supported = true;
    cudaError_t e = cudaSuccess;
    MIPWA_DISPATCH_HYBFL(f1, f2, rc, fl,
                         e = cudaFuncSetAttribute(k_grad_hybrid<R1, R2, RCT, FL>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                                  (int)(smem + mipwa_grad_ring_bytes(RCT)));
                         if (e == cudaSuccess)
                             e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(blocks_per_sm, k_grad_hybrid<R1, R2, RCT, FL>,
                                                                               MIPWA_GRAD_BLOCK, smem + mipwa_grad_ring_bytes(RCT)));
    return supported ? e : cudaErrorInvalidValue;
}

cudaError_t mipwa_launch_grad_hybrid(int f1, int f2, int rc, int fl, int grid, size_t smem, cudaStream_t st,
                                     const DevModel& m, const HybCoef& cc, const double* e12, const double* e13,
                                     const unsigned short* eseg, const double2* ev_cache, long long n_ev, const double* g12,
                                     const double* g13, const double* gw, const unsigned short* gseg,
                                     const double2* nm_cache, long long n_norm, double* partials, double2* f_ev,
                                     double2* f_nm)
{
    bool supported = true;
    MIPWA_DISPATCH_HYBFL(f1, f2, rc, fl,
                         (k_grad_hybrid<R1, R2, RCT, FL><<<grid, MIPWA_GRAD_BLOCK, smem + mipwa_grad_ring_bytes(RCT), st>>>(
                             m, cc, e12, e13, eseg, ev_cache, n_ev, g12, g13, gw, gseg, nm_cache, n_norm, partials, f_ev,
                             f_nm)));
    return supported ? cudaGetLastError() : cudaErrorInvalidValue;
}
